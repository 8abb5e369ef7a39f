#!/usr/bin/env python
"""bench.py -- headline benchmark: batched FP64 analysis + synthesis of HEALPix maps on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch: sht_synthesis (a_lm -> maps) followed by
sht_analysis (maps -> a_lm) of all `nmaps` maps of the workload (BASELINE.json metric: maps/s of
analysis+synthesis in FP64 at nside=512, lmax=1535; workload = BASELINE.json configs[2], K = 1000 maps).
`value` is measured with inputs resident in HBM; `e2e` through the host-buffer C-ABI entries
(sht_synthesis_host / sht_analysis_host) with pinned host buffers, H2D/D2H inside the timed region.
N > 1 (torchrun): every rank runs the same workload on its own maps (weak scaling, no collective on the
data path; maps are independent units).
`--impl reference` times the CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2208_10154_b200 import inputs, shard  # noqa: E402

FP64_NOMINAL_TFLOPS = 37.2     # 148 SMs x 64 FP64 FMA/clk x 2 x 1.965 GHz
def ncu_capture_row(config, nmaps, lambda_mode, kernel):
    """dram bytes per launch / DMMA pipe activity of `kernel` from the newest committed ncu capture of exactly this
    workload (profiles/ncu_latest.csv: config,nmaps,lambda_mode,kernel,dram_bytes,dmma_pipe_active,capture,commit), or
    None.  The values describe the commit named there; the line says so."""
    path = os.path.join(ROOT, "profiles", "ncu_latest.csv")
    if not os.path.exists(path):
        return None
    for ln in open(path):
        f = [x.strip() for x in ln.split(",")]
        if len(f) >= 8 and f[0] == str(config) and f[1] == str(nmaps) and f[2] == lambda_mode and f[3] == kernel:
            return {"traffic": int(float(f[4])), "dmma_pipe_active": float(f[5]), "capture": f[6], "commit": f[7]}
    return None


def read_measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def legendre_flops_per_direction(c):
    """folded, unpruned algorithmic flops n_alm * N_h * 2K * 2 (x4 for spin 2)."""
    f = inputs.nalm(c["lmax"]) * (2 * c["nside"]) * 2 * c["nmaps"] * 2
    return f * (4 if c["spin"] == 2 else 1)


def min_hbm_bytes_per_direction(c, kpad):
    ncomp = 2 if c["spin"] == 2 else 1
    maps = 8 * inputs.npix(c["nside"]) * c["nmaps"] * ncomp
    alm = 16 * inputs.nalm(c["lmax"]) * c["nmaps"] * ncomp
    F = 16 * (c["lmax"] + 1) * (2 * c["nside"]) * 2 * c["nmaps"] * ncomp
    return maps + alm + 2 * F


def oracle_timed_sample(c, ks):
    """The oracle as it stands on the box's host cores: full synthesis (every ring) then full analysis (every m) of the
    maps `ks` of the workload -- maps are independent units, so sample size / wall time is the oracle's throughput
    (SURVEY.md 8(d) "Oracle timing").  Nothing is extrapolated.  Returns (maps per second, seconds, threads)."""
    from oracle import oracle as O
    nside, lmax = c["nside"], c["lmax"]
    alm = inputs.gaussian_alm(lmax, np.asarray(ks), c["seed"], c["spin"])
    t0 = time.time()
    maps = O.synthesis(nside, lmax, alm, spin=c["spin"])
    O.analysis(nside, lmax, maps, spin=c["spin"])
    dt = time.time() - t0
    return len(ks) / dt, dt, O.num_threads()


def oracle_sample_size(c, n_calls):
    """Maps per oracle call, the same rule for the cpu_baseline leg and the --impl reference arm so that their numbers
    are comparable (the oracle shares its lambda / phase tables among the maps of a call, so its throughput depends on
    the sample size): the 8-map comparison subset of SURVEY.md 8(d) when the run makes few calls, fewer maps when the
    driver asks for many steps, so that the reference arm still ends within a few minutes."""
    n = 8 if n_calls <= 6 else 4 if n_calls <= 12 else 2 if n_calls <= 24 else 1
    return min(n, c["nmaps"])


def cpu_baseline(c, nsample):
    """cpu_baseline leg: one timed oracle call on the first `nsample` maps of the workload."""
    ks = list(range(min(nsample, c["nmaps"])))
    v, dt, cores = oracle_timed_sample(c, ks)
    return {"value": v, "unit": unit_of(c), "cores": cores, "kind": "oracle",
            "sample": "maps %d..%d of the workload: full synthesis (all %d rings) + full analysis (all %d orders m), "
                      "%.1f s of wall time, nothing extrapolated" % (ks[0], ks[-1], 4 * c["nside"] - 1, c["lmax"] + 1, dt)}


def unit_of(c):
    return "pairs/s" if c["spin"] == 2 else "maps/s"


def metric_of(c):
    """BASELINE.json's metric string with the workload's own sizes (the headline workload gives it verbatim)"""
    return "%s/sec (analysis+synthesis, FP64) at nside=%d lmax=%d" % ("(Q,U) pairs" if c["spin"] == 2 else "maps",
                                                                       c["nside"], c["lmax"])


def base_config(c):
    return {"workload": c["name"], "nside": c["nside"], "lmax": c["lmax"], "nmaps_per_gpu": c["nmaps"], "spin": c["spin"]}


def run_reference(args, c):
    """Reference arm = the oracle on the host cores (there is no other implementation of the paper here).  Each step
    transforms a bounded sample of the workload in full (oracle_sample_size).  ms_per_step is the wall time a step took."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    nsample = oracle_sample_size(c, args.steps + args.warmup)
    for _ in range(args.warmup):
        oracle_timed_sample(c, list(range(nsample)))
    vals, secs = [], []
    for _ in range(args.steps):
        v, dt, cores = oracle_timed_sample(c, list(range(nsample)))
        vals.append(v); secs.append(dt)
    v = float(nsample * len(secs) / sum(secs))
    cb = {"value": v, "unit": unit_of(c), "cores": cores, "kind": "oracle",
          "sample": "%d map(s) per step: full synthesis + full analysis, nothing extrapolated; %d steps, %.1f s per step"
                    % (nsample, args.steps, float(np.mean(secs)))}
    line = {"impl": "reference", "metric": metric_of(c), "value": v, "unit": unit_of(c), "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
            "maps_per_step": nsample,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": base_config(c), "cpu_baseline": cb,
            "e2e": {"value": v, "unit": unit_of(c), "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def cublas_dgemm_peak(dev, seconds=2.0, n=8192):
    """Reported comparison only (north_star: "cuBLAS DGEMM kept only as a reported comparison"; SURVEY.md 8(d) "quote all
    three"): torch.matmul FP64 n^3 (= cuBLAS DGEMM) back to back for `seconds`, with the SM clock sampled meanwhile.
    Lives in bench.py only; the library links no cuBLAS."""
    import torch
    a = torch.randn((n, n), dtype=torch.float64, device=dev)
    b = torch.randn((n, n), dtype=torch.float64, device=dev)
    o = torch.empty((n, n), dtype=torch.float64, device=dev)
    for _ in range(3):
        torch.matmul(a, b, out=o)
    torch.cuda.synchronize()
    smp = ClockSampler(dev.index or 0)
    smp.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, ms = 0, 0.0
    e0.record()
    while ms < seconds * 1e3:
        for _ in range(4):
            torch.matmul(a, b, out=o)
        reps += 4
        e1.record()
        e1.synchronize()
        ms = e0.elapsed_time(e1)
    clk = smp.stop()
    return {"tflops": 2.0 * n ** 3 * reps / (ms * 1e-3) * 1e-12, "n": n, "seconds": ms * 1e-3, "sm_mhz": clk.get("sm_mhz"),
            "reasons": clk.get("reasons")}


def cublas_per_m_dgemm(c, dev, mstep=1):
    """The paper's own formulation of the Legendre stage (Alg. 1 l.10; items 6-7, :220-224): one real DGEMM
    per order m of a materialised P_m against the ring spectra of all maps, timed with cuBLAS (torch.matmul) on matrices of
    the right shapes -- (lmax - m + 1) x rings times rings x 2K, analysis orientation; the synthesis product has the
    same flops.  DGEMM time does not depend on the values, so P_m and T_m are random here (the comparison is about the
    contraction, P_m generation is not included).  `unfolded`: all 4 nside - 1 rings, the paper's form; `folded`: two
    products per m over the 2 nside ring pairs (even / odd l - m), the north/south fold of north_star.  No ring pruning."""
    import torch
    nside, lmax, K = c["nside"], c["lmax"], c["nmaps"]
    ncomp = 2 if c["spin"] == 2 else 1
    nr, nh, ncol = 4 * nside - 1, 2 * nside, 2 * K * ncomp
    blk = (2 if c["spin"] == 2 else 1)                   # spin 2: the 2 x 2 block matrix [[F+,F-],[F-,F+]] (eq. 14)
    P = torch.randn((blk * (lmax + 1), blk * nr), dtype=torch.float64, device=dev)
    T = torch.randn((blk * nr, ncol // blk), dtype=torch.float64, device=dev)
    out = torch.empty((blk * (lmax + 1), ncol // blk), dtype=torch.float64, device=dev)
    res = {}
    for name in ("unfolded", "folded"):
        def run():
            for m in range(0, lmax + 1, mstep):
                nl = lmax - m + 1
                if name == "unfolded":
                    torch.matmul(P[:blk * nl, :], T, out=out[:blk * nl])
                else:
                    ne, no = (nl + 1) // 2, nl // 2
                    torch.matmul(P[:blk * ne, :blk * nh], T[:blk * nh], out=out[:blk * ne])
                    if no:
                        torch.matmul(P[:blk * no, :blk * nh], T[:blk * nh], out=out[:blk * no])
        run()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        run()
        e1.record()
        e1.synchronize()
        res[name + "_ms_per_direction"] = e0.elapsed_time(e1) * mstep
    res["mstep"] = mstep
    res["note"] = "cuBLAS DGEMM per m on random matrices of the paper's shapes; operands L2/HBM resident, P_m generation excluded"
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--nmaps", type=int, default=0, help="override the workload's map count (debug only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--pol", default="", choices=["", "E", "B"],
                    help="spin-2 workloads: time the E-only / B-only transforms (PAPER.md:228) instead of the full ones")
    ap.add_argument("--iter", type=int, default=-1,
                    help="time sht_analysis_iter with this many Jacobi rounds (Alg. 2; BASELINE.json configs[4] uses 3) "
                         "instead of the synthesis + analysis step")
    ap.add_argument("--iter-mode", default="tm", choices=["tm", "pixel", "immediate"],
                    help="with --iter: Alg. 2 with the residual on the ring spectra (tm, default) or as maps (pixel), or "
                         "Alg. 3, the immediate iteration (one order m at a time, spin 0)")
    ap.add_argument("--lambda-mode", default="", choices=["", "fused", "staged"],
                    help="where the P_lm tiles are generated (include/sht.h); default: the plan's own choice")
    ap.add_argument("--ring-path", default="", choices=["", "fast", "general"],
                    help="SHT_OPT_RING_PATH: belt / mixed-radix / chirp-z ring kernels (fast, the default) or the general ones only")
    ap.add_argument("--leg-tiles", type=int, default=-1, help="SHT_OPT_LEG_TILES_PER_CTA (default: the plan's)")
    ap.add_argument("--leg-split", type=int, default=-1, help="SHT_OPT_LEG_RING_SPLIT (default: the plan's)")
    ap.add_argument("--compare", default="", choices=["", "cublas"],
                    help="cublas: also time the paper's per-m cuBLAS DGEMM formulation of the Legendre stage (comparison only)")
    ap.add_argument("--no-cublas-peak", action="store_true",
                    help="skip the 2 s cuBLAS DGEMM peak measurement (comparison leg, after the timed region); used for the "
                         "ncu launch lists so that they hold the library's own kernels only")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-f32", action="store_true", help="also time the end-to-end step with FP32 storage at the ABI (e2e.fp32_storage)")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    c = dict(inputs.CONFIGS[args.config])
    if args.nmaps:
        c["nmaps"] = args.nmaps
        c["name"] += "_nmaps%d_DEBUG" % args.nmaps
    if args.impl == "reference":
        return run_reference(args, c)

    import torch
    import torch.distributed as dist
    from paper_2208_10154_b200.binding import Plan, sht_measure_fp64_mma_peak

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    nside, lmax, nmaps, spin = c["nside"], c["lmax"], c["nmaps"], c["spin"]
    ncomp = 2 if spin == 2 else 1
    npix, nalm = inputs.npix(nside), inputs.nalm(lmax)

    # ---- seeded synthetic inputs, resident in HBM (each rank its own maps: weak scaling) --------------
    alm = torch.empty((nmaps, ncomp, nalm), dtype=torch.complex128, device=dev)
    blk = 50
    for k0 in range(0, nmaps, blk):
        ks = shard.rank_map_indices(rank, world, nmaps)[k0:min(nmaps, k0 + blk)]
        alm[k0:k0 + len(ks)] = torch.from_numpy(inputs.gaussian_alm(lmax, ks, c["seed"], spin)).to(dev)
    maps = torch.empty((nmaps, ncomp, npix), dtype=torch.float64, device=dev)
    alm_out = torch.empty_like(alm)

    t0 = time.time()
    plan = Plan(nside, lmax, nmaps, spin)
    torch.cuda.synchronize()
    plan_s = time.time() - t0
    if args.lambda_mode:
        plan.sht_plan_set_lambda_mode(1 if args.lambda_mode == "staged" else 0)
    lambda_mode = "staged" if plan.sht_plan_lambda_mode() == 1 else "fused"
    if args.ring_path:
        plan.sht_plan_set_option(0, 1 if args.ring_path == "fast" else 0)
    if args.leg_tiles >= 0:
        plan.sht_plan_set_option(1, args.leg_tiles)
    if args.leg_split >= 0:
        plan.sht_plan_set_option(2, args.leg_split)
    options = {"ring_path": "fast" if plan.sht_plan_get_option(0) else "general",
               "leg_tiles_per_cta": plan.sht_plan_get_option(1), "leg_ring_split": plan.sht_plan_get_option(2)}
    stream = torch.cuda.current_stream()

    if args.pol:
        assert spin == 2, "--pol needs a spin-2 workload (--config 4)"
        which = 1 if args.pol == "E" else 2
        c["name"] += "_%s_only" % args.pol
        alm = alm[:, which - 1, :].contiguous()
        alm_out = torch.empty_like(alm)
        args.no_e2e = True

        def step():
            plan.sht_synthesis_pol(alm, maps, which, stream)
            plan.sht_analysis_pol(maps, alm_out, which, stream)
    elif args.iter >= 0:
        # Alg. 2 on maps synthesised once outside the timed region: 2 niter + 1 transforms per step (eq. B8)
        c["name"] += "_iter%d" % args.iter + ("" if args.iter_mode == "tm" else "_" + args.iter_mode)
        args.no_e2e = True
        plan.sht_plan_set_iter_mode({"tm": 0, "pixel": 1, "immediate": 2}[args.iter_mode])
        plan.sht_synthesis(alm, maps, stream)
        rms = torch.empty((max(args.iter, 1), nmaps * ncomp), dtype=torch.float64, device=dev)

        def step():
            plan.sht_analysis_iter(maps, alm_out, args.iter, rms, stream)
    else:
        def step():
            plan.sht_synthesis(alm, maps, stream)
            plan.sht_analysis(maps, alm_out, stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    plan.sht_plan_set_timing(True)
    l0 = plan.kernel_launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = plan.kernel_launches() - l0
    stage_ms, stage_n = plan.sht_plan_stage_ms()
    plan.sht_plan_set_timing(False)
    ms_total = shard.max_over_ranks(ms_total, dev)
    ms_step = ms_total / args.steps
    value = world * nmaps / (ms_step * 1e-3)

    # ---- roofline of the dominant kernel: k_legendre_analysis (the slower of the two Legendre launches; the synthesis
    # kernel, same design, is reported beside it in "stages") ---------------------------------------------------------
    peaks, peak_src = read_measured_peaks()
    fl_dir = legendre_flops_per_direction(c) / (2 if args.pol else 1)   # half of the block products
    # transforms per step inside the timed brackets of the Legendre stages (1 = analysis, 2 = synthesis).  Alg. 2: niter + 1
    # analyses, niter syntheses.  Alg. 3: the "analysis" brackets hold the initial analysis and the sweeps, and a sweep does
    # the analysis and the synthesis of every order (2 transforms); the one full synthesis is the initial residual
    dirs = {1: 1, 2: 1}
    if args.iter >= 0:
        dirs = {1: 2 * args.iter + 1, 2: 1} if args.iter_mode == "immediate" else {1: args.iter + 1, 2: max(args.iter, 1)}
    mma_peak = sht_measure_fp64_mma_peak(300.0)
    cublas_peak = cublas_dgemm_peak(dev) if (rank == 0 and not args.no_cublas_peak) else None
    cublas_cmp = cublas_per_m_dgemm(c, dev) if (args.compare == "cublas" and rank == 0) else None
    peak_note = ("FP64 DMMA.8x8x4 register-resident loop measured live in this run "
                 "(MEASURED_PEAKS.json has no FP64 entry; nominal 148 SM x 64 FMA/clk x 1.965 GHz = %.1f; "
                 "rule-derived bf16 %s x 45/2250 = %.1f)"
                 % (FP64_NOMINAL_TFLOPS, peak_src, peaks.get("bf16_tflops", 0) * 45.0 / 2250.0))

    # the committed captures describe the plain analysis + synthesis step with the default launch shapes only
    default_shapes = options == {"ring_path": "fast", "leg_tiles_per_cta": 2, "leg_ring_split": 3}
    plain_key = None if (args.pol or args.iter >= 0 or not default_shapes) else (args.config, nmaps, lambda_mode)

    def leg_roofline(stage, kernel):
        n = max(1, stage_n[stage])                          # timed brackets = calls of the stage (generator + contraction)
        launch_ms = stage_ms[stage] / n
        flops_per_launch = fl_dir * dirs[stage] * args.steps / n          # algorithmic (folded, unpruned) flops of one launch
        ach = flops_per_launch / (launch_ms * 1e-3) * 1e-12
        cap = None if plain_key is None else ncu_capture_row(*plain_key, kernel)
        # flops the contraction kernel really executes (pruning, l_safe skipping, tile padding), counted by the plan
        ex = plan.executed_flops(stage - 1) if not args.pol else -1.0
        ex_rate = ex * dirs[stage] * args.steps / n / (launch_ms * 1e-3) * 1e-12 if ex > 0 else None
        return {"bound": "tensor", "kernel": kernel, "achieved": ach, "peak": mma_peak, "unit": "TFLOP/s",
                "frac": ach / mma_peak, "traffic": cap["traffic"] if cap else None,
                "executed_flops_per_launch": ex * dirs[stage] * args.steps / n if ex > 0 else None,
                "achieved_executed": ex_rate, "frac_executed": ex_rate / mma_peak if ex_rate else None,
                "ncu_capture": cap,
                "algorithmic_flops_per_launch": flops_per_launch, "launch_ms": launch_ms,
                "share_of_step": stage_ms[stage] / ms_total}

    # staged mode: a Legendre "launch" is the lambda-block generator kernel plus the contraction kernel (both timed)
    roofline = leg_roofline(1, "k_legendre_analysis")
    roofline["peak_source"] = peak_note
    if cublas_peak:
        roofline["peak_cublas_dgemm"] = cublas_peak["tflops"]
        roofline["peak_cublas_dgemm_how"] = ("torch.matmul FP64 %d^3 back to back for %.1f s, SM clock median %s MHz, reasons %s "
                                             "(comparison only, bench.py; the library links no cuBLAS)"
                                             % (cublas_peak["n"], cublas_peak["seconds"], cublas_peak["sm_mhz"], cublas_peak["reasons"]))
    if cublas_cmp:
        roofline["cublas_per_m_dgemm"] = cublas_cmp
    roofline["traffic_source"] = ("dram__bytes_read.sum + dram__bytes_write.sum per launch from the capture named in ncu_capture "
                                  "(profiles/ncu_latest.csv); null if no capture of this exact workload is committed")
    roofline["note"] = ("achieved / frac = algorithmic (N/S-folded, UNPRUNED) flops / time, as SURVEY.md 8(d) defines the unit "
                        "(can exceed 1: ring pruning and l_safe skipping are the method's own saving); achieved_executed / "
                        "frac_executed = the DMMA flops the kernel really executes (sht_plan_executed_flops) / the same time = "
                        "the hardware rate against the same live peak")
    roofline_syn = leg_roofline(2, "k_legendre_synthesis")
    ring_ms = stage_ms[0] + stage_ms[3]
    ring_bytes = 2 * args.steps * (8 * npix * nmaps * ncomp + 16 * (lmax + 1) * 2 * nside * 2 * nmaps * ncomp)
    ring_gbs = ring_bytes / (ring_ms * 1e-3) * 1e-9 if ring_ms > 0 else None
    stages = {"legendre_synthesis_roofline": roofline_syn, "ring_fft_analysis_ms": stage_ms[0] / args.steps, "legendre_analysis_ms": stage_ms[1] / args.steps,
              "legendre_synthesis_ms": stage_ms[2] / args.steps, "ring_fft_synthesis_ms": stage_ms[3] / args.steps,
              "ring_fft_hbm": {"bound": "hbm", "achieved": ring_gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                               "frac": (ring_gbs / peaks["hbm_gbs"]) if ring_gbs else None,
                               "algorithmic_bytes": "maps (8 B/px) + workspace (16 B per (m, ring, map))",
                               "peak_source": peak_src},
              "min_hbm_bytes_per_direction": min_hbm_bytes_per_direction(c, 0)}

    # ---- end to end through the host-buffer ABI entries ------------------------------------------------
    e2e = None
    if not args.no_e2e:
        try:
            h_alm = torch.empty((nmaps, ncomp, nalm), dtype=torch.complex128).pin_memory()
            h_maps = torch.empty((nmaps, ncomp, npix), dtype=torch.float64).pin_memory()
            h_alm_out = torch.empty((nmaps, ncomp, nalm), dtype=torch.complex128).pin_memory()
            h_alm.copy_(alm.cpu())
            # device buffers of the resident run are not needed any more
            del alm_out
            torch.cuda.empty_cache()
            plan.sht_synthesis_host(h_alm, h_maps)          # warm-up (also allocates the staging buffers)
            plan.sht_analysis_host(h_maps, h_alm_out)
            if world > 1:
                dist.barrier()
            nrep = max(1, min(args.steps, 2))
            t0 = time.perf_counter()
            for _ in range(nrep):
                plan.sht_synthesis_host(h_alm, h_maps)
                plan.sht_analysis_host(h_maps, h_alm_out)
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / nrep
            dt = shard.max_over_ranks(dt, dev)
            bytes_alm = h_alm.numel() * 16
            bytes_maps = h_maps.numel() * 8
            e2e = {"value": world * nmaps / dt, "unit": unit_of(c), "h2d_bytes_per_step": bytes_alm + bytes_maps,
                   "d2h_bytes_per_step": bytes_alm + bytes_maps, "ms_per_step": dt * 1e3,
                   "api": "sht_synthesis_host + sht_analysis_host (pinned host buffers, chunked H2D/compute/D2H)"}
        except Exception as ex:  # host memory too small for pinned copies of the workload, etc.
            e2e = {"value": None, "unit": unit_of(c), "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                   "error": str(ex)[:200]}
        # the same step with FP32 storage at the ABI (float32 maps, complex64 a_lm in host memory, FP64 arithmetic on the
        # device): an extra line for callers whose maps are single precision; `e2e` above stays the FP64 metric
        if e2e.get("value") and args.e2e_f32:
            try:
                f_alm = h_alm.to(torch.complex64).pin_memory()
                del h_alm, h_alm_out, h_maps
                f_maps = torch.empty((nmaps, ncomp, npix), dtype=torch.float32).pin_memory()
                f_alm_out = torch.empty((nmaps, ncomp, nalm), dtype=torch.complex64).pin_memory()
                plan.sht_synthesis_host_f32(f_alm, f_maps)
                plan.sht_analysis_host_f32(f_maps, f_alm_out)
                if world > 1:
                    dist.barrier()
                t0 = time.perf_counter()
                for _ in range(nrep):
                    plan.sht_synthesis_host_f32(f_alm, f_maps)
                    plan.sht_analysis_host_f32(f_maps, f_alm_out)
                torch.cuda.synchronize()
                dt = shard.max_over_ranks((time.perf_counter() - t0) / nrep, dev)
                nb = f_alm.numel() * 8 + f_maps.numel() * 4
                e2e["fp32_storage"] = {"value": world * nmaps / dt, "unit": unit_of(c), "h2d_bytes_per_step": nb,
                                       "d2h_bytes_per_step": nb, "ms_per_step": dt * 1e3,
                                       "api": "sht_synthesis_host_f32 + sht_analysis_host_f32 (float32 / complex64 in pinned host "
                                              "memory; arithmetic unchanged FP64)"}
            except Exception as ex:
                e2e["fp32_storage"] = {"value": None, "error": str(ex)[:200]}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_baseline(c, oracle_sample_size(c, args.steps + args.warmup))

    if rank == 0:
        line = {"metric": metric_of(c), "value": value, "unit": unit_of(c), "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {**base_config(c),
                           "l2": "inputs (%.1f GB maps, %.1f GB a_lm per GPU) are far larger than the 126 MB L2"
                                 % (8e-9 * npix * nmaps * ncomp, 16e-9 * nalm * nmaps * ncomp),
                           "plan_create_s": plan_s, "chunk_maps": plan.chunk_maps(), "lambda_mode": lambda_mode, "options": options,
                           "workspace_GB": plan.workspace_bytes() * 1e-9},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "stages": stages, "cpu_baseline": cpu}
        print(json.dumps(line))
    plan.destroy()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
