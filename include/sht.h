/*
 * sht.h -- C ABI of the B200-native batched spherical-harmonic-transform library
 * (hot path of arXiv:2208.10154, "Accelerating spherical harmonic transforms for a large number of sky maps").
 *
 * What the calls compute (citations are /root/reference/PAPER.md line numbers):
 *   sht_analysis      Alg. 1: a_lm^k = sum_theta P_lm(theta) T_m^k(theta)     (eq. 1-3, :35-60)
 *                     spin 2: (A^E; iA^B)_m = [[F+,F-],[F-,F+]]_m (Q; iU)_m                      (eq. 14, :139)
 *   sht_synthesis     eq. 4-5: T_m = P_m^t A_m, then a backward FFT ring by ring;
 *                     spin 2: eq. 15 (:143)
 *   sht_analysis_iter Alg. 2, the "traditional" iteration of HEALPix (:300), kept
 *                     between T_m^k(theta) and a_lm because the ring FFT is lossless (item 8, :227)
 * on the HEALPix RING grid with constant quadrature weight dsigma = 4 pi / N_pix (:39),
 * mmax = lmax (Alg. 1 loops m = 0..lmax, :191).  Readings of everything the paper leaves open are
 * listed in DESIGN.md ("Readings of the paper").
 *
 * Conventions
 *   - extern "C", plain pointers and sizes; no C++ or torch types; nothing throws, exits or aborts.
 *   - Every entry returns sht_status_t; arguments are validated before anything is launched.
 *   - `maps`, `alm`, `resid_rms` of the device entries are DEVICE pointers owned by the caller
 *     (FP64, dense, 16-byte aligned); inputs are never modified; outputs are fully overwritten.
 *   - Device entries are asynchronous on `stream` (a cudaStream_t passed as void*, NULL = default
 *     stream); the library synchronises only in plan create/destroy, sht_plan_reserve_iter and the *_host
 *     entries.  One exception, stated at sht_analysis_iter: its first call on a plan that was not reserved
 *     allocates the second workspace (cudaMalloc); everything it queues is still ordered on `stream`.
 *   - A plan is used from one host thread at a time; distinct plans are independent.
 *   - There is no CPU fallback: without a CUDA device plan creation fails with SHT_ERR_CUDA.
 *
 * Layouts (ncomp = 1 for spin 0, 2 for spin 2)
 *   maps : [nmaps][ncomp][npix]    double, RING pixel order, components (Q,U); npix = 12 nside^2
 *   alm  : [nmaps][ncomp][nalm][2] double (re,im), components (E,B), m >= 0 only, m-major:
 *          idx(l,m) = m (2 lmax + 1 - m)/2 + l,  nalm = (lmax+1)(lmax+2)/2.
 *          Im(a_l0) is ignored on input and written as 0; spin 2: l < 2 ignored on input, written 0.
 */
#ifndef SHT_B200_H
#define SHT_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sht_plan_s* sht_plan_t;            /* opaque, owned by the library */

typedef enum {
    SHT_OK = 0,
    SHT_ERR_INVALID_ARG = -1,
    SHT_ERR_UNSUPPORTED = -2,
    SHT_ERR_ALLOC = -3,
    SHT_ERR_CUDA = -4,
    SHT_ERR_NULL = -5
} sht_status_t;

/* Plan: nside >= 1 (any integer, RING scheme; every nside <= 1024 is supported, larger ones return SHT_ERR_UNSUPPORTED
 * when a ring length does not fit the ring kernels' shared memory), lmax >= 0 (spin 2: lmax >= 2), nmaps >= 1 (spin 2: number of
 * (Q,U) pairs), spin in {0, 2}.  Builds on the current CUDA device: ring tables, FFT twiddles, recurrence
 * coefficients, the l_safe / seed table of PAPER.md:230-232 (item 11) and the T_m^k(theta) workspace.
 * This is the paper's "initialisation overhead", paid once and timed separately.
 * If the workspace for all nmaps does not fit, maps are processed in chunks internally. */
sht_status_t sht_plan_create(sht_plan_t* out, int nside, int lmax, int nmaps, int spin);
/* Same, with an upper bound (bytes, 0 = none) on the T_m^k(theta) workspace: maps are then processed in internal
 * chunks of sht_plan_chunk_maps() maps (a multiple of 64); SHT_ERR_ALLOC if not even one 64-map chunk fits. */
sht_status_t sht_plan_create_ex(sht_plan_t* out, int nside, int lmax, int nmaps, int spin, size_t workspace_limit);
sht_status_t sht_plan_destroy(sht_plan_t plan);   /* NULL is a no-op returning SHT_OK */

/* Where the P_lm (lambda; spin 2: F+/F-) tiles of the Legendre stage are produced (both run the same recurrence from
 * the same seeds and give bit-identical tiles, regenerated on every transform as in the paper):
 *   SHT_LAMBDA_FUSED  : inside the DMMA contraction kernel, by its generator warps, tiles never leave shared memory;
 *   SHT_LAMBDA_STAGED : by a separate kernel into an HBM scratch owned by the plan, streamed into the contraction
 *                       kernel with one bulk copy per stage (a scalar FP64 instruction next to DMMA costs the FP64 pipe
 *                       ~25 cycles on B200; this mode is the default when the scratch fits).
 * sht_plan_set_lambda_mode returns SHT_ERR_UNSUPPORTED if the plan cannot run the requested mode. */
enum { SHT_LAMBDA_FUSED = 0, SHT_LAMBDA_STAGED = 1 };
sht_status_t sht_plan_set_lambda_mode(sht_plan_t plan, int mode);
int sht_plan_lambda_mode(sht_plan_t plan);

/* Launch-shape options (measurement and comparison; every setting computes the same transforms, equal up to the order
 * of floating-point sums):
 *   SHT_OPT_RING_PATH         1 (default): the belt rings of a power-of-two nside, and the cap rings of 132 .. 2048 pixels,
 *                             go through the bulk-copy / TMA kernels (compiled power-of-two transforms, three-radix
 *                             mixed-radix transforms, chirp-z); 0: the general ring kernels do every ring
 *   SHT_OPT_LEG_TILES_PER_CTA spin-0 Legendre analysis: 0 = one CTA per (m, k-tile) walks all l tiles; n > 0 = one CTA per
 *                             (m, group of n l tiles, k-tile), so that the tiles of an order share T_m through L2 (default 2)
 *   SHT_OPT_LEG_RING_SPLIT    spin-0 Legendre synthesis: CTAs that share the ring blocks of an (m, k-tile) (default 3)
 *   SHT_OPT_ITER_HYBRID       SHT_ITER_IMMEDIATE: 1 (default) = the hybrid sweep when at least half of the ring pairs are
 *                             alias-free (see sht_plan_set_iter_mode); 0 = always the plain sweep, every ring pair in the chain
 *   SHT_OPT_ITER_ALIAS_FREE_FROM  read-only: the first ring pair (counted from the pole, a multiple of 64) from which on every
 *                             ring pair is alias-free for this plan's lmax; 2 nside if there is no such tail
 * SHT_ERR_INVALID_ARG for an unknown or read-only option or a negative value. */
enum { SHT_OPT_RING_PATH = 0, SHT_OPT_LEG_TILES_PER_CTA = 1, SHT_OPT_LEG_RING_SPLIT = 2, SHT_OPT_ITER_HYBRID = 3,
       SHT_OPT_ITER_ALIAS_FREE_FROM = 4 };
sht_status_t sht_plan_set_option(sht_plan_t plan, int option, int value);
int sht_plan_get_option(sht_plan_t plan, int option);    /* -1: unknown option */

/* Alg. 1: maps (device, in) -> alm (device, out). */
sht_status_t sht_analysis(sht_plan_t plan, const double* maps, double* alm, void* stream);
/* eq. 4-5: alm (device, in) -> maps (device, out). */
sht_status_t sht_synthesis(sht_plan_t plan, const double* alm, double* maps, void* stream);
/* Alg. 2: a(0) = analysis(map); niter x { a += analysis(map - synthesis(a)) }, niter >= 0.
 * resid_rms (device, may be NULL): [niter][nmaps*ncomp]; entry n = rms over pixels of
 * map - synthesis(a(n)) at the start of round n. */
sht_status_t sht_analysis_iter(sht_plan_t plan, const double* maps, double* alm, int niter,
                               double* resid_rms, void* stream);

/* Which iteration sht_analysis_iter runs and how it forms the residual.
 * Alg. 2, the "traditional" scheme, a_lm updated outside the m-loop -- two forms, same result up to
 * rounding:
 *   SHT_ITER_TM    : residual on the ring spectra T_m(theta), the maps are read once (item 8; default;
 *                    allocates a second workspace on the first call and falls back to SHT_ITER_PIXEL if that does not fit);
 *   SHT_ITER_PIXEL : as residual maps (one backward and one forward ring FFT more per round).
 * Alg. 3, the "immediate" scheme, a_lm updated inside the m-loop:
 *   SHT_ITER_IMMEDIATE : a(0) = analysis(map), r = map - synthesis(a(0)); then niter sweeps over m = 0 .. lmax in this
 *                    order: delta a_m = order m of analysis(r), a_m += delta a_m, r -= synthesis(delta a_m) at once, so the
 *                    orders after m see it through the ring aliasing (a Gauss-Seidel sweep; a different result from Alg. 2,
 *                    more accurate for lmax < 3 nside).  r is kept as ring spectra T_m(theta).  resid_rms
 *                    entry n = rms of r at the start of sweep n.  Spin 0 and spin 2 (E and B of an order together); needs
 *                    the second workspace (SHT_ERR_CUDA if it does not fit).  Sequential in m within each parity class of m:
 *                    3 launches per pair of orders (m even, m + 1).  Hybrid sweep (SHT_OPT_ITER_HYBRID): a ring of N
 *                    pixels on which every order present is <= N / 2 couples no two orders, so when at least half of the
 *                    ring pairs are such (lmax <= 2 nside) their share of every delta a_m is computed by one whole-
 *                    transform launch at the start of the sweep and their residual corrected by two launches at its end;
 *                    only the polar ring pairs and the low orders stay in the chain.  For 2 nside <= lmax < 4 nside (spin 0)
 *                    the belt ring pairs leave the chain in two groups of orders (below / from 2 nside: an order meets only
 *                    its mirror 4 nside - m there).  Same sweep, different order of the ring sums (results equal to
 *                    rounding). */
enum { SHT_ITER_TM = 0, SHT_ITER_PIXEL = 1, SHT_ITER_IMMEDIATE = 2 };
sht_status_t sht_plan_set_iter_mode(sht_plan_t plan, int mode);
/* Allocates (and zero-fills) the second workspace of SHT_ITER_TM / SHT_ITER_IMMEDIATE now and waits for it, so that
 * sht_analysis_iter never allocates or synchronises.  SHT_ERR_ALLOC if it does not fit (SHT_ITER_TM then runs as
 * SHT_ITER_PIXEL).  Without this call the first iterative call allocates it itself (one synchronous cudaMalloc; its
 * zero fill is queued on that call's stream). */
sht_status_t sht_plan_reserve_iter(sht_plan_t plan);

/* Spin-2 plans: transforms of a_lm^E or a_lm^B alone (item 9: "forward and backward transforms of a^E
 * and a^B separately ... the speed of SHTs can be increased by 100% for free"): half of the block products of eq. 14 /
 * eq. 15 are skipped.  `alm` holds ONE component: [nmaps][nalm][2] doubles, m-major.
 *   sht_analysis_pol : maps (Q,U) -> a^E (which = SHT_POL_E) or a^B (SHT_POL_B), equal to that component of sht_analysis
 *   sht_synthesis_pol: a^E or a^B -> maps (Q,U), equal to sht_synthesis with the other component set to zero */
enum { SHT_POL_E = 1, SHT_POL_B = 2 };
sht_status_t sht_analysis_pol(sht_plan_t plan, const double* maps, double* alm, int which, void* stream);
sht_status_t sht_synthesis_pol(sht_plan_t plan, const double* alm, double* maps, int which, void* stream);

/* Pixel-domain E/B decomposition (eq. 16 and 19): S^{E,B}_m = (F_m^t lambda^{E,B} F_m) S_m, i.e.
 * maps_out = sht_synthesis_pol(sht_analysis_pol(maps_in, which), which): the (Q,U) maps that carry only the E-family
 * (which = SHT_POL_E) or only the B-family (SHT_POL_B) part of maps_in -- the building block of the EB-leakage pipeline
 * (PAPER.md:273).  DEVICE pointers, [nmaps][2][npix]; maps_out may be maps_in; the a_lm of the one component live in a
 * stream-ordered scratch of the library.  Spin-2 plans only.  Asynchronous on `stream`. */
sht_status_t sht_eb_split(sht_plan_t plan, const double* maps_in, double* maps_out, int which, void* stream);

/* sht_eb_split for callers that cannot allocate (a stream under CUDA graph capture, a serving loop or a harness that
 * forbids cudaMalloc): same arguments, same result, but the a_lm scratch is a file-scope `__device__` array of the
 * library, SHT_EB_STATIC_MAX_BYTES long, instead of a stream-ordered allocation.  The call makes no cudaMalloc /
 * cudaMallocAsync / cudaFree and calls no allocating library routine (kernel launches and the plan's own workspace
 * only).  Every GPU that loads the library holds the array until the process exits.
 *   limit   : the scratch of one internal chunk, sht_plan_chunk_maps(plan) * sht_nalm(lmax) * 16 bytes, must fit:
 *             otherwise SHT_ERR_INVALID_ARG with the two sizes in sht_last_error (nothing is launched);
 *             create the plan with fewer maps, or use sht_eb_split.
 *   sharing : ALL calls, of all plans and streams on one device, use the same array.  Calls that overlap on the GPU
 *             race on it (undefined results, no fault): keep them on one stream or order them with events.  The
 *             array keeps the previous call's contents; nothing in it has to start at zero (the analysis half of a
 *             chunk writes every a_lm the synthesis half reads), so the call clears nothing.
 *   device  : the array's address is looked up once per device (cudaGetSymbolAddress with that device current), on
 *             the first call there; the plan's device must be the current one, as for every other call. */
#define SHT_EB_STATIC_MAX_BYTES (32u << 20)
sht_status_t sht_eb_split_static(sht_plan_t plan, const double* maps_in, double* maps_out, int which, void* stream);

/* Same transforms on HOST buffers (pinned or pageable; same layouts).  Each call copies its input to the
 * device, runs the device entry and copies the result back, in map chunks on the plan's own streams,
 * and returns after the result is complete in host memory.  They first wait for all device work queued before
 * (the chunk streams share the plan's workspace with the device entries).  These are the end-to-end calls bench.py times. */
sht_status_t sht_analysis_host(sht_plan_t plan, const double* maps_host, double* alm_host);
sht_status_t sht_synthesis_host(sht_plan_t plan, const double* alm_host, double* maps_host);

/* FP32 storage (NEXT row N4, north_star's optional FP32 path, tolerance 1e-4): the same transforms with `maps` and `alm`
 * held in single precision by the caller (float maps, complex64 a_lm; same layouts and index rules, 8-byte aligned).  The
 * arithmetic inside is unchanged FP64: inputs are widened and results rounded once, chunk by chunk, through the plan's
 * staging buffers, so the error against the FP64 result is one rounding of the output (relative 6e-8 of the largest
 * value) -- what these entries buy is half the bytes over PCIe and in the caller's memory, not a faster contraction (a
 * TF32 / tcgen05 contraction is not built).
 *   sht_*_f32       DEVICE pointers, asynchronous on `stream` like the FP64 entries (the first call allocates the
 *                   staging buffers: one synchronous cudaMalloc);
 *   sht_*_host_f32  HOST pointers, synchronous, chunked H2D -> widen -> transform -> round -> D2H on the plan's streams. */
sht_status_t sht_analysis_f32(sht_plan_t plan, const float* maps, float* alm, void* stream);
sht_status_t sht_synthesis_f32(sht_plan_t plan, const float* alm, float* maps, void* stream);
sht_status_t sht_analysis_host_f32(sht_plan_t plan, const float* maps_host, float* alm_host);
sht_status_t sht_synthesis_host_f32(sht_plan_t plan, const float* alm_host, float* maps_host);

/* The paper's packed storage (eq. A7): all a_lm of one map in a real (lmax+1) x (lmax+1) matrix,
 * row-major, Re a_lm at (row l, column m), Im a_lm (m >= 1) at (row l - m, column lmax - m + 1); Im a_l0 is not stored
 * and reads back as 0 (0-based indices, reading G20).  Converters between it and the m-major `alm` layout:
 * `rows` = nmaps * ncomp matrices, DEVICE pointers, asynchronous on `stream`; no plan needed. */
sht_status_t sht_alm_pack_a7(int lmax, long long rows, const double* alm, double* packed, void* stream);
sht_status_t sht_alm_unpack_a7(int lmax, long long rows, const double* packed, double* alm, void* stream);

/* Introspection (host, pure). */
long long sht_npix(int nside);                       /* 12 nside^2                                  */
long long sht_nalm(int lmax);                        /* (lmax+1)(lmax+2)/2                          */
long long sht_alm_index(int lmax, int l, int m);     /* m(2 lmax+1-m)/2 + l; -1 if out of range     */
size_t sht_plan_workspace_bytes(sht_plan_t plan);    /* device bytes held by the plan               */
int sht_plan_chunk_maps(sht_plan_t plan);            /* maps processed per internal chunk           */
/* FP64 tensor-core flops ONE call of sht_analysis (direction 0) / sht_synthesis (1) executes in its contraction kernel
 * after ring pruning (item 10), l_safe row skipping (item 11, :230-232) and tile padding -- the kernels' skip
 * logic replayed on the plan's tables (measurement only: bench.py's hardware-rate roofline fraction).  Spin-2 plans: the
 * count of the E-and-B transforms (the E-only / B-only entries execute half of it).  -1: bad arguments. */
double sht_plan_executed_flops(sht_plan_t plan, int direction);
long long sht_plan_kernel_launches(sht_plan_t plan); /* kernels launched by this plan so far        */
const char* sht_status_string(sht_status_t s);       /* static storage                              */
const char* sht_last_error(sht_plan_t plan);         /* plan-owned, valid until the next call       */

/* Per-stage device timing (measurement only; PAPER.md:54 quotes the FFT + FFT-mapping share of the time).
 * With timing enabled every kernel launched by the plan on the caller's stream is bracketed by CUDA events.
 * sht_plan_stage_ms waits for the recorded events and returns, accumulated since the last call, the device
 * milliseconds ms[4] and launch counts n[4] of: 0 ring-FFT analysis, 1 Legendre analysis, 2 Legendre synthesis,
 * 3 ring-FFT synthesis; then resets the accumulation.  SHT_ERR_ALLOC (sums incomplete) if a bracket could not be recorded. */
sht_status_t sht_plan_set_timing(sht_plan_t plan, int enable);
sht_status_t sht_plan_stage_ms(sht_plan_t plan, double* ms4, int* n4);

/* Measurement helper used by bench.py for the roofline denominator: runs a register-resident
 * DMMA.8x8x4 loop on every SM for about `ms` milliseconds and returns the sustained FP64
 * tensor-core rate in TFLOP/s (<= 0 on error).  Not part of the transform path. */
double sht_measure_fp64_mma_peak(double ms);

#ifdef __cplusplus
}
#endif
#endif /* SHT_B200_H */
