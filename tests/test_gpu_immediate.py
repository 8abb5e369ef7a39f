"""GPU parity of Alg. 3, the "immediate" iteration (SHT_ITER_IMMEDIATE; reading G21), against
the oracle's sweep over the orders m written on the pixels (oracle.analysis_iter_immediate, pinned in
tests/test_oracle_immediate.py): element by element on the a_lm, and the per-sweep residual rms.  Tolerance as for the
plain transforms: per map max|x - ref| / max|ref| <= 1e-10."""
import numpy as np
import pytest

from paper_2208_10154_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _dev():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch.device("cuda:0")


def _run(plan, maps, niter, mode):
    import torch
    plan.sht_plan_set_iter_mode(mode)
    mp = torch.from_numpy(np.ascontiguousarray(maps)).to(_dev())
    alm = torch.full((plan.nmaps, plan.ncomp, plan.nalm), float("nan"), dtype=torch.complex128, device=_dev())
    rms = torch.full((max(niter, 1), plan.nmaps * plan.ncomp), float("nan"), dtype=torch.float64, device=_dev())
    plan.sht_analysis_iter(mp, alm, niter, rms)
    torch.cuda.synchronize()
    return alm.cpu().numpy(), rms.cpu().numpy()[:niter]


@pytest.mark.parametrize("nside,lmax,nmaps,niter,noise", [
    (16, 31, 5, 3, 0.0),       # band-limited to 2 nside - 1
    (16, 47, 3, 2, 0.0),       # lmax = 3 nside - 1: the orders alias on every cap ring
    (16, 47, 4, 3, 0.3),       # not band-limited (white noise): uncovered ring bins enter the rms
    (32, 95, 70, 2, 0.0),      # two k-tiles
    (48, 100, 2, 3, 0.1),      # nside not a power of two: Bluestein / prime ring lengths
    (64, 191, 3, 1, 0.0),      # two l tiles per order (192 > 128 rows): the order is split over CTAs
    (3, 8, 2, 3, 0.2),         # tiny rings: an order shares its bin with many others
    (8, 15, 2, 0, 0.0),        # zero sweeps: the plain analysis
])
def test_immediate_iteration_against_oracle(nside, lmax, nmaps, niter, noise):
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 91)
    maps = O.synthesis(nside, lmax, alm_true)
    if noise > 0.0:
        maps = maps + inputs.white_noise(nside, np.arange(nmaps), 92, noise)
    ref_alm, ref_rms = O.analysis_iter_immediate(nside, lmax, maps, niter)
    plan = Plan(nside, lmax, nmaps, 0)
    got_alm, got_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    plan.destroy()
    assert np.isfinite(got_alm).all()
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    if niter > 0:
        assert np.abs(got_rms - ref_rms).max() <= 1e-9 * ref_rms[0].max()


def test_immediate_differs_from_traditional_and_is_more_accurate():
    """the two schemes are different iterations: on a map band-limited to lmax = 3 nside - 1 they disagree
    far above rounding, each agrees with its own oracle, and the immediate one ends closer to the input a_lm"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE, SHT_ITER_TM
    nside, lmax, nmaps, niter = 32, 95, 4, 3
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 93)
    maps = O.synthesis(nside, lmax, alm_true)
    plan = Plan(nside, lmax, nmaps, 0)
    a_imm, _ = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    a_trad, _ = _run(plan, maps, niter, SHT_ITER_TM)
    plan.destroy()
    assert inputs.rel_err(a_imm, a_trad) > 1e-7
    assert inputs.rel_err(a_trad, O.analysis_iter(nside, lmax, maps, niter)[0]) <= TOL
    assert inputs.rel_err(a_imm, O.analysis_iter_immediate(nside, lmax, maps, niter)[0]) <= TOL
    assert inputs.rel_err(a_imm, alm_true) < inputs.rel_err(a_trad, alm_true)


@pytest.mark.parametrize("nside,lmax", [(16, 47), (64, 127)], ids=["plain_sweep", "hybrid_sweep"])
def test_immediate_chunked_workspace_and_repeat(nside, lmax):
    """a workspace limit that forces 64-map chunks gives the same a_lm as one chunk; a second call on the same plan
    (workspaces reused, their roles swapped inside a call) repeats the first bit for bit"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE
    nmaps, niter = 100, 2
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 94)
    maps = O.synthesis(nside, lmax, alm_true)
    full = Plan(nside, lmax, nmaps, 0)
    per_map = 2 * nside * (lmax + 1) * 2 * 16
    small = Plan(nside, lmax, nmaps, 0, workspace_limit=70 * per_map)
    assert full.chunk_maps() == nmaps and small.chunk_maps() == 64
    a_full, r_full = _run(full, maps, niter, SHT_ITER_IMMEDIATE)
    a_again, _ = _run(full, maps, niter, SHT_ITER_IMMEDIATE)
    a_small, r_small = _run(small, maps, niter, SHT_ITER_IMMEDIATE)
    full.destroy(); small.destroy()
    assert np.array_equal(a_full, a_again)
    assert np.array_equal(a_full, a_small)
    assert np.allclose(r_full, r_small, rtol=1e-12, atol=0.0)


@pytest.mark.parametrize("nside,lmax,nmaps,niter,noise", [
    (16, 31, 3, 3, 0.0),
    (16, 47, 2, 2, 0.2),       # lmax = 3 nside - 1, not band-limited
    (32, 95, 40, 2, 0.0),      # two k-tiles of 32 pairs
    (64, 150, 2, 1, 0.0),      # two l tiles per order
    (5, 14, 2, 3, 0.1),
])
def test_immediate_iteration_spin2_against_oracle(nside, lmax, nmaps, niter, noise):
    """spin 2: E and B of an order are corrected together; (Q, U) residual kept as ring spectra of Q and iU"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 95, 2)
    maps = O.synthesis(nside, lmax, alm_true, spin=2)
    if noise > 0.0:
        maps = maps + inputs.white_noise(nside, np.arange(nmaps), 96, noise, spin=2)
    ref_alm, ref_rms = O.analysis_iter_immediate(nside, lmax, maps, niter, spin=2)
    plan = Plan(nside, lmax, nmaps, 2)
    got_alm, got_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    plan.destroy()
    assert np.isfinite(got_alm).all()
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    assert np.abs(got_rms - ref_rms).max() <= 1e-9 * ref_rms[0].max()


@pytest.mark.parametrize("nside,lmax,nmaps,niter,noise,spin", [
    (64, 127, 3, 2, 0.0, 0),      # lmax = 2 nside - 1: the belt is alias-free, the caps are not
    (64, 127, 70, 1, 0.2, 0),     # two k-tiles, not band-limited
    (64, 100, 2, 3, 0.1, 0),      # the chain ends well before lmax
    (128, 255, 1, 1, 0.0, 0),     # two blocks of 64 alias-free ring pairs, two l tiles
    (128, 150, 3, 1, 0.0, 0),     # the alias-free tail starts inside the caps
    (64, 127, 3, 2, 0.0, 2),      # spin 2: E and B of an order together
    (64, 100, 34, 1, 0.1, 2),     # spin 2, two k-tiles of 32 pairs, not band-limited
    (128, 150, 2, 1, 0.0, 2),     # spin 2, tail inside the caps
])
def test_immediate_hybrid_sweep_against_oracle_and_plain_sweep(nside, lmax, nmaps, niter, noise, spin):
    """the hybrid sweep (include/sht.h, SHT_OPT_ITER_HYBRID: the alias-free ring pairs leave the chain of dependent steps)
    against the oracle's pixel-space sweep, and against the plain sweep of the same plan (equal up to the order of the
    ring sums)"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE, SHT_OPT_ITER_HYBRID, SHT_OPT_ITER_ALIAS_FREE_FROM
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 95, spin)
    maps = O.synthesis(nside, lmax, alm_true, spin=spin)
    if noise > 0.0:
        maps = maps + inputs.white_noise(nside, np.arange(nmaps), 96, noise, spin=spin)
    ref_alm, ref_rms = O.analysis_iter_immediate(nside, lmax, maps, niter, spin=spin)
    plan = Plan(nside, lmax, nmaps, spin)
    pstar = plan.sht_plan_get_option(SHT_OPT_ITER_ALIAS_FREE_FROM)
    assert pstar % 64 == 0 and 0 < pstar <= nside, "this size is meant to take the hybrid sweep (alias-free from %d)" % pstar
    assert plan.sht_plan_get_option(SHT_OPT_ITER_HYBRID) == 1
    l0 = plan.kernel_launches()
    got_alm, got_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    l_hybrid = plan.kernel_launches() - l0
    plan.sht_plan_set_option(SHT_OPT_ITER_HYBRID, 0)
    l0 = plan.kernel_launches()
    plain_alm, plain_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    l_plain = plan.kernel_launches() - l0
    plan.destroy()
    assert np.isfinite(got_alm).all()
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    assert inputs.rel_err(plain_alm, ref_alm) <= TOL
    assert inputs.rel_err(got_alm, plain_alm) <= 1e-12
    assert np.abs(got_rms - ref_rms).max() <= 1e-9 * ref_rms[0].max()
    assert np.abs(got_rms - plain_rms).max() <= 1e-11 * ref_rms[0].max()
    assert l_hybrid != l_plain                                   # the two sweeps really are different launch sequences


@pytest.mark.parametrize("nside,lmax,nmaps,niter,noise", [
    (64, 191, 3, 2, 0.0),      # lmax = 3 nside - 1: every order from nside + 1 on meets its mirror 4 nside - m on the belt
    (64, 150, 70, 1, 0.2),     # two k-tiles, not band-limited
    (64, 129, 2, 3, 0.0),      # the second group is the two orders 2 nside, 2 nside + 1
    (128, 300, 1, 1, 0.0),     # two blocks of belt ring pairs, three l tiles
])
def test_immediate_two_phase_sweep_against_oracle_and_plain_sweep(nside, lmax, nmaps, niter, noise):
    """2 nside <= lmax < 4 nside (spin 0): the belt ring pairs leave the chain of dependent steps in two groups of orders
    (below / from 2 nside), DESIGN.md section 6.  Against the oracle's pixel-space sweep and the plain sweep of the plan."""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan, SHT_ITER_IMMEDIATE, SHT_OPT_ITER_HYBRID, SHT_OPT_ITER_ALIAS_FREE_FROM
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 97)
    maps = O.synthesis(nside, lmax, alm_true)
    if noise > 0.0:
        maps = maps + inputs.white_noise(nside, np.arange(nmaps), 98, noise)
    ref_alm, ref_rms = O.analysis_iter_immediate(nside, lmax, maps, niter)
    plan = Plan(nside, lmax, nmaps, 0)
    assert plan.sht_plan_get_option(SHT_OPT_ITER_ALIAS_FREE_FROM) > nside        # not the one-phase hybrid sweep
    l0 = plan.kernel_launches()
    got_alm, got_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    l_two = plan.kernel_launches() - l0
    plan.sht_plan_set_option(SHT_OPT_ITER_HYBRID, 0)
    l0 = plan.kernel_launches()
    plain_alm, plain_rms = _run(plan, maps, niter, SHT_ITER_IMMEDIATE)
    l_plain = plan.kernel_launches() - l0
    plan.destroy()
    assert l_two != l_plain                                       # the two sweeps really are different launch sequences
    assert np.isfinite(got_alm).all()
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    assert inputs.rel_err(plain_alm, ref_alm) <= TOL
    assert inputs.rel_err(got_alm, plain_alm) <= 1e-12
    assert np.abs(got_rms - ref_rms).max() <= 1e-9 * ref_rms[0].max()
    assert np.abs(got_rms - plain_rms).max() <= 1e-11 * ref_rms[0].max()
