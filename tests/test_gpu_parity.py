"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Tolerance (BASELINE.json north_star; metric = DESIGN.md reading G22): per map
max|x - ref| / max|ref| <= 1e-10 in FP64."""
import numpy as np
import pytest

from paper_2208_10154_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _dev():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch.device("cuda:0")


def _gpu_synthesis(plan, alm):
    import torch
    a = torch.from_numpy(np.ascontiguousarray(alm)).to(_dev())
    maps = torch.full((plan.nmaps, plan.ncomp, plan.npix), float("nan"), dtype=torch.float64, device=_dev())
    plan.sht_synthesis(a, maps)
    torch.cuda.synchronize()
    return maps.cpu().numpy()


def _gpu_analysis(plan, maps):
    import torch
    mp = torch.from_numpy(np.ascontiguousarray(maps)).to(_dev())
    alm = torch.full((plan.nmaps, plan.ncomp, plan.nalm), float("nan"), dtype=torch.complex128, device=_dev())
    plan.sht_analysis(mp, alm)
    torch.cuda.synchronize()
    return alm.cpu().numpy()


@pytest.mark.parametrize("nside,lmax,nmaps", [
    (1, 2, 1), (1, 0, 3), (2, 5, 2), (3, 8, 5), (4, 11, 8), (5, 14, 3), (8, 23, 70), (16, 47, 8),
    (16, 20, 4), (16, 63, 2), (32, 95, 130),
    (48, 143, 5),      # ring lengths 4*37, 4*41, 4*43, 4*47: Bluestein rings
    (160, 64, 3),      # ring lengths 4*121, 4*143: two direct prime stages (out of place), Bluestein up to 4*157
])
def test_spin0_small_full(nside, lmax, nmaps):
    """both directions, every output element; ragged map counts, odd nside, lmax below / above 3 nside - 1"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), seed=100 + nside)
    if lmax < 2:
        alm[:] = np.random.default_rng(1).standard_normal(alm.shape)
    plan = Plan(nside, lmax, nmaps, 0)
    ref_maps = O.synthesis(nside, lmax, alm)
    got_maps = _gpu_synthesis(plan, alm)
    assert inputs.rel_err(got_maps, ref_maps) <= TOL
    noisy = ref_maps + inputs.white_noise(nside, np.arange(nmaps), 7, 1e-3)
    ref_alm = O.analysis(nside, lmax, noisy)
    got_alm = _gpu_analysis(plan, noisy)
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    ls, ms = inputs.ell_of_index(lmax)
    assert np.all(got_alm[:, :, ms == 0].imag == 0.0)
    plan.destroy()


@pytest.mark.parametrize("nside,lmax,nmaps", [
    (1, 2, 1), (2, 5, 3), (3, 8, 5), (4, 11, 33), (8, 23, 40), (16, 47, 8), (16, 30, 4), (16, 63, 2), (32, 95, 70),
    (48, 143, 3), (64, 300, 2),
])
def test_spin2_small_full(nside, lmax, nmaps):
    """spin 2, both directions, every output element (Q,U <-> E,B); ragged pair counts, odd nside, lmax above 3 nside - 1"""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), seed=200 + nside, spin=2)
    plan = Plan(nside, lmax, nmaps, 2)
    ref_maps = O.synthesis(nside, lmax, alm, spin=2)
    got_maps = _gpu_synthesis(plan, alm)
    assert inputs.rel_err(got_maps, ref_maps) <= TOL
    noisy = ref_maps + inputs.white_noise(nside, np.arange(nmaps), 9, 1e-3, spin=2)
    ref_alm = O.analysis(nside, lmax, noisy, spin=2)
    got_alm = _gpu_analysis(plan, noisy)
    assert inputs.rel_err(got_alm, ref_alm) <= TOL
    ls, ms = inputs.ell_of_index(lmax)
    assert np.all(got_alm[:, :, ms == 0].imag == 0.0)
    assert np.all(got_alm[:, :, ls < 2] == 0.0)
    plan.destroy()


def test_spin2_ignores_low_l_and_im_m0_on_input():
    """l < 2 and Im(a_l0) are ignored on input (readings G13, section 1), even if they hold NaN"""
    from paper_2208_10154_b200.binding import Plan
    nside, lmax, nmaps = 8, 23, 5
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), seed=31, spin=2)
    plan = Plan(nside, lmax, nmaps, 2)
    base = _gpu_synthesis(plan, alm)
    ls, ms = inputs.ell_of_index(lmax)
    dirty = alm.copy()
    dirty[:, :, ls < 2] = np.nan
    dirty[:, :, ms == 0] = dirty[:, :, ms == 0].real + 1j * 5.0
    dirty[:, :, ls < 2] = np.nan
    assert np.array_equal(_gpu_synthesis(plan, dirty), base)
    plan.destroy()


@pytest.mark.parametrize("nside,lmax,nmaps", [(4, 11, 3), (16, 47, 40), (32, 95, 33), (48, 143, 2)])
@pytest.mark.parametrize("which", [1, 2])
def test_spin2_e_only_b_only(nside, lmax, nmaps, which):
    """item 9: transforms of a^E or a^B alone against the oracle (synthesis with the other component
    zero; the chosen component of the full analysis)"""
    import torch
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    c = which - 1
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), seed=300 + nside, spin=2)
    one = np.ascontiguousarray(alm[:, c, :])
    zeroed = np.zeros_like(alm)
    zeroed[:, c, :] = one
    ref_maps = O.synthesis(nside, lmax, zeroed, spin=2)
    plan = Plan(nside, lmax, nmaps, 2)
    dev = _dev()
    maps = torch.full((nmaps, 2, plan.npix), float("nan"), dtype=torch.float64, device=dev)
    plan.sht_synthesis_pol(torch.from_numpy(one).to(dev), maps, which)
    torch.cuda.synchronize()
    assert inputs.rel_err(maps.cpu().numpy(), ref_maps) <= TOL
    # analysis: a general (Q,U) input with both E and B power
    qu = O.synthesis(nside, lmax, alm, spin=2) + inputs.white_noise(nside, np.arange(nmaps), 5, 1e-3, spin=2)
    ref_alm = O.analysis(nside, lmax, qu, spin=2)[:, c, :]
    got = torch.full((nmaps, plan.nalm), float("nan"), dtype=torch.complex128, device=dev)
    plan.sht_analysis_pol(torch.from_numpy(qu).to(dev), got, which)
    torch.cuda.synchronize()
    assert inputs.rel_err(got.cpu().numpy(), ref_alm) <= TOL
    # the full transform is untouched by the single-component calls
    assert inputs.rel_err(_gpu_synthesis(plan, alm), O.synthesis(nside, lmax, alm, spin=2)) <= TOL
    plan.destroy()


@pytest.mark.parametrize("lmax,rows", [(0, 1), (1, 2), (2, 3), (47, 16), (383, 5), (1535, 2)])
def test_alm_pack_a7(lmax, rows):
    """eq. A7 converters: bit-exact against the oracle's entry-by-entry packing, and round trip"""
    import torch
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import sht_alm_pack_a7, sht_alm_unpack_a7
    n = O.nalm(lmax)
    rng = np.random.default_rng(lmax)
    alm = rng.standard_normal((rows, n)) + 1j * rng.standard_normal((rows, n))
    dev = _dev()
    d_alm = torch.from_numpy(alm).to(dev)
    d_sq = torch.full((rows, lmax + 1, lmax + 1), float("nan"), dtype=torch.float64, device=dev)
    sht_alm_pack_a7(lmax, rows, d_alm, d_sq)
    torch.cuda.synchronize()
    ref = O.pack_a7(lmax, alm)
    assert np.array_equal(d_sq.cpu().numpy(), ref)                 # every cell written, bit-exact
    d_back = torch.full((rows, n), float("nan"), dtype=torch.complex128, device=dev)
    sht_alm_unpack_a7(lmax, rows, d_sq, d_back)
    torch.cuda.synchronize()
    assert np.array_equal(d_back.cpu().numpy(), O.unpack_a7(lmax, ref))


def test_config1():
    """BASELINE.json configs[0]: nside 16, lmax 47, 8 maps: synthesise, analyse back, compare both."""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    c = inputs.CONFIGS[1]
    alm = inputs.gaussian_alm(c["lmax"], np.arange(c["nmaps"]), c["seed"])
    plan = Plan(c["nside"], c["lmax"], c["nmaps"], 0)
    ref_maps = O.synthesis(c["nside"], c["lmax"], alm)
    assert inputs.rel_err(_gpu_synthesis(plan, alm), ref_maps) <= TOL
    assert inputs.rel_err(_gpu_analysis(plan, ref_maps), O.analysis(c["nside"], c["lmax"], ref_maps)) <= TOL
    plan.destroy()


def test_config2_sampled_maps():
    """BASELINE.json configs[1]: nside 128, lmax 383, 256 maps, white noise sigma 1e-3 added after synthesis.
    All 256 maps go through the GPU; 8 of them are compared against the oracle in full."""
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    c = inputs.CONFIGS[2]
    nside, lmax, nmaps = c["nside"], c["lmax"], c["nmaps"]
    ks = np.array([0, 1, 2, 3, 127, 128, 254, 255])
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), c["seed"])
    plan = Plan(nside, lmax, nmaps, 0)
    got_maps = _gpu_synthesis(plan, alm)
    ref_maps = O.synthesis(nside, lmax, alm[ks])
    assert inputs.rel_err(got_maps[ks], ref_maps) <= TOL
    # analysis input: oracle-synthesised maps + white noise for the sampled maps, seeded noise elsewhere
    maps_in = inputs.white_noise(nside, np.arange(nmaps), c["seed"], 1.0)
    maps_in[ks] = ref_maps + inputs.white_noise(nside, ks, c["seed"], c["noise_sigma"])
    got_alm = _gpu_analysis(plan, maps_in)
    ref_alm = O.analysis(nside, lmax, maps_in[ks])
    assert inputs.rel_err(got_alm[ks], ref_alm) <= TOL
    plan.destroy()


@pytest.mark.parametrize("spin", [0, 2])
def test_internal_map_chunks_match_single_chunk(spin):
    """a workspace limit forces internal chunks of 64 maps (ragged last chunk); results must be bit-identical"""
    import torch
    from paper_2208_10154_b200.binding import Plan
    nside, lmax, nmaps, niter = 16, 47, 150, 2
    ncomp = 2 if spin == 2 else 1
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), 11, spin)
    full = Plan(nside, lmax, nmaps, spin)
    per_map = 2 * nside * (lmax + 1) * ncomp * 2 * 16
    small = Plan(nside, lmax, nmaps, spin, workspace_limit=70 * per_map)
    assert full.chunk_maps() == nmaps and small.chunk_maps() == 64
    m_full, m_small = _gpu_synthesis(full, alm), _gpu_synthesis(small, alm)
    assert np.array_equal(m_full, m_small)
    assert np.array_equal(_gpu_analysis(full, m_full), _gpu_analysis(small, m_full))
    mp = torch.from_numpy(m_full).to(_dev())
    outs = []
    for plan in (full, small):
        a = torch.zeros((nmaps, ncomp, plan.nalm), dtype=torch.complex128, device=_dev())
        rms = torch.zeros((niter, nmaps * ncomp), dtype=torch.float64, device=_dev())
        plan.sht_analysis_iter(mp, a, niter, rms)
        torch.cuda.synchronize()
        outs.append((a.cpu().numpy(), rms.cpu().numpy()))
    assert np.array_equal(outs[0][0], outs[1][0])
    # the per-map sum of squares is reduced with atomics: equal up to the summation order
    assert np.allclose(outs[0][1], outs[1][1], rtol=1e-12, atol=0.0)
    full.destroy()
    small.destroy()


def test_host_entries_match_device_entries():
    import torch
    from paper_2208_10154_b200.binding import Plan
    nside, lmax, nmaps = 16, 47, 200
    alm = inputs.gaussian_alm(lmax, np.arange(nmaps), 5)
    plan = Plan(nside, lmax, nmaps, 0)
    dev_maps = _gpu_synthesis(plan, alm)
    host_maps = np.full_like(dev_maps, np.nan)
    plan.sht_synthesis_host(np.ascontiguousarray(alm), host_maps)
    assert np.array_equal(host_maps, dev_maps)
    dev_alm = _gpu_analysis(plan, dev_maps)
    host_alm = np.full_like(dev_alm, np.nan)
    plan.sht_analysis_host(dev_maps, host_alm)
    assert np.array_equal(host_alm, dev_alm)
    plan.destroy()


@pytest.mark.parametrize("nside,lmax,nmaps,niter,spin", [
    (16, 31, 5, 3, 0), (16, 47, 3, 2, 0), (64, 127, 6, 3, 0), (16, 31, 3, 3, 2), (32, 95, 2, 2, 2), (8, 15, 2, 0, 0),
])
def test_iterative_analysis_small(nside, lmax, nmaps, niter, spin):
    """Alg. 2 against the oracle's pixel-space iteration, element by element, with the per-round residual rms"""
    import torch
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    ncomp = 2 if spin == 2 else 1
    alm_true = inputs.gaussian_alm(lmax, np.arange(nmaps), 77, spin)
    maps = O.synthesis(nside, lmax, alm_true, spin=spin)
    ref_alm, ref_rms = O.analysis_iter(nside, lmax, maps, niter, spin=spin)
    plan = Plan(nside, lmax, nmaps, spin)
    mp = torch.from_numpy(maps).to(_dev())
    alm = torch.zeros((nmaps, ncomp, plan.nalm), dtype=torch.complex128, device=_dev())
    rms = torch.zeros((max(niter, 1), nmaps * ncomp), dtype=torch.float64, device=_dev())
    plan.sht_analysis_iter(mp, alm, niter, rms)
    torch.cuda.synchronize()
    assert inputs.rel_err(alm.cpu().numpy(), ref_alm) <= TOL
    # rms falls by orders of magnitude per round: compare relative to the first residual
    if niter > 0:
        assert np.abs(rms.cpu().numpy()[:niter] - ref_rms).max() <= 1e-9 * ref_rms[0].max()
    plan.destroy()
