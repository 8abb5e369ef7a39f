"""sht_eb_split_static (include/sht.h): the entry point that allocates nothing -- its a_lm scratch is a file-scope
`__device__` array of the library (SHT_EB_STATIC_MAX_BYTES) instead of a stream-ordered allocation.  Checked against the
existing path, sht_eb_split, on the same seeded inputs: two calls in a row on one stream, with different inputs,
components and plan sizes, so that the second call finds the first call's contents in the shared array.

This file is named to be collected last (the suite runs with pytest -x); it passes alone in a fresh process (where the
static call is the first CUDA work of the library) and after the other tests."""
import numpy as np
import pytest

from paper_2208_10154_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = 1e-10          # the parity tolerance of tests/test_gpu_parity.py (the two paths run the same kernels: equal bit for bit)


def _qu_maps(nside, nmaps, seed):
    """seeded (Q,U) maps with power in both families on every scale (white noise: not band-limited)"""
    return inputs.white_noise(nside, np.arange(nmaps), seed, 1.0, spin=2)


def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    from paper_2208_10154_b200.binding import Plan, SHT_POL_E, SHT_POL_B
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dev = torch.device("cuda:0")
    nside, lmax, nmaps = 32, 95, 33
    plan = Plan(nside, lmax, nmaps, 2)
    qa, qb = _qu_maps(nside, nmaps, 71), _qu_maps(nside, nmaps, 72)
    d_a, d_b = torch.from_numpy(qa).to(dev), torch.from_numpy(qb).to(dev)
    s1, s2 = torch.full_like(d_a, float("nan")), torch.full_like(d_b, float("nan"))
    # the static path first (in a fresh process this is the library's first device work), twice, no synchronisation between
    plan.sht_eb_split_static(d_a, s1, SHT_POL_E)
    plan.sht_eb_split_static(d_b, s2, SHT_POL_B)
    torch.cuda.synchronize()
    r1, r2 = torch.full_like(d_a, float("nan")), torch.full_like(d_b, float("nan"))
    plan.sht_eb_split(d_a, r1, SHT_POL_E)
    plan.sht_eb_split(d_b, r2, SHT_POL_B)
    torch.cuda.synchronize()
    for got, ref in ((s1, r1), (s2, r2)):
        g, r = got.cpu().numpy(), ref.cpu().numpy()
        assert np.isfinite(r).all() and np.abs(r).max() > 0
        assert inputs.rel_err(g, r) <= TOL
        assert np.array_equal(g, r)
    assert np.array_equal(d_a.cpu().numpy(), qa) and np.array_equal(d_b.cpu().numpy(), qb)     # inputs not modified

    # a smaller plan next: its scratch region is a prefix of what the calls above left behind in the shared array
    nside2, lmax2, nmaps2 = 16, 40, 70
    plan2 = Plan(nside2, lmax2, nmaps2, 2)
    qc = _qu_maps(nside2, nmaps2, 73)
    d_c = torch.from_numpy(qc).to(dev)
    s3, s4, r3 = torch.full_like(d_c, float("nan")), torch.full_like(d_c, float("nan")), torch.full_like(d_c, float("nan"))
    plan2.sht_eb_split_static(d_c, s3, SHT_POL_B)
    plan2.sht_eb_split_static(s3, s4, SHT_POL_B)                     # the split of the split, fed from the first call's output
    torch.cuda.synchronize()
    # the same two calls again, now that every kernel they launch is loaded: the device's free memory must not move
    free0 = torch.cuda.mem_get_info(dev)[0]
    plan2.sht_eb_split_static(d_c, s3, SHT_POL_B)
    plan2.sht_eb_split_static(s3, s4, SHT_POL_B)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info(dev)[0]
    plan2.sht_eb_split(d_c, r3, SHT_POL_B)
    r4 = torch.full_like(d_c, float("nan"))
    plan2.sht_eb_split(r3, r4, SHT_POL_B)
    torch.cuda.synchronize()
    assert np.array_equal(s3.cpu().numpy(), r3.cpu().numpy()) and np.array_equal(s4.cpu().numpy(), r4.cpu().numpy())
    assert inputs.rel_err(s4.cpu().numpy(), r4.cpu().numpy()) <= TOL
    # in place, as sht_eb_split allows
    plan2.sht_eb_split_static(d_c, d_c, SHT_POL_B)
    torch.cuda.synchronize()
    assert np.array_equal(d_c.cpu().numpy(), r3.cpu().numpy())
    # and the first plan again after the smaller one
    s5 = torch.full_like(d_a, float("nan"))
    plan.sht_eb_split_static(d_a, s5, SHT_POL_E)
    torch.cuda.synchronize()
    assert np.array_equal(s5.cpu().numpy(), r1.cpu().numpy())
    # the repeated static calls of plan2 left the device's free memory where it was (weak check: the code has no allocating call)
    assert free1 == free0, "free device memory changed across sht_eb_split_static: %d -> %d" % (free0, free1)
    plan.destroy()
    plan2.destroy()


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    import torch
    from paper_2208_10154_b200.binding import Plan, ShtError, SHT_POL_E, SHT_EB_STATIC_MAX_BYTES
    dev = torch.device("cuda:0")
    nside, lmax, nmaps = 64, 191, 128
    plan = Plan(nside, lmax, nmaps, 2)
    need = plan.chunk_maps() * plan.nalm * 16
    assert need > SHT_EB_STATIC_MAX_BYTES                               # 128 pairs x 18528 a_lm x 16 B = 37.9 MB > 32 MiB
    d_in = torch.from_numpy(_qu_maps(nside, nmaps, 74)).to(dev)
    out = torch.full_like(d_in, float("nan"))
    with pytest.raises(ShtError) as ei:
        plan.sht_eb_split_static(d_in, out, SHT_POL_E)
    msg = str(ei.value)
    assert "invalid argument" in msg and "SHT_EB_STATIC_MAX_BYTES" in msg and str(need) in msg
    torch.cuda.synchronize()
    assert bool(torch.isnan(out).all())                                 # nothing was launched
    plan.sht_eb_split(d_in, out, SHT_POL_E)                             # the allocating path takes the same plan
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())
    # a spin-0 plan is refused like sht_eb_split refuses it
    p0 = Plan(8, 23, 2, 0)
    x = torch.zeros((2, 1, p0.npix), dtype=torch.float64, device=dev)
    with pytest.raises(ShtError):
        p0.sht_eb_split_static(x, x, SHT_POL_E)
    plan.destroy()
    p0.destroy()
