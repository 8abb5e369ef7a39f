"""FP32 storage at the ABI (include/sht.h: sht_*_f32, sht_*_host_f32; NEXT row N4, north_star's optional FP32 path with
its tolerance 1e-4): float32 maps / complex64 a_lm in the caller's memory, FP64 arithmetic inside.  Against the oracle on
the same single-precision inputs (widened exactly): the only difference is the rounding of the output, so besides the
north_star bound the tests hold the entries to a few single-precision ulps of the largest value."""
import numpy as np
import pytest

from paper_2208_10154_b200 import inputs

pytestmark = pytest.mark.gpu
TOL_F32 = 1e-4            # BASELINE.json north_star: "<= 1e-4 for an optional FP32 path"
ULP = 2.0 ** -23          # what the path really does: one rounding of each output to float32 (relative 6e-8), with margin


@pytest.mark.parametrize("nside,lmax,nmaps,spin", [
    (8, 23, 3, 0), (16, 47, 70, 0), (32, 64, 130, 0), (48, 100, 5, 0), (16, 47, 66, 2), (32, 95, 5, 2),
])
def test_f32_storage_against_oracle(nside, lmax, nmaps, spin):
    import torch
    from oracle import oracle as O
    from paper_2208_10154_b200.binding import Plan
    dev = torch.device("cuda:0")
    ncomp = 2 if spin == 2 else 1
    alm64 = inputs.gaussian_alm(lmax, np.arange(nmaps), 500 + nside, spin)
    alm32 = alm64.astype(np.complex64)                                    # what a single-precision caller holds
    ref_maps = O.synthesis(nside, lmax, alm32.astype(np.complex128), spin=spin)
    plan = Plan(nside, lmax, nmaps, spin)
    d_alm = torch.from_numpy(alm32).to(dev)
    d_maps = torch.full((nmaps, ncomp, plan.npix), float("nan"), dtype=torch.float32, device=dev)
    plan.sht_synthesis_f32(d_alm, d_maps)
    torch.cuda.synchronize()
    got_maps = d_maps.cpu().numpy()
    assert got_maps.dtype == np.float32 and np.isfinite(got_maps).all()
    e = inputs.rel_err(got_maps.astype(np.float64), ref_maps)
    assert e <= TOL_F32 and e <= 2 * ULP, e
    # analysis of single-precision maps (the synthesised ones plus noise, so that they are not band-limited)
    maps32 = (ref_maps + inputs.white_noise(nside, np.arange(nmaps), 7, 1e-2, spin=spin)).astype(np.float32)
    ref_alm = O.analysis(nside, lmax, maps32.astype(np.float64), spin=spin)
    d_in = torch.from_numpy(maps32).to(dev)
    d_out = torch.full((nmaps, ncomp, plan.nalm), float("nan"), dtype=torch.complex64, device=dev)
    plan.sht_analysis_f32(d_in, d_out)
    torch.cuda.synchronize()
    got_alm = d_out.cpu().numpy()
    assert got_alm.dtype == np.complex64 and np.isfinite(got_alm).all()
    e = inputs.rel_err(got_alm.astype(np.complex128), ref_alm)
    assert e <= TOL_F32 and e <= 2 * ULP, e
    assert np.array_equal(d_in.cpu().numpy(), maps32)                     # inputs are not modified
    # host entries: the same numbers as the device entries, bit for bit (same kernels, same chunks)
    h_alm = np.full((nmaps, ncomp, plan.nalm), np.nan, dtype=np.complex64)
    plan.sht_analysis_host_f32(maps32, h_alm)
    assert np.array_equal(h_alm, got_alm)
    h_maps = np.full((nmaps, ncomp, plan.npix), np.nan, dtype=np.float32)
    plan.sht_synthesis_host_f32(alm32, h_maps)
    assert np.array_equal(h_maps, got_maps)
    # and equal to the FP64 entries' results rounded once
    d_alm64 = torch.from_numpy(alm32.astype(np.complex128)).to(dev)
    d_maps64 = torch.empty((nmaps, ncomp, plan.npix), dtype=torch.float64, device=dev)
    plan.sht_synthesis(d_alm64, d_maps64)
    torch.cuda.synchronize()
    assert np.array_equal(d_maps64.cpu().numpy().astype(np.float32), got_maps)
    plan.destroy()


def test_f32_host_entries_repeat_and_mix_with_f64():
    """the single-precision host entries share the chunk streams and staging of the FP64 host entries: calls of both kinds
    in a row on one plan give their own results again"""
    import torch
    from paper_2208_10154_b200.binding import Plan
    nside, lmax, nmaps = 32, 95, 200
    plan = Plan(nside, lmax, nmaps, 0)
    alm64 = inputs.gaussian_alm(lmax, np.arange(nmaps), 77)
    alm32 = alm64.astype(np.complex64)
    m32a = np.empty((nmaps, 1, plan.npix), dtype=np.float32)
    m64 = np.empty((nmaps, 1, plan.npix), dtype=np.float64)
    m32b = np.empty_like(m32a)
    plan.sht_synthesis_host_f32(alm32, m32a)
    plan.sht_synthesis_host(alm32.astype(np.complex128), m64)
    plan.sht_synthesis_host_f32(alm32, m32b)
    assert np.array_equal(m32a, m32b)
    assert np.array_equal(m64.astype(np.float32), m32a)
    a32 = np.empty((nmaps, 1, plan.nalm), dtype=np.complex64)
    a64 = np.empty((nmaps, 1, plan.nalm), dtype=np.complex128)
    plan.sht_analysis_host_f32(m32a, a32)
    plan.sht_analysis_host(m32a.astype(np.float64), a64)
    assert np.array_equal(a64.astype(np.complex64), a32)
    plan.destroy()
