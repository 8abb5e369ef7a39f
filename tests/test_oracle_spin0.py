"""Pins for the oracle's spin-0 analysis (O3) and synthesis (O4).  CPU only."""
import os

import numpy as np
import pytest
from scipy.special import sph_harm_y

from oracle import oracle as O
from paper_2208_10154_b200 import inputs
from tests.helpers import pix2ang_ring, ylm_matrix, full_alm

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "nside1_worked_values.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            k, v = line.split("=")
            GOLD[k.strip()] = float(v)


def test_phi0_convention_pin():
    """G3: nside 1, a_22 = 1 -> rings 1,3 vanish, ring 2 = (+c,-c,+c,-c), c = 2 sqrt(15/32 pi)."""
    lmax = 2
    alm = np.zeros((1, 1, O.nalm(lmax)), complex)
    alm[0, 0, O.alm_index(lmax, 2, 2)] = 1.0
    mp = O.synthesis(1, lmax, alm)[0, 0]
    c = GOLD["synth_a22_ring2_first_pixel"]
    assert c == pytest.approx(2 * np.sqrt(15 / (32 * np.pi)), rel=1e-15)
    assert np.allclose(mp, [0, 0, 0, 0, c, -c, c, -c, 0, 0, 0, 0], atol=1e-15)


def test_nside1_a20_roundtrip_worked_values():
    """G4: no ring weights -> analysis(synthesis(a_20 = 1)) gives a_20 = 55/108, a_00 = -sqrt(5)/18."""
    lmax = 2
    alm = np.zeros((1, 1, O.nalm(lmax)), complex)
    alm[0, 0, O.alm_index(lmax, 2, 0)] = 1.0
    mp = O.synthesis(1, lmax, alm)
    assert np.allclose(mp[0, 0, 0:4], GOLD["synth_a20_ring1"], atol=1e-13)
    assert np.allclose(mp[0, 0, 4:8], GOLD["synth_a20_ring2"], atol=1e-13)
    assert np.allclose(mp[0, 0, 8:12], GOLD["synth_a20_ring3"], atol=1e-13)
    a = O.analysis(1, lmax, mp)[0, 0]
    assert a[O.alm_index(lmax, 2, 0)] == pytest.approx(55 / 108, abs=1e-15)
    assert a[O.alm_index(lmax, 0, 0)] == pytest.approx(-np.sqrt(5) / 18, abs=1e-15)
    assert GOLD["analysis_a20"] == pytest.approx(55 / 108) and GOLD["analysis_a00"] == pytest.approx(-np.sqrt(5) / 18)


@pytest.mark.parametrize("nside,lmax", [(2, 5), (4, 11), (16, 47)])
def test_constant_map(nside, lmax):
    c = 2.5
    a = O.analysis(nside, lmax, np.full((1, 1, 12 * nside * nside), c))[0, 0]
    assert a[0] == pytest.approx(np.sqrt(4 * np.pi) * c, rel=1e-14)
    ls, ms = inputs.ell_of_index(lmax)
    assert np.abs(a[ms % 4 != 0]).max() < 1e-14                # 4-fold symmetry of every ring
    assert np.all(a[ms == 0].imag == 0.0)


@pytest.mark.parametrize("nside,lmax", [(3, 8), (4, 11), (5, 14), (8, 23), (16, 47)])
def test_analysis_vs_brute_force(nside, lmax):
    """O0: a_lm = dsigma sum_pix T(p) conj(Y_lm(p)) with scipy's Y_lm on per-pixel angles."""
    theta, phi = pix2ang_ring(nside)
    Y = ylm_matrix(lmax, theta, phi)
    rng = np.random.default_rng(11 + nside)
    maps = rng.standard_normal((3, 1, 12 * nside * nside))
    ref = (4 * np.pi / (12 * nside * nside)) * maps[:, 0, :] @ np.conj(Y).T
    got = O.analysis(nside, lmax, maps)[:, 0, :]
    ls, ms = inputs.ell_of_index(lmax)
    ref[:, ms == 0] = ref[:, ms == 0].real
    assert np.abs(got - ref).max() / np.abs(ref).max() < 2e-13


@pytest.mark.parametrize("nside,lmax", [(3, 8), (4, 11), (8, 23), (16, 47)])
def test_synthesis_vs_brute_force(nside, lmax):
    """O0: T(p) = sum_{l, -l<=m<=l} a_lm Y_lm(p), the full complex sum with a_{l,-m} = (-1)^m conj(a_lm)."""
    theta, phi = pix2ang_ring(nside)
    alm = inputs.gaussian_alm(lmax, [0, 1], seed=5 + nside)
    got = O.synthesis(nside, lmax, alm)[:, 0, :]
    for k in range(2):
        fa = full_alm(lmax, alm[k, 0])
        ref = np.zeros(len(theta), complex)
        for (l, m), a in fa.items():
            ref += a * sph_harm_y(l, m, theta, phi)
        assert np.abs(ref.imag).max() < 1e-12
        assert np.abs(got[k] - ref.real).max() / np.abs(ref.real).max() < 2e-13


@pytest.mark.parametrize("l,m", [(0, 0), (1, 0), (5, 3), (20, 20), (47, 1), (47, 46), (40, 17)])
def test_single_lm_synthesis_is_ylm(l, m):
    """a_lm = 1 -> map = w_m Re Y_lm at every pixel, including l far above N_r/2 of the polar rings."""
    nside, lmax = 8, 47
    theta, phi = pix2ang_ring(nside)
    alm = np.zeros((1, 1, O.nalm(lmax)), complex)
    alm[0, 0, O.alm_index(lmax, l, m)] = 1.0
    got = O.synthesis(nside, lmax, alm)[0, 0]
    ref = (1.0 if m == 0 else 2.0) * sph_harm_y(l, m, theta, phi).real
    assert np.abs(got - ref).max() < 5e-13


def test_im_al0_ignored_and_linearity():
    nside, lmax = 4, 11
    alm = inputs.gaussian_alm(lmax, [0, 1], seed=3)
    alm2 = alm.copy()
    ls, ms = inputs.ell_of_index(lmax)
    alm2[:, :, ms == 0] += 0.37j
    assert np.array_equal(O.synthesis(nside, lmax, alm), O.synthesis(nside, lmax, alm2))
    rng = np.random.default_rng(2)
    t = rng.standard_normal((2, 1, 12 * nside * nside))
    comb = 0.3 * t[0:1] - 1.7 * t[1:2]
    a = O.analysis(nside, lmax, t); ac = O.analysis(nside, lmax, comb)
    assert np.abs(ac[0] - (0.3 * a[0] - 1.7 * a[1])).max() < 1e-14
    s = O.synthesis(nside, lmax, alm); sc = O.synthesis(nside, lmax, 0.3 * alm[0:1] - 1.7 * alm[1:2])
    assert np.abs(sc[0] - (0.3 * s[0] - 1.7 * s[1])).max() < 1e-13


def test_partial_m_and_ring_lists_match_full():
    nside, lmax = 8, 23
    alm = inputs.gaussian_alm(lmax, [0, 1, 2], seed=9)
    full = O.synthesis(nside, lmax, alm)
    part = O.synthesis(nside, lmax, alm, rlist=[1, 5, 16, 31])
    for r in (1, 5, 16, 31):
        n, s, _, _ = O.ring_info(nside, r)
        assert np.array_equal(part[:, :, s:s + n], full[:, :, s:s + n])
    a_full = O.analysis(nside, lmax, full)
    a_part = O.analysis(nside, lmax, full, mlist=[0, 3, 23])
    ls, ms = inputs.ell_of_index(lmax)
    sel = np.isin(ms, [0, 3, 23])
    assert np.array_equal(a_part[:, :, sel], a_full[:, :, sel]) and np.all(a_part[:, :, ~sel] == 0)
