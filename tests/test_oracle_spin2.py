"""Pins for the oracle's spin-2 functions and transforms (O5).  CPU only."""
from math import pi, sqrt

import numpy as np
import pytest
from scipy.special import sph_harm_y

from oracle import oracle as O
from paper_2208_10154_b200 import inputs
from tests.helpers import pix2ang_ring, sYlm, sYlm_mp, full_alm


def test_helper_sylm_is_pinned():
    """The independent reference itself: s = 0 reduces to scipy's Y_lm; l = 2 closed forms (Z&S)."""
    th = np.array([0.3, 0.9, 2.2]); ph = 0.4
    for l, m in [(0, 0), (1, 1), (2, 1), (3, -2), (5, 3), (7, -7)]:
        assert np.allclose(sYlm(0, l, m, th, ph), sph_harm_y(l, m, th, ph), rtol=1e-13)
    x = np.cos(th)
    assert np.allclose(sYlm(2, 2, 2, th, ph), sqrt(5 / (64 * pi)) * (1 - x) ** 2 * np.exp(2j * ph), rtol=1e-13)
    assert np.allclose(sYlm(-2, 2, 2, th, ph), sqrt(5 / (64 * pi)) * (1 + x) ** 2 * np.exp(2j * ph), rtol=1e-13)


def test_x1_x2_closed_forms_l2():
    for z in (-0.7, 0.0, 0.31, 0.95):
        x1, x2 = O.spin2_x(2, 2, z)
        assert x1[0] == pytest.approx(sqrt(5 / (64 * pi)) * (1 + z * z), rel=1e-14)
        assert x2[0] == pytest.approx(-sqrt(5 / (64 * pi)) * 2 * z, rel=1e-14, abs=1e-17)


@pytest.mark.parametrize("m", [0, 1, 2, 3, 8, 15])
def test_x1_x2_vs_spin_weighted_harmonics(m):
    """X1 = (+2Y + -2Y)/2, X2 = (+2Y - -2Y)/2 at phi = 0 (PAPER.md:449 eq. A5 with F+- = -X1,2)."""
    lmax = 40
    for th in (0.2, 1.1, 2.5):
        x1, x2 = O.spin2_x(lmax, m, np.cos(th))
        for l in range(max(m, 2), lmax + 1):
            p = sYlm_mp(2, l, m, th); q = sYlm_mp(-2, l, m, th)        # F+- are real
            assert x1[l - m] == pytest.approx((p + q) / 2, rel=1e-12, abs=1e-15)
            assert x2[l - m] == pytest.approx((p - q) / 2, rel=1e-12, abs=1e-15)
        if m < 2:
            assert np.all(x1[:2 - m] == 0) and np.all(x2[:2 - m] == 0)


def test_x1_x2_parity_and_m0():
    lmax = 60
    for m in (0, 1, 2, 9):
        l = np.arange(m, lmax + 1)
        a1, a2 = O.spin2_x(lmax, m, 0.37); b1, b2 = O.spin2_x(lmax, m, -0.37)
        sgn = (-1.0) ** (l + m)
        assert np.allclose(b1, sgn * a1, rtol=1e-12, atol=1e-300)
        assert np.allclose(b2, -sgn * a2, rtol=1e-12, atol=1e-300)
        if m == 0:
            assert np.all(a2 == 0)


def _brute_synthesis(nside, lmax, ae, ab):
    """Q +- iU = sum_{l,m} a_{+-2,lm} +-2Y_lm (eq. 8), a_{+-2} = -(a_E +- i a_B) (eq. 10)."""
    theta, phi = pix2ang_ring(nside)
    fe, fb = full_alm(lmax, ae), full_alm(lmax, ab)
    P = np.zeros(len(theta), complex); M = np.zeros(len(theta), complex)
    for (l, m), e in fe.items():
        if l < 2:
            continue
        b = fb[(l, m)]
        P += -(e + 1j * b) * sYlm(2, l, m, theta, phi)
        M += -(e - 1j * b) * sYlm(-2, l, m, theta, phi)
    Q = (P + M) / 2; U = (P - M) / 2j
    assert np.abs(Q.imag).max() < 1e-12 and np.abs(U.imag).max() < 1e-12
    return Q.real, U.real


@pytest.mark.parametrize("nside,lmax", [(2, 5), (4, 11), (3, 8)])
def test_spin2_synthesis_vs_brute_force(nside, lmax):
    alm = inputs.gaussian_alm(lmax, [0], seed=21 + nside, spin=2)
    got = O.synthesis(nside, lmax, alm, spin=2)[0]
    Q, U = _brute_synthesis(nside, lmax, alm[0, 0], alm[0, 1])
    assert np.abs(got[0] - Q).max() < 5e-13 and np.abs(got[1] - U).max() < 5e-13


@pytest.mark.parametrize("nside,lmax", [(2, 5), (4, 11), (3, 8)])
def test_spin2_analysis_vs_brute_force(nside, lmax):
    """a_{+-2,lm} = dsigma sum_p (Q +- iU)(p) conj(+-2Y_lm(p)); a_E = -(a_2 + a_-2)/2, a_B = i(a_2 - a_-2)/2
    (eq. 10)."""
    theta, phi = pix2ang_ring(nside)
    rng = np.random.default_rng(31 + nside)
    qu = rng.standard_normal((1, 2, 12 * nside * nside))
    got = O.analysis(nside, lmax, qu, spin=2)[0]
    ds = 4 * pi / (12 * nside * nside)
    P = qu[0, 0] + 1j * qu[0, 1]; M = qu[0, 0] - 1j * qu[0, 1]
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            i = O.alm_index(lmax, l, m)
            if l < 2:
                assert got[0, i] == 0 and got[1, i] == 0
                continue
            a2 = ds * np.sum(P * np.conj(sYlm(2, l, m, theta, phi)))
            am2 = ds * np.sum(M * np.conj(sYlm(-2, l, m, theta, phi)))
            e = -(a2 + am2) / 2; b = 1j * (a2 - am2) / 2
            if m == 0:
                e, b = e.real, b.real
            assert abs(got[0, i] - e) < 5e-14 and abs(got[1, i] - b) < 5e-14


def test_pure_e_and_m0_structure():
    nside, lmax = 4, 11
    alm = inputs.gaussian_alm(lmax, [0], seed=77, spin=2)
    ls, ms = inputs.ell_of_index(lmax)
    only_m0 = alm.copy(); only_m0[:, :, ms != 0] = 0
    e_only = only_m0.copy(); e_only[:, 1] = 0
    b_only = only_m0.copy(); b_only[:, 0] = 0
    qe = O.synthesis(nside, lmax, e_only, spin=2)[0]; qb = O.synthesis(nside, lmax, b_only, spin=2)[0]
    assert np.abs(qe[1]).max() < 1e-15 and np.abs(qb[0]).max() < 1e-15     # m = 0: X2 = 0
    assert np.abs(qe[0]).max() > 1e-3 and np.abs(qb[1]).max() > 1e-3
