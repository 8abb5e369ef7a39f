"""Pins for the oracle's geometry (O1) and normalised Legendre functions (O2).  CPU only."""
import os

import mpmath
import numpy as np
import pytest
from scipy.special import sph_harm_y

from oracle import oracle as O
from tests.helpers import pix2ang_ring


@pytest.mark.parametrize("nside", [1, 2, 3, 4, 5, 16, 128])
def test_geometry_invariants(nside):
    nr = 4 * nside - 1
    info = [O.ring_info(nside, i) for i in range(1, nr + 1)]
    n = np.array([r[0] for r in info]); start = np.array([r[1] for r in info])
    z = np.array([r[2] for r in info]); phi0 = np.array([r[3] for r in info])
    assert n.sum() == 12 * nside * nside                       # N_pix = 12 nside^2
    assert np.all(start == np.concatenate([[0], np.cumsum(n)[:-1]]))
    assert abs((n * z).sum()) < 1e-9                           # sum over pixels of z = 0
    assert np.all(n == n[::-1]) and np.allclose(phi0, phi0[::-1], atol=0) and np.allclose(z, -z[::-1], atol=0)
    assert z[0] == pytest.approx(1 - 1 / (3 * nside ** 2), abs=3e-16)
    assert np.all(np.diff(z) < 0)
    # caps: N = 4i; belt: N = 4 nside
    for i in range(1, nside):
        assert n[i - 1] == 4 * i and phi0[i - 1] == pytest.approx(np.pi / (4 * i), rel=1e-15)
    assert np.all(n[nside - 1:3 * nside] == 4 * nside)


@pytest.mark.parametrize("nside", [1, 2, 3, 8])
def test_geometry_matches_per_pixel_formulas(nside):
    theta, phi = pix2ang_ring(nside)
    for i in range(1, 4 * nside):
        n, s, z, p0 = O.ring_info(nside, i)
        assert np.allclose(np.cos(theta[s:s + n]), z, atol=2e-16)
        assert np.allclose(phi[s:s + n], p0 + 2 * np.pi * np.arange(n) / n, atol=1e-14)


def test_geometry_nside1():
    r = [O.ring_info(1, i) for i in (1, 2, 3)]
    assert [x[0] for x in r] == [4, 4, 4]
    assert np.allclose([x[2] for x in r], [2 / 3, 0, -2 / 3], atol=3e-16)
    assert np.allclose([x[3] for x in r], [np.pi / 4, 0, np.pi / 4], atol=1e-16)


def _dfact_ratio(m):                     # (2m-1)!!/(2m)!!
    r = 1.0
    for j in range(1, m + 1):
        r *= (2 * j - 1) / (2 * j)
    return r


@pytest.mark.parametrize("m", [0, 1, 2, 5, 20, 47])
def test_lambda_seeds_closed_form(m):
    for z in (0.3, -0.8, 0.999):
        s = np.sqrt((1 - z) * (1 + z))
        lam = O.lambda_lm(m + 1, m, z)
        lmm = (-1) ** m * np.sqrt((2 * m + 1) / (4 * np.pi) * _dfact_ratio(m)) * s ** m
        assert lam[0] == pytest.approx(lmm, rel=1e-14)
        assert lam[1] == pytest.approx(z * np.sqrt(2 * m + 3) * lmm, rel=1e-14)


def test_lambda_poles_and_parity():
    lmax = 200
    l = np.arange(lmax + 1)
    assert np.allclose(O.lambda_lm(lmax, 0, 1.0), np.sqrt((2 * l + 1) / (4 * np.pi)), rtol=1e-13)
    assert np.allclose(O.lambda_lm(lmax, 0, -1.0), (-1.0) ** l * np.sqrt((2 * l + 1) / (4 * np.pi)), rtol=1e-13)
    for m in (0, 1, 2, 7, 60):
        for z in (0.1, 0.77):
            a = O.lambda_lm(lmax, m, z); b = O.lambda_lm(lmax, m, -z)
            sgn = (-1.0) ** (np.arange(m, lmax + 1) + m)
            assert np.allclose(b, sgn * a, rtol=1e-13, atol=1e-300)


def test_lambda_addition_theorem():
    lmax = 150
    for z in (0.0, 0.5, -0.93):
        tot = np.zeros(lmax + 1)
        for m in range(lmax + 1):
            lam = O.lambda_lm(lmax, m, z)
            tot[m:] += (1.0 if m == 0 else 2.0) * lam ** 2
        assert np.allclose(tot, (2 * np.arange(lmax + 1) + 1) / (4 * np.pi), rtol=1e-12)


@pytest.mark.parametrize("m", [0, 1, 3, 17, 64, 100])
def test_lambda_vs_scipy(m):
    lmax = 100
    for th in (0.05, 0.7, 1.5707963, 2.9):
        lam = O.lambda_lm(lmax, m, np.cos(th))
        ref = np.array([sph_harm_y(l, m, th, 0.0).real for l in range(m, lmax + 1)])
        assert np.allclose(lam, ref, rtol=1e-11, atol=1e-13)


def test_lambda_high_l_vs_mpmath():
    """l up to 2047 against mpmath at 50 digits (a handful of cells)."""
    mpmath.mp.dps = 50
    for (l, m, z) in [(1535, 0, 0.3), (1535, 700, 0.1), (2047, 1500, -0.2), (1000, 999, 0.05)]:
        lam = O.lambda_lm(l, m, z)[-1]
        zz = mpmath.mpf(z)
        ref = mpmath.sqrt((2 * l + 1) / (4 * mpmath.pi) * mpmath.factorial(l - m) / mpmath.factorial(l + m)) \
            * mpmath.legenp(l, m, zz, type=2)
        assert float(abs(lam - ref) / abs(ref)) < 1e-11


def test_lambda_extended_range_nside1024():
    """Paper item 11: above nside 512 the seed sin^m(theta) underflows a 64-bit float
    although the ring matters.  Cell located with the oracle itself, values checked against mpmath:
    nside=1024, m=600, ring 325 has a seed ~1e-354 yet lambda_lm reaches ~1e-12 before l = 2047."""
    nside, m, lmax, ring = 1024, 600, 2047, 325
    mant, expo = O.lambda_ring(nside, ring, lmax, m)
    log10 = np.log10(np.abs(mant)) + expo * np.log10(2.0)
    assert log10[0] < -307                                     # seed not representable as a normal double
    assert log10.max() > -20                                   # but the ring matters
    # cross-check the seed and one high-l cell against mpmath
    mpmath.mp.dps = 60
    z = 1 - mpmath.mpf(ring * ring) / (3 * nside * nside)
    s = mpmath.sqrt((1 - z) * (1 + z))
    seed = (-1) ** m * mpmath.sqrt((2 * m + 1) / (4 * mpmath.pi) * mpmath.rf(mpmath.mpf(1) / 2, m) / mpmath.factorial(m)) * s ** m
    got = mpmath.mpf(float(mant[0])) * mpmath.mpf(2) ** int(expo[0])
    assert abs(got - seed) / abs(seed) < 1e-13
    l = 2047
    ref = mpmath.sqrt((2 * l + 1) / (4 * mpmath.pi) * mpmath.factorial(l - m) / mpmath.factorial(l + m)) \
        * mpmath.legenp(l, m, z, type=2)
    got = mpmath.mpf(float(mant[l - m])) * mpmath.mpf(2) ** int(expo[l - m])
    assert abs(got - ref) / abs(ref) < 1e-10
