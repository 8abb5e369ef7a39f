"""Independent references used to pin the oracle ("one level below the oracle").

Nothing here is shared with oracle/ or with the CUDA path: the pixel geometry is retyped from the
HEALPix paper's RING formulas (Gorski et al. 2005, the pixelisation PAPER.md:211 names), Y_lm comes from
scipy.special.sph_harm_y (a library routine), spin-weighted harmonics from the explicit finite sum of
Goldberg et al. (1967), itself pinned in tests/test_oracle_spin2.py against scipy (s = 0) and the l = 2
closed forms.
"""
from math import comb, factorial, pi, sqrt

import numpy as np
from scipy.special import sph_harm_y


def pix2ang_ring(nside):
    """theta, phi of every pixel of the RING scheme, from the per-pixel formulas (not ring tables)."""
    npix = 12 * nside * nside
    ncap = 2 * nside * (nside - 1)
    p = np.arange(npix)
    theta = np.empty(npix)
    phi = np.empty(npix)
    # north cap
    q = p[p < ncap]
    ph = (q + 1) / 2.0
    i = np.floor(np.sqrt(ph - np.sqrt(np.floor(ph)))).astype(int) + 1
    j = q + 1 - 2 * i * (i - 1)
    theta[q] = np.arccos(1.0 - i * i / (3.0 * nside * nside))
    phi[q] = (j - 0.5) * pi / (2.0 * i)
    # belt
    q = p[(p >= ncap) & (p < npix - ncap)]
    ip = q - ncap
    i = ip // (4 * nside) + nside
    j = ip % (4 * nside) + 1
    fodd = 0.5 * (1 + (i + nside) % 2)
    theta[q] = np.arccos((2 * nside - i) * 2.0 / (3.0 * nside))
    phi[q] = (j - fodd) * pi / (2.0 * nside)
    # south cap
    q = p[p >= npix - ncap]
    ip = npix - q
    ph = ip / 2.0
    i = np.floor(np.sqrt(ph - np.sqrt(np.floor(ph)))).astype(int) + 1
    j = 4 * i + 1 - (ip - 2 * i * (i - 1))
    theta[q] = np.arccos(-1.0 + i * i / (3.0 * nside * nside))
    phi[q] = (j - 0.5) * pi / (2.0 * i)
    return theta, phi


def ylm_matrix(lmax, theta, phi):
    """Y[idx(l,m), pixel] for m >= 0 in the m-major alm order, from scipy."""
    rows = []
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            rows.append(sph_harm_y(l, m, theta, phi))
    return np.array(rows)


def sYlm(s, l, m, theta, phi):
    """Spin-weighted spherical harmonic, explicit finite sum (Goldberg et al. 1967)."""
    theta = np.asarray(theta, dtype=np.float64)
    pref = (-1) ** (l + m - s) * sqrt(
        factorial(l + m) * factorial(l - m) * (2 * l + 1) / (4 * pi * factorial(l + s) * factorial(l - s)))
    tot = np.zeros_like(theta)
    cot = np.cos(theta / 2) / np.sin(theta / 2)
    for r in range(0, l - s + 1):
        k = r + s - m
        if k < 0 or k > l + s:
            continue
        tot = tot + (-1) ** r * comb(l - s, r) * comb(l + s, k) * cot ** (2 * r + s - m)
    return pref * np.sin(theta / 2) ** (2 * l) * tot * np.exp(1j * m * phi)


def full_alm(lmax, alm_mpos):
    """dict (l,m) -> a_lm for -l <= m <= l from the m >= 0 half, a_{l,-m} = (-1)^m conj(a_lm)."""
    out = {}
    idx = 0
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            a = alm_mpos[idx]
            idx += 1
            if m == 0:
                out[(l, 0)] = complex(a.real, 0.0)
            else:
                out[(l, m)] = a
                out[(l, -m)] = (-1) ** m * np.conj(a)
    return out


def sYlm_mp(s, l, m, theta, dps=40):
    """Same finite sum at phi = 0 in mpmath (the alternating sum cancels badly in float64 for l >~ 15)."""
    import mpmath
    with mpmath.workdps(dps):
        th = mpmath.mpf(theta)
        pref = (-1) ** (l + m - s) * mpmath.sqrt(
            mpmath.factorial(l + m) * mpmath.factorial(l - m) * (2 * l + 1)
            / (4 * mpmath.pi * mpmath.factorial(l + s) * mpmath.factorial(l - s)))
        cot = mpmath.cos(th / 2) / mpmath.sin(th / 2)
        tot = mpmath.mpf(0)
        for r in range(0, l - s + 1):
            k = r + s - m
            if k < 0 or k > l + s:
                continue
            tot += (-1) ** r * mpmath.binomial(l - s, r) * mpmath.binomial(l + s, k) * cot ** (2 * r + s - m)
        return float(pref * mpmath.sin(th / 2) ** (2 * l) * tot)
