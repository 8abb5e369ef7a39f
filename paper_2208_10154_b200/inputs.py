"""Seeded synthetic inputs shared by the CUDA path's tests/bench and by the oracle's tests.

This module holds NONE of the method's arithmetic (no geometry, no Legendre functions, no transforms):
only NumPy random draws shaped like the paper's workloads (mock CMB skies) and the
table of BASELINE.json configs.  It imports neither the CUDA binding nor the oracle.

Recipe: per map k and component c an independent PCG64 stream
``default_rng([seed, k, c])`` (so any single map can be regenerated on its own, which the full-size
sampled parity tests need); a_lm = sqrt(C_l/2) (g1 + i g2) for m > 0, a_l0 = sqrt(C_l) g1 (real),
g ~ N(0,1) drawn as one (nalm, 2) block in the m-major alm order; C_l = 1/(l(l+1)) for l >= 2,
a_00 = a_1m = 0 (map rms ~ 1).  Spin 2: C_l^EE = C_l, C_l^BB = 0.1 C_l^EE.
"""
import numpy as np

# BASELINE.json "configs", restated.  niter only for the iterative config.
CONFIGS = {
    1: dict(name="cfg1_spin0_nside16", nside=16, lmax=47, nmaps=8, spin=0, seed=1001),
    2: dict(name="cfg2_spin0_nside128", nside=128, lmax=383, nmaps=256, spin=0, seed=2002, noise_sigma=1e-3),
    3: dict(name="cfg3_spin0_nside512_headline", nside=512, lmax=1535, nmaps=1000, spin=0, seed=3003),
    4: dict(name="cfg4_spin2_nside256", nside=256, lmax=767, nmaps=1000, spin=2, seed=4004),
    5: dict(name="cfg5_iter_nside1024", nside=1024, lmax=2047, nmaps=200, spin=0, seed=5005, niter=3),
}


def npix(nside):
    return 12 * nside * nside


def nalm(lmax):
    return (lmax + 1) * (lmax + 2) // 2


def ell_of_index(lmax):
    """l and m of every m-major alm slot: idx(l,m) = m(2 lmax + 1 - m)/2 + l."""
    ms = np.repeat(np.arange(lmax + 1), lmax + 1 - np.arange(lmax + 1))
    starts = np.cumsum(np.concatenate([[0], lmax + 1 - np.arange(lmax)]))
    ls = np.arange(nalm(lmax)) - starts[ms] + ms
    return ls, ms


def power_spectrum(lmax, scale=1.0):
    """C_l = scale / (l (l+1)) for l >= 2, 0 for l < 2."""
    l = np.arange(lmax + 1, dtype=np.float64)
    cl = np.zeros(lmax + 1)
    cl[2:] = scale / (l[2:] * (l[2:] + 1.0))
    return cl


def gaussian_alm(lmax, ks, seed, spin=0):
    """Seeded Gaussian a_lm for the map indices `ks` -> complex128 [len(ks)][ncomp][nalm]."""
    ks = np.atleast_1d(np.asarray(ks, dtype=np.int64))
    ncomp = 2 if spin == 2 else 1
    ls, ms = ell_of_index(lmax)
    out = np.empty((len(ks), ncomp, nalm(lmax)), dtype=np.complex128)
    for c in range(ncomp):
        cl = power_spectrum(lmax, 1.0 if c == 0 else 0.1)
        amp_m0 = np.sqrt(cl[ls])
        amp = np.sqrt(cl[ls] / 2.0)
        for j, k in enumerate(ks):
            g = np.random.default_rng([int(seed), int(k), c]).standard_normal((nalm(lmax), 2))
            a = amp * (g[:, 0] + 1j * g[:, 1])
            a[ms == 0] = amp_m0[ms == 0] * g[ms == 0, 0]
            out[j, c] = a
    return out


def white_noise(nside, ks, seed, sigma, spin=0):
    """Seeded per-pixel white noise for the map indices `ks` -> float64 [len(ks)][ncomp][npix]."""
    ks = np.atleast_1d(np.asarray(ks, dtype=np.int64))
    ncomp = 2 if spin == 2 else 1
    out = np.empty((len(ks), ncomp, npix(nside)))
    for j, k in enumerate(ks):
        for c in range(ncomp):
            out[j, c] = sigma * np.random.default_rng([int(seed), int(k), c, 7]).standard_normal(npix(nside))
    return out


def rel_err(x, ref):
    """Parity metric (reading G22): per map, max|x - ref| / max|ref|; returns the worst map."""
    x = np.asarray(x).reshape(np.asarray(ref).shape[0], -1)
    r = np.asarray(ref).reshape(x.shape)
    den = np.abs(r).max(axis=1)
    den[den == 0] = 1.0
    return float((np.abs(x - r).max(axis=1) / den).max())
