"""Pins for the oracle's Alg. 3 ("immediate" iteration; reading G21 in DESIGN.md).

The oracle runs the sweep as a loop over m on the pixels.  Here the same iteration is written as linear algebra on tiny
grids: with A (analysis) and S (synthesis) as dense real matrices -- built column by column from the oracle's plain
transforms, which have their own pins -- one Gauss-Seidel sweep over the order blocks is the block-triangular solve
    delta = (I + L)^-1 A r,   L = strictly block-lower part of A S (blocks = orders m, in increasing m),
followed by a += delta, r -= S delta.  A loop that used the old residual (Jacobi), swept the orders in another order,
dropped the in-place update or had the wrong sign fails the comparison."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2208_10154_b200 import inputs


def _real_basis(lmax, ncomp):
    """real parametrisation of the a_lm: (component, slot, part) with part 0 = Re, 1 = Im (m >= 1 only), and the order m"""
    ls, ms = inputs.ell_of_index(lmax)
    basis, order = [], []
    for c in range(ncomp):
        for i in range(len(ls)):
            basis.append((c, i, 0)); order.append(ms[i])
            if ms[i] > 0:
                basis.append((c, i, 1)); order.append(ms[i])
    return basis, np.array(order)


def _dense(nside, lmax, spin):
    ncomp = 2 if spin == 2 else 1
    npix, nalm = O.npix(nside), O.nalm(lmax)
    basis, order = _real_basis(lmax, ncomp)
    nb = len(basis)
    unit = np.zeros((nb, ncomp, nalm), dtype=np.complex128)
    for j, (c, i, part) in enumerate(basis):
        unit[j, c, i] = 1.0 if part == 0 else 1.0j
    S = O.synthesis(nside, lmax, unit, spin=spin).reshape(nb, ncomp * npix).T.copy()          # (ncomp npix) x nb
    alm = O.analysis(nside, lmax, np.eye(ncomp * npix).reshape(ncomp * npix, ncomp, npix), spin=spin)
    A = np.empty((nb, ncomp * npix))
    for j, (c, i, part) in enumerate(basis):
        A[j] = alm[:, c, i].real if part == 0 else alm[:, c, i].imag
    return A, S, basis, order


def _to_complex(x, basis, ncomp, nalm):
    a = np.zeros((ncomp, nalm), dtype=np.complex128)
    for j, (c, i, part) in enumerate(basis):
        a[c, i] += x[j] if part == 0 else 1j * x[j]
    return a


@pytest.mark.parametrize("nside,lmax,spin", [(2, 5, 0), (2, 7, 0), (4, 11, 0), (2, 5, 2), (4, 9, 2)])
def test_immediate_equals_block_triangular_solve(nside, lmax, spin):
    ncomp = 2 if spin == 2 else 1
    A, S, basis, order = _dense(nside, lmax, spin)
    nb = len(basis)
    M = A @ S
    L = np.where(order[:, None] > order[None, :], M, 0.0)             # rows of order m, columns of the orders before it
    rng = np.random.default_rng(42)
    maps = rng.standard_normal((2, ncomp, O.npix(nside)))
    niter = 3
    got, rms = O.analysis_iter_immediate(nside, lmax, maps, niter, spin=spin)
    jac, _ = O.analysis_iter(nside, lmax, maps, niter, spin=spin)
    for k in range(2):
        x = A @ maps[k].reshape(-1)
        r = maps[k].reshape(-1) - S @ x
        rr = []
        for _ in range(niter):
            rr.append(np.sqrt(np.mean(r.reshape(ncomp, -1) ** 2, axis=1)))
            delta = np.linalg.solve(np.eye(nb) + L, A @ r)
            x = x + delta
            r = r - S @ delta
        ref = _to_complex(x, basis, ncomp, O.nalm(lmax))
        scale = np.abs(ref).max()
        assert np.abs(got[k] - ref).max() <= 1e-12 * scale
        assert np.allclose(rms[:, k * ncomp:(k + 1) * ncomp], np.array(rr), rtol=1e-11, atol=0)
        # the pin can tell the two schemes apart on this grid (polar rings alias heavily)
        assert np.abs(jac[k] - ref).max() > 1e-6 * scale


def test_immediate_zero_rounds_is_plain_analysis():
    nside, lmax = 4, 9
    maps = np.random.default_rng(1).standard_normal((2, 1, O.npix(nside)))
    a, rms = O.analysis_iter_immediate(nside, lmax, maps, 0)
    assert rms.shape == (0, 2)
    assert np.array_equal(a, O.analysis(nside, lmax, maps))


def test_immediate_fixed_point_band_limited():
    """a band-limited map (lmax <= 2 nside - 1) is reproduced: the sweeps converge to the a_lm it was made from, and the
    residual rms falls every round (the paper: both schemes give negligible errors there)"""
    nside, lmax = 8, 15
    alm = inputs.gaussian_alm(lmax, np.arange(2), 7)
    maps = O.synthesis(nside, lmax, alm)
    a3, rms = O.analysis_iter_immediate(nside, lmax, maps, 3)
    a0 = O.analysis(nside, lmax, maps)
    e0 = np.abs(a0 - alm).max()
    e3 = np.abs(a3 - alm).max()
    assert e3 < 1e-2 * e0
    assert np.all(rms[1:] < 0.5 * rms[:-1])
