"""Pins of the oracle's eq. A7 packing: the hand-worked lmax = 2 layout, and the bijection of
{Re a_lm} u {Im a_lm, m >= 1} onto the (lmax+1)^2 square (Re fills l >= m, Im the strict upper triangle)."""
import os

import numpy as np
import pytest

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "a7_lmax2_layout.txt")


def test_a7_hand_worked_layout_lmax2():
    lmax = 2
    rows = [ln.strip() for ln in open(GOLD) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 3
    alm = np.zeros((1, O.nalm(lmax)), dtype=np.complex128)
    tag = {}
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            i = O.alm_index(lmax, l, m)
            alm[0, i] = (100 + 10 * l + m) + 1j * (200 + 10 * l + m)
            tag[("R", l, m)] = 100 + 10 * l + m
            tag[("I", l, m)] = 200 + 10 * l + m
    sq = O.pack_a7(lmax, alm)[0]
    for r, line in enumerate(rows):
        for c, cell in enumerate(line.split("|")):
            kind, l, m = cell.split()
            assert sq[r, c] == tag[(kind, int(l), int(m))], (r, c, cell)


@pytest.mark.parametrize("lmax", [0, 1, 2, 7, 40])
def test_a7_is_a_bijection_and_roundtrips(lmax):
    n = O.nalm(lmax)
    rng = np.random.default_rng(lmax)
    alm = rng.standard_normal((3, n)) + 1j * rng.standard_normal((3, n))
    m0 = np.array([O.alm_index(lmax, l, 0) for l in range(lmax + 1)])
    alm[:, m0] = alm[:, m0].real                      # Im a_l0 = 0 is not stored
    sq = O.pack_a7(lmax, alm)
    # every cell of the square is written exactly once: the multiset of cells equals the multiset of stored reals
    stored = np.concatenate([alm.real.ravel(), np.delete(alm.imag, m0, axis=1).ravel()])
    assert sq.size == stored.size == 3 * (lmax + 1) ** 2
    assert np.array_equal(np.sort(sq.ravel()), np.sort(stored))
    # Re fills the lower triangle (l >= m), Im the strict upper triangle
    for l in range(lmax + 1):
        for m in range(l + 1):
            assert np.array_equal(sq[:, l, m], alm[:, O.alm_index(lmax, l, m)].real)
    assert np.array_equal(O.unpack_a7(lmax, sq), alm)
