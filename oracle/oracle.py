"""ctypes binding of the CPU oracle (oracle/sht_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
``--impl reference`` legs of bench.py.  Nothing here imports, links or reads the CUDA library.
Argument marshalling only -- all arithmetic is in the C file, which cites PAPER.md passage by passage -- with two
exceptions written here in numpy on top of the C transforms: the eq. A7 packed format (pack_a7 / unpack_a7, pinned by
tests/test_oracle_a7.py) and Alg. 3's sweep over the orders m (analysis_iter_immediate, pinned by
tests/test_oracle_immediate.py against a dense block-triangular solve).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sht_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force=False):
    """Compile sht_oracle.c with gcc (long double x87 arithmetic, OpenMP over m / rings)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        c_int, c_ll, c_dp, c_ip = ctypes.c_int, ctypes.c_longlong, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        _lib.oracle_npix.restype = c_ll
        _lib.oracle_nalm.restype = c_ll
        _lib.oracle_alm_index.restype = c_ll
        _lib.oracle_ring_info.argtypes = [c_int, c_int, ctypes.POINTER(c_ll), ctypes.POINTER(c_ll), c_dp, c_dp]
        _lib.oracle_lambda.argtypes = [c_int, c_int, ctypes.c_double, c_dp]
        _lib.oracle_lambda_ring.argtypes = [c_int, c_int, c_int, c_int, c_dp, c_ip]
        _lib.oracle_spin2_x.argtypes = [c_int, c_int, ctypes.c_double, c_dp, c_dp]
        _lib.oracle_analysis.argtypes = [c_int, c_int, c_int, c_int, c_dp, c_dp, c_ip, c_int]
        _lib.oracle_synthesis.argtypes = [c_int, c_int, c_int, c_int, c_dp, c_dp, c_ip, c_int]
        _lib.oracle_analysis_iter.argtypes = [c_int, c_int, c_int, c_int, c_dp, c_dp, c_int, c_dp]
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ip(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def num_threads():
    return int(lib().oracle_num_threads())


def npix(nside):
    return 12 * nside * nside


def nalm(lmax):
    return (lmax + 1) * (lmax + 2) // 2


def alm_index(lmax, l, m):
    return int(lib().oracle_alm_index(lmax, l, m))


def ring_info(nside, i):
    """ring i (1-based, north to south) -> (npix_ring, first_pixel, z, phi0)"""
    n, s = ctypes.c_longlong(), ctypes.c_longlong()
    z, p = ctypes.c_double(), ctypes.c_double()
    lib().oracle_ring_info(nside, i, ctypes.byref(n), ctypes.byref(s), ctypes.byref(z), ctypes.byref(p))
    return int(n.value), int(s.value), float(z.value), float(p.value)


def lambda_lm(lmax, m, z):
    """lambda_lm(z) for l = m..lmax (array of lmax-m+1 doubles)"""
    out = np.zeros(lmax - m + 1)
    lib().oracle_lambda(lmax, m, float(z), _dp(out))
    return out


def lambda_ring(nside, iring, lmax, m):
    """lambda_lm on ring iring as (mantissa, exponent) arrays: value = mant * 2**expo"""
    mant = np.zeros(lmax - m + 1)
    expo = np.zeros(lmax - m + 1, dtype=np.int32)
    lib().oracle_lambda_ring(nside, iring, lmax, m, _dp(mant), _ip(expo))
    return mant, expo


def spin2_x(lmax, m, z):
    """X1_lm(z), X2_lm(z) for l = m..lmax"""
    x1 = np.zeros(lmax - m + 1)
    x2 = np.zeros(lmax - m + 1)
    lib().oracle_spin2_x(lmax, m, float(z), _dp(x1), _dp(x2))
    return x1, x2


def _ncomp(spin):
    if spin not in (0, 2):
        raise ValueError("spin must be 0 or 2")
    return 2 if spin == 2 else 1


def analysis(nside, lmax, maps, spin=0, mlist=None, out=None):
    """maps [nmaps][ncomp][npix] -> alm complex128 [nmaps][ncomp][nalm].
    mlist: only these m are computed (other entries keep the value of `out`, zeros if out is None)."""
    nc = _ncomp(spin)
    maps = np.ascontiguousarray(maps, dtype=np.float64).reshape(-1, nc, npix(nside))
    nm = maps.shape[0]
    alm = np.zeros((nm, nc, nalm(lmax)), dtype=np.complex128) if out is None else out
    assert alm.flags.c_contiguous and alm.dtype == np.complex128
    if mlist is None:
        lib().oracle_analysis(nside, lmax, nm, spin, _dp(maps), _dp(alm.view(np.float64)), None, 0)
    else:
        ml = np.ascontiguousarray(mlist, dtype=np.int32)
        lib().oracle_analysis(nside, lmax, nm, spin, _dp(maps), _dp(alm.view(np.float64)), _ip(ml), len(ml))
    return alm


def synthesis(nside, lmax, alm, spin=0, rlist=None, out=None):
    """alm complex128 [nmaps][ncomp][nalm] -> maps [nmaps][ncomp][npix].
    rlist: only these rings (1-based) are computed (other pixels keep the value of `out`)."""
    nc = _ncomp(spin)
    alm = np.ascontiguousarray(alm, dtype=np.complex128).reshape(-1, nc, nalm(lmax))
    nm = alm.shape[0]
    maps = np.zeros((nm, nc, npix(nside))) if out is None else out
    assert maps.flags.c_contiguous and maps.dtype == np.float64
    if rlist is None:
        lib().oracle_synthesis(nside, lmax, nm, spin, _dp(alm.view(np.float64)), _dp(maps), None, 0)
    else:
        rl = np.ascontiguousarray(rlist, dtype=np.int32)
        lib().oracle_synthesis(nside, lmax, nm, spin, _dp(alm.view(np.float64)), _dp(maps), _ip(rl), len(rl))
    return maps


def analysis_iter(nside, lmax, maps, niter, spin=0):
    """Alg. 2 (Jacobi). Returns (alm, resid_rms[niter][nmaps*ncomp])."""
    nc = _ncomp(spin)
    maps = np.ascontiguousarray(maps, dtype=np.float64).reshape(-1, nc, npix(nside))
    nm = maps.shape[0]
    alm = np.zeros((nm, nc, nalm(lmax)), dtype=np.complex128)
    rms = np.zeros((max(niter, 1), nm * nc))
    lib().oracle_analysis_iter(nside, lmax, nm, spin, _dp(maps), _dp(alm.view(np.float64)), niter, _dp(rms))
    return alm, rms[:niter]


def analysis_iter_immediate(nside, lmax, maps, niter, spin=0):
    """Alg. 3, the "immediate" iteration, in the reading DESIGN.md lists as G21: a Gauss-Seidel
    sweep over the orders m.  a^0 = analysis(map) and r = map - synthesis(a^0); then, niter times, for m = 0 .. lmax in
    this order: delta a_m = the order-m part of analysis(r) (line 13, P . T remapped from the *current* F), a_m += delta
    a_m, and r -= synthesis(delta a_m) at once (lines 8-9, "update F from delta T_m"), so that the orders that follow
    see, through the ring aliasing, the corrections already made.  Written out on the pixels with the single-order
    analysis and the plain synthesis of this oracle; no ring-spectrum shortcuts.
    Returns (alm, resid_rms[niter][nmaps*ncomp]): the rms of r at the start of each sweep."""
    nc = _ncomp(spin)
    maps = np.ascontiguousarray(maps, dtype=np.float64).reshape(-1, nc, npix(nside))
    nm = maps.shape[0]
    alm = analysis(nside, lmax, maps, spin)
    rms = np.zeros((niter, nm * nc))
    if niter == 0:
        return alm, rms
    res = maps - synthesis(nside, lmax, alm, spin)
    for it in range(niter):
        rms[it] = np.sqrt(np.mean(res * res, axis=2)).reshape(-1)
        for m in range(lmax + 1):
            da = analysis(nside, lmax, res, spin, mlist=[m])
            alm += da
            res -= synthesis(nside, lmax, da, spin)
    return alm, rms


def pack_a7(lmax, alm):
    """eq. A7, written out entry by entry: alm complex128 [rows][nalm] (m-major) ->
    real squares [rows][lmax+1][lmax+1] with Re a_lm at (l, m) and Im a_lm (m >= 1) at (l - m, lmax - m + 1)."""
    alm = np.asarray(alm, dtype=np.complex128).reshape(-1, nalm(lmax))
    sq = np.zeros((alm.shape[0], lmax + 1, lmax + 1))
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            i = m * (2 * lmax + 1 - m) // 2 + l
            sq[:, l, m] = alm[:, i].real
            if m >= 1:
                sq[:, l - m, lmax - m + 1] = alm[:, i].imag
    return sq


def unpack_a7(lmax, sq):
    """inverse of pack_a7; Im a_l0 is not stored and comes back as 0"""
    sq = np.asarray(sq, dtype=np.float64).reshape(-1, lmax + 1, lmax + 1)
    alm = np.zeros((sq.shape[0], nalm(lmax)), dtype=np.complex128)
    for m in range(lmax + 1):
        for l in range(m, lmax + 1):
            i = m * (2 * lmax + 1 - m) // 2 + l
            alm[:, i] = sq[:, l, m] + (1j * sq[:, l - m, lmax - m + 1] if m >= 1 else 0.0)
    return alm
