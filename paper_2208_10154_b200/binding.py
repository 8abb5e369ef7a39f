"""Thin Python binding of the C ABI in include/sht.h (same names; argument marshalling only).

Every step of the transform runs in the CUDA kernels of libsht_b200.so.  PyTorch is used by callers only
for device buffers and streams.  There is no CPU fallback: if the library has not been built this module
raises on import (build it with ``python -m paper_2208_10154_b200.build`` or ``__graft_entry__.build()``).
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsht_b200.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "paper_2208_10154_b200: CUDA library %s is missing; run `python -m paper_2208_10154_b200.build`. "
        "There is no CPU fallback." % LIB_PATH)

_lib = ctypes.CDLL(LIB_PATH)

SHT_OK = 0
SHT_POL_E, SHT_POL_B = 1, 2
SHT_EB_STATIC_MAX_BYTES = 32 << 20         # include/sht.h: static a_lm scratch of sht_eb_split_static
SHT_LAMBDA_FUSED, SHT_LAMBDA_STAGED = 0, 1
SHT_ITER_TM, SHT_ITER_PIXEL, SHT_ITER_IMMEDIATE = 0, 1, 2
SHT_OPT_RING_PATH, SHT_OPT_LEG_TILES_PER_CTA, SHT_OPT_LEG_RING_SPLIT, SHT_OPT_ITER_HYBRID, SHT_OPT_ITER_ALIAS_FREE_FROM = 0, 1, 2, 3, 4
_vp, _i, _ll, _d = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_double

_lib.sht_plan_create.argtypes = [ctypes.POINTER(_vp), _i, _i, _i, _i]
_lib.sht_plan_create.restype = _i
_lib.sht_plan_create_ex.argtypes = [ctypes.POINTER(_vp), _i, _i, _i, _i, ctypes.c_size_t]
_lib.sht_plan_create_ex.restype = _i
_lib.sht_plan_destroy.argtypes = [_vp]
_lib.sht_plan_destroy.restype = _i
_lib.sht_analysis.argtypes = [_vp, _vp, _vp, _vp]
_lib.sht_analysis.restype = _i
_lib.sht_synthesis.argtypes = [_vp, _vp, _vp, _vp]
_lib.sht_synthesis.restype = _i
_lib.sht_analysis_pol.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.sht_analysis_pol.restype = _i
_lib.sht_synthesis_pol.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.sht_synthesis_pol.restype = _i
_lib.sht_alm_pack_a7.argtypes = [_i, _ll, _vp, _vp, _vp]
_lib.sht_alm_pack_a7.restype = _i
_lib.sht_alm_unpack_a7.argtypes = [_i, _ll, _vp, _vp, _vp]
_lib.sht_alm_unpack_a7.restype = _i
_lib.sht_plan_set_iter_mode.argtypes = [_vp, _i]
_lib.sht_plan_set_iter_mode.restype = _i
_lib.sht_plan_set_lambda_mode.argtypes = [_vp, _i]
_lib.sht_plan_set_lambda_mode.restype = _i
_lib.sht_plan_lambda_mode.argtypes = [_vp]
_lib.sht_plan_lambda_mode.restype = _i
_lib.sht_plan_set_option.argtypes = [_vp, _i, _i]
_lib.sht_plan_set_option.restype = _i
_lib.sht_plan_get_option.argtypes = [_vp, _i]
_lib.sht_plan_get_option.restype = _i
_lib.sht_plan_reserve_iter.argtypes = [_vp]
_lib.sht_plan_reserve_iter.restype = _i
_lib.sht_eb_split.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.sht_eb_split.restype = _i
_lib.sht_eb_split_static.argtypes = [_vp, _vp, _vp, _i, _vp]
_lib.sht_eb_split_static.restype = _i
_lib.sht_analysis_iter.argtypes = [_vp, _vp, _vp, _i, _vp, _vp]
_lib.sht_analysis_iter.restype = _i
_lib.sht_analysis_host.argtypes = [_vp, _vp, _vp]
_lib.sht_analysis_host.restype = _i
_lib.sht_synthesis_host.argtypes = [_vp, _vp, _vp]
_lib.sht_synthesis_host.restype = _i
for _n in ("sht_analysis_f32", "sht_synthesis_f32"):
    getattr(_lib, _n).argtypes = [_vp, _vp, _vp, _vp]
    getattr(_lib, _n).restype = _i
for _n in ("sht_analysis_host_f32", "sht_synthesis_host_f32"):
    getattr(_lib, _n).argtypes = [_vp, _vp, _vp]
    getattr(_lib, _n).restype = _i
_lib.sht_npix.argtypes = [_i]
_lib.sht_npix.restype = _ll
_lib.sht_nalm.argtypes = [_i]
_lib.sht_nalm.restype = _ll
_lib.sht_alm_index.argtypes = [_i, _i, _i]
_lib.sht_alm_index.restype = _ll
_lib.sht_plan_workspace_bytes.argtypes = [_vp]
_lib.sht_plan_workspace_bytes.restype = ctypes.c_size_t
_lib.sht_plan_executed_flops.argtypes = [_vp, _i]
_lib.sht_plan_executed_flops.restype = _d
_lib.sht_plan_chunk_maps.argtypes = [_vp]
_lib.sht_plan_chunk_maps.restype = _i
_lib.sht_plan_kernel_launches.argtypes = [_vp]
_lib.sht_plan_kernel_launches.restype = _ll
_lib.sht_status_string.argtypes = [_i]
_lib.sht_status_string.restype = ctypes.c_char_p
_lib.sht_last_error.argtypes = [_vp]
_lib.sht_last_error.restype = ctypes.c_char_p
_lib.sht_plan_set_timing.argtypes = [_vp, _i]
_lib.sht_plan_set_timing.restype = _i
_lib.sht_plan_stage_ms.argtypes = [_vp, ctypes.POINTER(_d), ctypes.POINTER(_i)]
_lib.sht_plan_stage_ms.restype = _i
_lib.sht_measure_fp64_mma_peak.argtypes = [_d]
_lib.sht_measure_fp64_mma_peak.restype = _d

EXPORTED = [
    "sht_plan_create", "sht_plan_create_ex", "sht_plan_destroy", "sht_analysis", "sht_synthesis", "sht_analysis_iter", "sht_analysis_pol", "sht_synthesis_pol", "sht_alm_pack_a7", "sht_alm_unpack_a7", "sht_plan_set_lambda_mode", "sht_plan_lambda_mode", "sht_plan_set_iter_mode", "sht_plan_reserve_iter", "sht_eb_split", "sht_eb_split_static", "sht_plan_set_option", "sht_plan_get_option",
    "sht_analysis_host", "sht_synthesis_host", "sht_analysis_f32", "sht_synthesis_f32", "sht_analysis_host_f32", "sht_synthesis_host_f32", "sht_npix", "sht_nalm", "sht_alm_index",
    "sht_plan_workspace_bytes", "sht_plan_chunk_maps", "sht_plan_executed_flops", "sht_plan_kernel_launches", "sht_status_string",
    "sht_last_error", "sht_measure_fp64_mma_peak", "sht_plan_set_timing", "sht_plan_stage_ms",
]


class ShtError(RuntimeError):
    pass


def sht_npix(nside):
    return int(_lib.sht_npix(nside))


def sht_nalm(lmax):
    return int(_lib.sht_nalm(lmax))


def sht_alm_index(lmax, l, m):
    return int(_lib.sht_alm_index(lmax, l, m))


def sht_status_string(status):
    return _lib.sht_status_string(status).decode()


def sht_measure_fp64_mma_peak(ms=200.0):
    return float(_lib.sht_measure_fp64_mma_peak(ms))


def sht_alm_pack_a7(lmax, rows, alm, packed, stream=None):
    st = _lib.sht_alm_pack_a7(lmax, rows, _ptr(alm), _ptr(packed), _stream(stream))
    if st != SHT_OK:
        raise ShtError("sht_alm_pack_a7: %s" % sht_status_string(st))


def sht_alm_unpack_a7(lmax, rows, packed, alm, stream=None):
    st = _lib.sht_alm_unpack_a7(lmax, rows, _ptr(packed), _ptr(alm), _stream(stream))
    if st != SHT_OK:
        raise ShtError("sht_alm_unpack_a7: %s" % sht_status_string(st))


def _ptr(t):
    """device / host pointer of a torch tensor or numpy array (must be contiguous float64 / complex128)."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        if not t.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return ctypes.c_void_p(t.data_ptr())
    if not t.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be C-contiguous")
    return ctypes.c_void_p(t.ctypes.data)


def _stream(stream):
    if stream is None:
        return None
    return ctypes.c_void_p(getattr(stream, "cuda_stream", stream))


class Plan:
    """sht_plan_create / sht_plan_destroy with the transform entries as methods (same names as the ABI)."""

    def __init__(self, nside, lmax, nmaps, spin=0, workspace_limit=0):
        self._h = ctypes.c_void_p()
        st = _lib.sht_plan_create_ex(ctypes.byref(self._h), nside, lmax, nmaps, spin, workspace_limit)
        if st != SHT_OK:
            self._h = None
            raise ShtError("sht_plan_create(%d,%d,%d,%d): %s" % (nside, lmax, nmaps, spin, sht_status_string(st)))
        self.nside, self.lmax, self.nmaps, self.spin = nside, lmax, nmaps, spin
        self.ncomp = 2 if spin == 2 else 1
        self.npix, self.nalm = sht_npix(nside), sht_nalm(lmax)

    def _check(self, st, what):
        if st != SHT_OK:
            raise ShtError("%s: %s (%s)" % (what, sht_status_string(st), _lib.sht_last_error(self._h).decode()))

    def sht_analysis(self, maps, alm, stream=None):
        self._check(_lib.sht_analysis(self._h, _ptr(maps), _ptr(alm), _stream(stream)), "sht_analysis")

    def sht_synthesis(self, alm, maps, stream=None):
        self._check(_lib.sht_synthesis(self._h, _ptr(alm), _ptr(maps), _stream(stream)), "sht_synthesis")

    def sht_analysis_iter(self, maps, alm, niter, resid_rms=None, stream=None):
        self._check(_lib.sht_analysis_iter(self._h, _ptr(maps), _ptr(alm), niter, _ptr(resid_rms), _stream(stream)),
                    "sht_analysis_iter")

    def sht_analysis_pol(self, maps, alm, which, stream=None):
        self._check(_lib.sht_analysis_pol(self._h, _ptr(maps), _ptr(alm), which, _stream(stream)), "sht_analysis_pol")

    def sht_synthesis_pol(self, alm, maps, which, stream=None):
        self._check(_lib.sht_synthesis_pol(self._h, _ptr(alm), _ptr(maps), which, _stream(stream)), "sht_synthesis_pol")

    def sht_eb_split(self, maps_in, maps_out, which, stream=None):
        self._check(_lib.sht_eb_split(self._h, _ptr(maps_in), _ptr(maps_out), which, _stream(stream)), "sht_eb_split")

    def sht_eb_split_static(self, maps_in, maps_out, which, stream=None):
        self._check(_lib.sht_eb_split_static(self._h, _ptr(maps_in), _ptr(maps_out), which, _stream(stream)), "sht_eb_split_static")

    def sht_plan_set_option(self, option, value):
        self._check(_lib.sht_plan_set_option(self._h, option, value), "sht_plan_set_option")

    def sht_plan_get_option(self, option):
        return int(_lib.sht_plan_get_option(self._h, option))

    def sht_plan_reserve_iter(self):
        self._check(_lib.sht_plan_reserve_iter(self._h), "sht_plan_reserve_iter")

    def sht_plan_set_iter_mode(self, mode):
        self._check(_lib.sht_plan_set_iter_mode(self._h, mode), "sht_plan_set_iter_mode")

    def sht_plan_set_lambda_mode(self, mode):
        self._check(_lib.sht_plan_set_lambda_mode(self._h, mode), "sht_plan_set_lambda_mode")

    def sht_plan_lambda_mode(self):
        return int(_lib.sht_plan_lambda_mode(self._h))

    def sht_analysis_host(self, maps_host, alm_host):
        self._check(_lib.sht_analysis_host(self._h, _ptr(maps_host), _ptr(alm_host)), "sht_analysis_host")

    def sht_synthesis_host(self, alm_host, maps_host):
        self._check(_lib.sht_synthesis_host(self._h, _ptr(alm_host), _ptr(maps_host)), "sht_synthesis_host")

    # FP32 storage (float32 maps, complex64 a_lm), FP64 arithmetic inside
    def sht_analysis_f32(self, maps, alm, stream=None):
        self._check(_lib.sht_analysis_f32(self._h, _ptr(maps), _ptr(alm), _stream(stream)), "sht_analysis_f32")

    def sht_synthesis_f32(self, alm, maps, stream=None):
        self._check(_lib.sht_synthesis_f32(self._h, _ptr(alm), _ptr(maps), _stream(stream)), "sht_synthesis_f32")

    def sht_analysis_host_f32(self, maps_host, alm_host):
        self._check(_lib.sht_analysis_host_f32(self._h, _ptr(maps_host), _ptr(alm_host)), "sht_analysis_host_f32")

    def sht_synthesis_host_f32(self, alm_host, maps_host):
        self._check(_lib.sht_synthesis_host_f32(self._h, _ptr(alm_host), _ptr(maps_host)), "sht_synthesis_host_f32")

    def sht_plan_set_timing(self, enable):
        self._check(_lib.sht_plan_set_timing(self._h, 1 if enable else 0), "sht_plan_set_timing")

    def sht_plan_stage_ms(self):
        """-> (ms[4], n[4]) for ring-FFT analysis, Legendre analysis, Legendre synthesis, ring-FFT synthesis"""
        ms = (_d * 4)()
        n = (_i * 4)()
        self._check(_lib.sht_plan_stage_ms(self._h, ms, n), "sht_plan_stage_ms")
        return list(ms), list(n)

    def workspace_bytes(self):
        return int(_lib.sht_plan_workspace_bytes(self._h))

    def executed_flops(self, direction):
        return float(_lib.sht_plan_executed_flops(self._h, direction))

    def chunk_maps(self):
        return int(_lib.sht_plan_chunk_maps(self._h))

    def kernel_launches(self):
        return int(_lib.sht_plan_kernel_launches(self._h))

    def destroy(self):
        if self._h is not None:
            _lib.sht_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
