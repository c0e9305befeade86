"""Thin ctypes binding of librmsynth.so: argument marshalling only, same names as include/rmsynth.h.

Every step of the hot path runs in the library's CUDA kernels; torch is used by callers for
device memory and streams only.  There is no CPU fallback: if the library is missing this
module raises at import, and every call raises RmsynthError on a non-OK status.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
# RMSYNTH_LIB selects another build of the same sources (the timeline debug build); default = the product library,
# recompiled here if the sources on disk are not the ones it was built from (content hash, see build.py).
LIB_PATH = os.environ.get("RMSYNTH_LIB") or _build.build()
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1810_06250_b200.build` (no CPU fallback exists)")
_lib = C.CDLL(LIB_PATH)

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED = range(5)
IN_LOS_MAJOR, IN_FREQ_MAJOR, OUT_LOS_MAJOR, OUT_PHI_MAJOR = 0, 1, 0, 2
SCHEME_AUTO, SCHEME_TF32X3, SCHEME_F16X3, SCHEME_FP32_TABLE, SCHEME_FP32_SINCOS = 0, 1, 2, 3, 4

EXPORTS = ["rmsynth_plan_create", "rmsynth_plan_destroy", "rmsynth_plan_info", "rmsynth_plan_phase_matrix",
           "rmsynth_execute", "rmsynth_execute_peaks", "rmsynth_execute_ex", "rmsynth_execute_host", "rmsynth_execute_stream",
           "rmsynth_rmsf", "rmsynth_rmclean", "rmsynth_execute_fft", "rmsynth_peaks_static",
           "rmsynth_launch_count", "rmsynth_strerror", "rmsynth_last_error", "rmsynth_version"]


class Options(C.Structure):
    _fields_ = [("struct_size", C.c_int), ("scheme", C.c_int), ("lambda0_mode", C.c_int),
                ("device", C.c_int), ("lambda0_sq", C.c_double), ("host_chunk_pixels", C.c_longlong)]


class Outputs(C.Structure):
    _fields_ = [("struct_size", C.c_int), ("FQ", C.c_void_p), ("FU", C.c_void_p), ("F_abs", C.c_void_p),
                ("peak_amp", C.c_void_p), ("peak_phi", C.c_void_p), ("pa_lambda0", C.c_void_p),
                ("pa_zero", C.c_void_p), ("peak_index", C.c_void_p)]


_dp, _fp, _ip, _vp = C.POINTER(C.c_double), C.c_void_p, C.c_void_p, C.c_void_p
_lib.rmsynth_plan_create.argtypes = [C.POINTER(_vp), _dp, _dp, C.c_int, _dp, C.c_int, C.POINTER(Options)]
_lib.rmsynth_plan_destroy.argtypes = [_vp]
_lib.rmsynth_plan_info.argtypes = [_vp, _dp, _dp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
_lib.rmsynth_plan_phase_matrix.argtypes = [_vp, _vp, _vp]
_lib.rmsynth_execute.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, _fp, _fp, _vp]
_lib.rmsynth_execute_peaks.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, _fp, _fp, _fp, _fp, _fp, _fp, _ip, _vp]
_lib.rmsynth_execute_ex.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, C.POINTER(Outputs), _vp]
_lib.rmsynth_execute_host.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, _fp, _fp, _fp, _fp, _fp, _fp, _ip]
FILL_FN = C.CFUNCTYPE(C.c_longlong, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_longlong)
DRAIN_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_longlong, C.c_longlong, C.POINTER(Outputs))
WANT_CUBES, WANT_MAPS = 1, 2
_lib.rmsynth_execute_stream.argtypes = [_vp, C.c_int, C.c_int, FILL_FN, DRAIN_FN, C.c_void_p, C.POINTER(C.c_longlong)]


class CleanParams(C.Structure):
    _fields_ = [("struct_size", C.c_int), ("gain", C.c_float), ("cutoff", C.c_float), ("max_iter", C.c_int), ("fwhm", C.c_float)]


class FftParams(C.Structure):
    _fields_ = [("struct_size", C.c_int), ("window", C.c_int), ("oversampling", C.c_float)]


_lib.rmsynth_execute_fft.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, _fp, _fp, C.POINTER(FftParams), _vp]
_lib.rmsynth_rmclean.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_int, C.POINTER(CleanParams), _fp, _fp, _fp, _fp, _fp, _fp, _ip, _vp]
_lib.rmsynth_peaks_static.argtypes = [_vp, _fp, _fp, C.c_longlong, C.c_longlong, C.c_int, _fp, _fp, _fp, _fp, _ip, _vp]
_lib.rmsynth_rmsf.argtypes = [_vp, _dp, C.c_int, _dp, _dp]
_lib.rmsynth_launch_count.argtypes = [C.c_int]
_lib.rmsynth_launch_count.restype = C.c_longlong
_lib.rmsynth_strerror.argtypes = [C.c_int]
for _n in ("rmsynth_strerror", "rmsynth_last_error", "rmsynth_version"):
    getattr(_lib, _n).restype = C.c_char_p


class RmsynthError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        super().__init__(f"rmsynth status {status} ({_lib.rmsynth_strerror(status).decode()}): "
                         f"{_lib.rmsynth_last_error().decode()}")


def _check(status: int):
    if status != OK:
        raise RmsynthError(status)


def _ptr(t):
    """Device/host address of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags.c_contiguous
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def rmsynth_version() -> str:
    return _lib.rmsynth_version().decode()


if not os.environ.get("RMSYNTH_LIB") and _build.source_hash() not in rmsynth_version():
    raise ImportError(f"{LIB_PATH} was not built from the sources on disk ({rmsynth_version()} vs {_build.source_hash()})")


def rmsynth_launch_count(reset: bool = False) -> int:
    return int(_lib.rmsynth_launch_count(int(reset)))


class Plan:
    """Owns an rmsynth_plan*.  Methods carry the C entry-point names without the prefix."""

    def __init__(self, nu_hz, w, phi, scheme=SCHEME_AUTO, lambda0_mode=0, lambda0_sq=0.0, device=-1, host_chunk_pixels=0):
        nu = np.ascontiguousarray(nu_hz, dtype=np.float64)
        ph = np.ascontiguousarray(phi, dtype=np.float64)
        ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        if ww is not None and ww.size != nu.size:
            raise ValueError("w and nu_hz differ in length")
        opt = Options(C.sizeof(Options), scheme, lambda0_mode, device, lambda0_sq, host_chunk_pixels)
        self._h = _vp()
        _check(_lib.rmsynth_plan_create(C.byref(self._h), _d(nu), _d(ww), nu.size, _d(ph), ph.size, C.byref(opt)))
        K, l0 = C.c_double(), C.c_double()
        nc, npz, sc = C.c_int(), C.c_int(), C.c_int()
        _check(_lib.rmsynth_plan_info(self._h, C.byref(l0), C.byref(K), C.byref(nc), C.byref(npz), C.byref(sc)))
        self.K, self.lambda0_sq, self.n_chan, self.n_phi, self.scheme = K.value, l0.value, nc.value, npz.value, sc.value

    def destroy(self):
        if getattr(self, "_h", None) and _lib is not None:      # _lib is None while the interpreter shuts down
            _lib.rmsynth_plan_destroy(self._h)
            self._h = None

    __del__ = destroy

    def phase_matrix(self):
        c = np.empty((self.n_chan, self.n_phi), dtype=np.float32)
        s = np.empty_like(c)
        _check(_lib.rmsynth_plan_phase_matrix(self._h, c.ctypes.data, s.ctypes.data))
        return c, s

    def rmsf(self, phi_eval=None):
        ph = None if phi_eval is None else np.ascontiguousarray(phi_eval, dtype=np.float64)
        n = self.n_phi if ph is None else ph.size
        re, im = np.empty(n), np.empty(n)
        _check(_lib.rmsynth_rmsf(self._h, _d(ph), n, _d(re), _d(im)))
        return re + 1j * im

    def execute(self, Q, U, n_pix, layout, FQ, FU, stream=None):
        """Q,U,FQ,FU: CUDA float32 tensors (contiguous). stream: int cudaStream_t or None."""
        _check(_lib.rmsynth_execute(self._h, _ptr(Q), _ptr(U), n_pix, layout, _ptr(FQ), _ptr(FU), stream))

    def execute_peaks(self, Q, U, n_pix, layout, FQ=None, FU=None, peak_amp=None, peak_phi=None,
                      pa_lambda0=None, pa_zero=None, peak_index=None, stream=None):
        _check(_lib.rmsynth_execute_peaks(self._h, _ptr(Q), _ptr(U), n_pix, layout, _ptr(FQ), _ptr(FU),
                                          _ptr(peak_amp), _ptr(peak_phi), _ptr(pa_lambda0), _ptr(pa_zero),
                                          _ptr(peak_index), stream))

    def execute_ex(self, Q, U, n_pix, layout, FQ=None, FU=None, F_abs=None, peak_amp=None, peak_phi=None,
                   pa_lambda0=None, pa_zero=None, peak_index=None, stream=None):
        """Any subset of the outputs (cubes FQ/FU, |F| cube, maps) in one call; all DEVICE tensors."""
        out = Outputs(C.sizeof(Outputs), _ptr(FQ), _ptr(FU), _ptr(F_abs), _ptr(peak_amp), _ptr(peak_phi),
                      _ptr(pa_lambda0), _ptr(pa_zero), _ptr(peak_index))
        _check(_lib.rmsynth_execute_ex(self._h, _ptr(Q), _ptr(U), n_pix, layout, C.byref(out), stream))

    def execute_host(self, Q, U, n_pix, layout, FQ=None, FU=None, peak_amp=None, peak_phi=None,
                     pa_lambda0=None, pa_zero=None, peak_index=None):
        """All arrays in HOST memory (numpy or CPU torch tensors, ideally pinned)."""
        _check(_lib.rmsynth_execute_host(self._h, _ptr(Q), _ptr(U), n_pix, layout, _ptr(FQ), _ptr(FU),
                                         _ptr(peak_amp), _ptr(peak_phi), _ptr(pa_lambda0), _ptr(pa_zero),
                                         _ptr(peak_index)))

    def execute_fft(self, Q, U, n_pix, layout, FQ, FU, window=0, oversampling=0.0, stream=None):
        """Approximate FFT variant of execute() (NEXT-4); window / oversampling 0 = defaults (6, 2)."""
        prm = FftParams(C.sizeof(FftParams), window, oversampling)
        _check(_lib.rmsynth_execute_fft(self._h, _ptr(Q), _ptr(U), n_pix, layout, _ptr(FQ), _ptr(FU), C.byref(prm), stream))

    def rmclean(self, FQ, FU, n_pix, layout, gain, cutoff, max_iter, model_q, model_u, resid_q, resid_u,
                rest_q=None, rest_u=None, n_iter=None, fwhm=0.0, stream=None):
        """RM-CLEAN of device-resident dirty cubes (all DEVICE tensors, laid out per the OUT_* bit of `layout`)."""
        prm = CleanParams(C.sizeof(CleanParams), gain, cutoff, max_iter, fwhm)
        _check(_lib.rmsynth_rmclean(self._h, _ptr(FQ), _ptr(FU), n_pix, layout, C.byref(prm), _ptr(model_q), _ptr(model_u),
                                    _ptr(resid_q), _ptr(resid_u), _ptr(rest_q), _ptr(rest_u), _ptr(n_iter), stream))

    def peaks_static(self, FQ, FU, n_pix, layout, ld=0, peak_amp=None, peak_phi=None, pa_lambda0=None, pa_zero=None,
                     peak_index=None, stream=None):
        """Peak maps of DEVICE cubes through the entry point that never allocates (records in the library's static
        32 MiB array; n_pix <= 1048576 per call; calls that may overlap on the GPU race on that array)."""
        _check(_lib.rmsynth_peaks_static(self._h, _ptr(FQ), _ptr(FU), n_pix, ld, layout, _ptr(peak_amp), _ptr(peak_phi),
                                         _ptr(pa_lambda0), _ptr(pa_zero), _ptr(peak_index), stream))

    def execute_stream(self, layout, outputs, fill, drain):
        """fill(i, Q, U, max_pix) -> n and drain(i, n, out) are Python callables; Q, U are numpy views of the
        library's pinned staging buffers (flat, max_pix * n_chan floats each), out is a dict of numpy views that are
        valid only during the call.  Returns the number of lines of sight processed."""
        nc, npz = self.n_chan, self.n_phi

        def _fill(_, i, q, u, max_pix):
            qa = np.ctypeslib.as_array(C.cast(q, C.POINTER(C.c_float)), shape=(max_pix * nc,))
            ua = np.ctypeslib.as_array(C.cast(u, C.POINTER(C.c_float)), shape=(max_pix * nc,))
            return int(fill(i, qa, ua, max_pix))

        def _drain(_, i, n, out):
            o = out.contents
            view = {}
            for name in ("FQ", "FU"):
                a = getattr(o, name)
                if a:
                    view[name] = np.ctypeslib.as_array(C.cast(a, C.POINTER(C.c_float)), shape=(n * npz,))
            for name in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
                a = getattr(o, name)
                if a:
                    view[name] = np.ctypeslib.as_array(C.cast(a, C.POINTER(C.c_float)), shape=(n,))
            if o.peak_index:
                view["peak_index"] = np.ctypeslib.as_array(C.cast(o.peak_index, C.POINTER(C.c_int)), shape=(n,))
            drain(i, n, view)

        done = C.c_longlong(0)
        cb_fill, cb_drain = FILL_FN(_fill), DRAIN_FN(_drain)
        _check(_lib.rmsynth_execute_stream(self._h, layout, outputs, cb_fill, cb_drain, None, C.byref(done)))
        return done.value
