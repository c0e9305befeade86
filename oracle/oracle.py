"""ctypes wrapper around oracle/rmsynth_oracle.c (argument marshalling only).

TEST INFRASTRUCTURE ONLY -- see the header of rmsynth_oracle.c.  All arithmetic of
the method is in the C file; this module converts numpy arrays to pointers.
All cubes are LOS-major: Q[p, i], F[p, k].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rmsynth_oracle.c")
_LIB = os.path.join(_HERE, "librmsynth_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (FP64, no fast-math so libm cos/sin are used as written)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = C.CDLL(_LIB)
        dp, fp, ip = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
        lib.oracle_lambda_sq.argtypes = [dp, C.c_int, dp]
        lib.oracle_lambda_sq.restype = None
        lib.oracle_plan_scalars.argtypes = [dp, dp, C.c_int, C.c_int, C.c_double, dp, dp]
        lib.oracle_plan_scalars.restype = C.c_int
        lib.oracle_rmsf.argtypes = [dp, dp, C.c_int, C.c_double, C.c_double, dp, C.c_int, dp, dp]
        lib.oracle_rmsf.restype = None
        common = [fp, fp, C.c_longlong, dp, dp, C.c_int, C.c_double, C.c_double, dp, C.c_int, dp, dp]
        lib.oracle_naive.argtypes = common
        lib.oracle_naive.restype = None
        lib.oracle_table.argtypes = common + [C.c_int]
        lib.oracle_table.restype = C.c_int
        lib.oracle_tolerance_scale.argtypes = [fp, fp, C.c_longlong, dp, C.c_int, C.c_double, dp]
        lib.oracle_tolerance_scale.restype = None
        lib.oracle_peaks.argtypes = [dp, dp, C.c_longlong, dp, C.c_int, C.c_double, ip, dp, dp, dp, dp]
        lib.oracle_peaks.restype = None
        lib.oracle_rmclean.argtypes = [dp, dp, C.c_longlong, C.c_int, dp, dp, C.c_double, C.c_double, C.c_int,
                                       C.c_double, C.c_double, dp, dp, dp, dp, dp, dp, ip, dp]
        lib.oracle_rmclean.restype = None
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _f32(a):
    a = np.asarray(a)
    if a.dtype != np.float32:
        raise TypeError("Q/U cubes are FP32 (reading A12)")
    return np.ascontiguousarray(a)


def lambda_sq(nu_hz):
    nu = _f64(nu_hz)
    out = np.empty_like(nu)
    _load().oracle_lambda_sq(_d(nu), nu.size, _d(out))
    return out


def plan_scalars(lam2, w, lambda0_mode=0, lambda0_in=0.0):
    lam2, w = _f64(lam2), _f64(w)
    K, l0 = C.c_double(), C.c_double()
    rc = _load().oracle_plan_scalars(_d(lam2), _d(w), lam2.size, lambda0_mode, lambda0_in,
                                     C.byref(K), C.byref(l0))
    if rc != 0:
        raise ValueError("sum of weights is zero")
    return K.value, l0.value


@dataclass
class Plan:
    lam2: np.ndarray
    w: np.ndarray
    phi: np.ndarray
    K: float
    lambda0_sq: float


def make_plan(nu_hz, w, phi, lambda0_mode=0, lambda0_in=0.0) -> Plan:
    lam2 = lambda_sq(nu_hz)
    w = np.ones_like(lam2) if w is None else _f64(w)
    K, l0 = plan_scalars(lam2, w, lambda0_mode, lambda0_in)
    return Plan(lam2, w, _f64(phi), K, l0)


def rmsf(plan: Plan, phi_eval=None):
    phi = plan.phi if phi_eval is None else _f64(phi_eval)
    re, im = np.empty(phi.size), np.empty(phi.size)
    _load().oracle_rmsf(_d(plan.lam2), _d(plan.w), plan.lam2.size, plan.K, plan.lambda0_sq,
                        _d(phi), phi.size, _d(re), _d(im))
    return re + 1j * im


def _synth(fn, plan, Q, U, extra=()):
    Q, U = _f32(Q), _f32(U)
    n_pix, n_chan = Q.shape
    assert U.shape == Q.shape and n_chan == plan.lam2.size
    FQ = np.empty((n_pix, plan.phi.size))
    FU = np.empty((n_pix, plan.phi.size))
    r = fn(_f(Q), _f(U), n_pix, _d(plan.lam2), _d(plan.w), n_chan, plan.K, plan.lambda0_sq,
           _d(plan.phi), plan.phi.size, _d(FQ), _d(FU), *extra)
    return FQ, FU, r


def synth_naive(plan: Plan, Q, U):
    """Literal Eqs. 15-16: trig inside the innermost loop. Q,U: [n_pix, n_chan] float32."""
    FQ, FU, _ = _synth(_load().oracle_naive, plan, Q, U)
    return FQ, FU


def synth_table(plan: Plan, Q, U, n_threads=0, return_threads=False):
    """Same sums with the (i,k) trig table hoisted and OpenMP over lines of sight."""
    FQ, FU, used = _synth(_load().oracle_table, plan, Q, U, (int(n_threads),))
    if used < 0:
        raise MemoryError("oracle_table")
    return (FQ, FU, used) if return_threads else (FQ, FU)


def tolerance_scale(plan: Plan, Q, U):
    Q, U = _f32(Q), _f32(U)
    T = np.empty(Q.shape[0])
    _load().oracle_tolerance_scale(_f(Q), _f(U), Q.shape[0], _d(plan.w), Q.shape[1], plan.K, _d(T))
    return T


def peaks(plan: Plan, FQ, FU):
    FQ, FU = _f64(FQ), _f64(FU)
    n = FQ.shape[0]
    k = np.empty(n, dtype=np.int32)
    amp, ph, pa0, paz = (np.empty(n) for _ in range(4))
    _load().oracle_peaks(_d(FQ), _d(FU), n, _d(plan.phi), plan.phi.size, plan.lambda0_sq,
                         k.ctypes.data_as(C.POINTER(C.c_int)), _d(amp), _d(ph), _d(pa0), _d(paz))
    return dict(kstar=k, peak_amp=amp, peak_phi=ph, pa_lambda0=pa0, pa_zero=paz)


def rmsf_double_width(plan: Plan):
    """R on the double-width grid of reading C1: R(m dphi), m = -(n_phi-1) .. n_phi-1 (uniform plan grid required)."""
    n = plan.phi.size
    dphi = (plan.phi[-1] - plan.phi[0]) / (n - 1) if n > 1 else 1.0
    if n > 2 and np.max(np.abs(np.diff(plan.phi) - dphi)) > 1e-9 * abs(dphi):
        raise ValueError("RM-CLEAN needs a uniform depth grid (reading C1)")
    return rmsf(plan, np.arange(-(n - 1), n) * dphi), dphi


def rmclean(plan: Plan, FQ, FU, gain=0.1, cutoff=0.0, max_iter=100, fwhm=None, restore=True):
    """Hogbom RM-CLEAN per line of sight (readings C1-C8).  FQ, FU: dirty cubes [n_pix, n_phi] (any float type, promoted
    to FP64).  Returns dict(model, residual, restored (or None), n_iter, min_margin); cubes complex128 [n_pix, n_phi]."""
    FQ, FU = _f64(FQ), _f64(FU)
    n_pix, n_phi = FQ.shape
    assert n_phi == plan.phi.size
    R, dphi = rmsf_double_width(plan)
    Rre, Rim = _f64(R.real), _f64(R.imag)
    mq, mu, rq, ru = (np.empty((n_pix, n_phi)) for _ in range(4))
    sq, su = (np.empty((n_pix, n_phi)), np.empty((n_pix, n_phi))) if restore else (None, None)
    it = np.empty(n_pix, dtype=np.int32)
    margin = np.empty(n_pix)
    null = C.POINTER(C.c_double)()
    _load().oracle_rmclean(_d(FQ), _d(FU), n_pix, n_phi, _d(Rre), _d(Rim), float(gain), float(cutoff), int(max_iter),
                           float(dphi), float(fwhm if fwhm is not None else 1.0),
                           _d(mq), _d(mu), _d(rq), _d(ru), _d(sq) if restore else null, _d(su) if restore else null,
                           it.ctypes.data_as(C.POINTER(C.c_int)), _d(margin))
    return dict(model=mq + 1j * mu, residual=rq + 1j * ru, restored=(sq + 1j * su) if restore else None,
                n_iter=it, min_margin=margin)
