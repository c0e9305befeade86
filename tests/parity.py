"""Shared parity checks: CUDA path (through the C-ABI binding) vs the FP64 oracle.

Tolerances (BASELINE.json north_star):
  cubes : max_k |F_gpu - F_oracle| <= 1e-5 * T_p per pixel, T_p = K sum_i w_i |P_i|
  index : k* equal, unless the oracle's |F| at the two indices differ by <= 2e-5 * T_p
  maps  : compared only where indices agree (error propagation of the parabola, reading A8)
"""
import numpy as np

TOL = 1e-5


def oracle_reference(oracle, nu, w, phi, q_los, u_los, lambda0_mode=0, lambda0_sq=0.0):
    plan = oracle.make_plan(nu, w, phi, lambda0_mode, lambda0_sq)
    FQ, FU = oracle.synth_table(plan, q_los, u_los)
    T = oracle.tolerance_scale(plan, q_los, u_los)
    return plan, FQ, FU, T


def check_cubes(FQ_gpu, FU_gpu, FQ, FU, T, what=""):
    """FQ_gpu/FU_gpu: float32 [n_pix, n_phi] (already brought to LOS-major)."""
    # |F_gpu - F_oracle| of the complex samples (the north_star's quantity), not the larger of its two components
    err = np.hypot(FQ_gpu.astype(np.float64) - FQ, FU_gpu.astype(np.float64) - FU).max(axis=1)
    Tsafe = np.where(T > 0, T, 1.0)
    ratio = err / Tsafe
    worst = float(ratio.max()) if ratio.size else 0.0
    assert np.all(np.isfinite(ratio)) and worst <= TOL, f"{what}: max err/T_p = {worst:.3e} > {TOL}"
    return worst


def check_peaks(oracle, oplan, FQ, FU, T, got, dphi_min, what=""):
    """got: dict of numpy arrays kstar, peak_amp, peak_phi, pa_lambda0, pa_zero (GPU)."""
    ref = oracle.peaks(oplan, FQ, FU)
    y = np.sqrt(FQ ** 2 + FU ** 2)
    n = y.shape[0]
    rows = np.arange(n)
    kg, ko = got["kstar"].astype(np.int64), ref["kstar"].astype(np.int64)
    # reading A17: lines of sight with a non-finite |F| report -1 / NaN on both sides and are compared no further
    dead = ko < 0
    if dead.any():
        assert np.array_equal(kg[dead], ko[dead]), f"{what}: non-finite lines of sight must report index -1"
        for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
            assert np.all(np.isnan(got[k][dead])), f"{what}: {k} must be NaN on a non-finite line of sight"
        live = ~dead
        got = {k: v[live] for k, v in got.items()}
        return check_peaks(oracle, oplan, FQ[live], FU[live], T[live], got, dphi_min, what) if live.any() else 0
    assert kg.min() >= 0 and kg.max() < y.shape[1]
    gap = y[rows, ko] - y[rows, kg]
    bad = (kg != ko) & (gap > 2 * TOL * T)
    assert not bad.any(), f"{what}: {bad.sum()} peak indices differ beyond tolerance"
    same = kg == ko
    n_phi = y.shape[1]
    k = ko
    inner = same & (k > 0) & (k < n_phi - 1)
    y0 = y[rows, k]
    ym = y[rows, np.maximum(k - 1, 0)]
    yp = y[rows, np.minimum(k + 1, n_phi - 1)]
    curv = np.maximum(np.abs(ym - 2 * y0 + yp), 1e-300)
    # refinement is ill-conditioned when the curvature is within the error budget: skip those
    well = inner & (curv > 40 * TOL * T)
    tol_phi = dphi_min * (4 * TOL * T) / curv + 2e-6 * np.abs(ref["peak_phi"]) + 1e-6
    sel = np.where(inner, well, same)
    dphi = np.abs(got["peak_phi"] - ref["peak_phi"])
    assert np.all(dphi[sel] <= tol_phi[sel] + (~inner[sel]) * 1e-5), f"{what}: peak_phi off by {dphi[sel].max()}"
    damp = np.abs(got["peak_amp"] - ref["peak_amp"])
    assert np.all(damp[sel] <= 4 * TOL * T[sel] + 1e-6 * y0[sel]), f"{what}: peak_amp off by {damp[sel].max()}"
    ysafe = np.maximum(y0, 1e-30)
    tol_pa = 2 * TOL * T / ysafe + 2e-6
    dpa = np.abs(got["pa_lambda0"] - ref["pa_lambda0"])
    dpa = np.minimum(dpa, np.abs(dpa - np.pi))
    strong = sel & (y0 > 100 * TOL * T)
    assert np.all(dpa[strong] <= tol_pa[strong]), f"{what}: pa_lambda0 off by {dpa[strong].max()}"
    dpz = np.abs(got["pa_zero"] - ref["pa_zero"])
    dpz = np.minimum(dpz, np.abs(dpz - np.pi))
    tol_pz = tol_pa + dphi * abs(oplan.lambda0_sq) + tol_phi * abs(oplan.lambda0_sq) + 1e-5
    assert np.all(dpz[strong] <= tol_pz[strong]), f"{what}: pa_zero off by {dpz[strong].max()}"
    assert np.all((got["pa_zero"] >= -np.pi / 2 - 1e-6) & (got["pa_zero"] <= np.pi / 2 + 1e-6))
    return int((~same).sum())
