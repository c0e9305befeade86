"""Pins that fix the FP64 oracle to something other than itself.

CPU only.  Each test names the passage of PAPER.md (P:L<n>) or the mathematical fact it
checks, and which plausible oracle mistake it would catch.
"""
import os

import numpy as np
import pytest

C = 299792458.0
GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) >= 3:
                out[line[0]] = (float(line[1]), float(line[2]))
    return out


def lofar_like(n=64, lo=120e6, hi=168e6):
    return lo + np.arange(n) * (hi - lo) / (n - 1)


def rand_weights(n, rng, flag=0.1):
    w = rng.uniform(0.5, 1.0, n)
    w[rng.random(n) < flag] = 0.0
    return w


# ---------------------------------------------------------------- P9: paper-printed values
def test_p9_lambda_sq_against_paper_printed_lofar_numbers(oracle_mod):
    """lambda^2 = (c/nu)^2 (A1) + Eq. 20/21 reproduce the numbers printed at P:L247.
    Catches: wrong c, nu in MHz, lambda instead of lambda^2."""
    g = golden()
    nu_lo, nu_hi, dnu = g["lofar_lr_nu_lo_hz"][0], g["lofar_lr_nu_hi_hz"][0], g["lofar_lr_chan_width_hz"][0]
    lam2 = oracle_mod.lambda_sq(np.array([nu_lo, nu_hi, nu_lo + dnu]))
    big_delta = lam2[0] - lam2[1]            # total lambda^2 span
    small_delta = lam2[0] - lam2[2]          # channel width in lambda^2 at the low end
    res, tol = g["lofar_lr_resolution"]
    assert abs(2 * np.sqrt(3) / big_delta - res) <= tol          # Eq. 20 -> "1.17"
    pm, tol = g["lofar_lr_phi_max"]
    assert abs(np.sqrt(3) / small_delta - pm) <= tol             # Eq. 21 -> "about 350"


def test_p9_rmsf_fwhm_close_to_eq20(oracle_mod):
    """Measured FWHM of |R| for the LOFAR_LR grid is within 25 % of Eq. 20's 1.17.
    Eq. 20 is itself approximate ("~"): it is the FWHM of a top hat in lambda^2 up to ~10 %, and
    channels uniform in frequency sample lambda^2 non-uniformly (measured: 1.384).
    Catches: a factor 2 in the phase (FWHM would halve/double)."""
    g = golden()
    n = int(g["lofar_lr_n_chan"][0])
    nu = g["lofar_lr_nu_lo_hz"][0] + np.arange(n) * g["lofar_lr_chan_width_hz"][0]
    phi = np.linspace(-3, 3, 6001)
    plan = oracle_mod.make_plan(nu, None, phi)
    a = np.abs(oracle_mod.rmsf(plan))
    above = phi[a >= 0.5]
    fwhm = above.max() - above.min()
    assert abs(fwhm / g["lofar_lr_resolution"][0] - 1.0) < 0.25


def test_p10_work_count_matches_paper():
    """15 * N_pix*N_chan*N_phi = 1.27 TFLOP for the WSRT shape: pins the MAC counter."""
    import rmsynth_inputs as ri
    g = golden()
    cfg = ri.CubeConfig("wsrt", 512, 512, int(g["wsrt_n_chan"][0]), 1e9, 2e9, -200.0, 1.0,
                        int(g["wsrt_n_phi"][0]), "unit", "one_source", 0.0, "los", "los", 0)
    assert cfg.n_pix == g["wsrt_n_pix"][0]
    tflop = g["flop_per_term"][0] * cfg.cmac / 1e12
    assert abs(tflop - g["wsrt_tflop"][0]) <= g["wsrt_tflop"][1]


# ---------------------------------------------------------------- P1-P3, P5, P6: RMSF
def test_p1_p2_p3_rmsf_invariants(oracle_mod):
    """R(0)=1 (Eq. 12+13), R(-phi)=conj R(phi), |R|<=1.  Catches: K missing, wrong sign symmetry."""
    rng = np.random.default_rng(1)
    nu = lofar_like(97)
    w = rand_weights(97, rng)
    phi = np.linspace(-60, 60, 241)
    plan = oracle_mod.make_plan(nu, w, phi)
    R = oracle_mod.rmsf(plan)
    assert abs(R[120] - 1.0) < 1e-14
    assert np.max(np.abs(R - np.conj(R[::-1]))) < 1e-14
    assert np.all(np.abs(R) <= 1.0 + 1e-14)


def test_p5_weighted_mean_lambda0_kills_first_derivative(oracle_mod):
    """Reading A2: dR/dphi(0) = -2iK sum w (lam2 - lam0^2) = 0 iff lam0^2 is the WEIGHTED mean
    (the purpose stated at P:L119).  Catches: plain mean used with non-unit weights."""
    rng = np.random.default_rng(2)
    nu = lofar_like(128)
    w = rand_weights(128, rng, flag=0.2)
    h = 1e-4
    for mode, expect_zero in ((0, True), (1, False)):
        plan = oracle_mod.make_plan(nu, w, [-h, h], lambda0_mode=mode)
        R = oracle_mod.rmsf(plan)
        d = (R[1] - R[0]) / (2 * h)
        lam2 = (C / nu) ** 2
        analytic = -2j * plan.K * np.sum(w * (lam2 - plan.lambda0_sq))
        assert abs(d - analytic) < 1e-6
        assert (abs(d) < 1e-7) == expect_zero      # central difference leaves O(h^2 R''') ~ 1e-9
    # explicit mode returns the caller's value (Fig. 1 left uses lambda0^2 = 0)
    assert oracle_mod.make_plan(nu, w, [0.0], lambda0_mode=2, lambda0_in=0.0).lambda0_sq == 0.0


def test_lambda0_modes_by_value(oracle_mod):
    """P:L119 "set to the mean of lambda_i^2", reading A2: mode 0 = weighted mean, mode 1 = plain mean over ALL
    channels (flagged ones included), mode 2 = the caller's value.  Values formed here from c/nu with numpy and
    with exact rational weights, on a grid where the two means differ in the second digit.
    Catches: mode 1 silently returning the weighted mean, or a mean over the unflagged channels only."""
    nu = np.array([100e6, 125e6, 150e6, 200e6])
    w = np.array([1.0, 0.0, 1.0, 2.0])
    lam2 = (C / nu) ** 2
    weighted = (lam2[0] + lam2[2] + 2.0 * lam2[3]) / 4.0           # 4.369
    plain = lam2.sum() / 4.0                                       # 5.245
    unflagged_plain = (lam2[0] + lam2[2] + lam2[3]) / 3.0          # 5.076
    assert abs(weighted - plain) > 0.03 * plain and abs(unflagged_plain - plain) > 0.03 * plain
    K0, l0 = oracle_mod.plan_scalars(lam2, w, 0)
    K1, l1 = oracle_mod.plan_scalars(lam2, w, 1)
    K2, l2 = oracle_mod.plan_scalars(lam2, w, 2, 1.25)
    assert K0 == K1 == K2 == 0.25                                  # Eq. 13 with sum w = 4, exact
    assert abs(l0 - weighted) <= 1e-15 * weighted
    assert abs(l1 - plain) <= 1e-15 * plain
    assert l2 == 1.25
    # lambda^2 itself by value: nu = 100 MHz -> lambda = 2.99792458 m
    assert abs(oracle_mod.lambda_sq(np.array([100e6]))[0] - 2.99792458 ** 2) < 1e-14


def test_p6_dirichlet_kernel_closed_form(oracle_mod):
    """Uniform lambda^2 sampling, unit weights: R(phi) = sin(N phi d)/(N sin(phi d)), purely real.
    Catches: dropped factor 2 in the exponent, off-by-one in the channel sum."""
    N, a, d = 50, 1.0, 0.04
    lam2 = a + d * np.arange(N)
    nu = C / np.sqrt(lam2)
    phi = np.linspace(-30, 30, 301) + 0.013
    plan = oracle_mod.make_plan(nu, None, phi)
    assert np.max(np.abs(plan.lam2 - lam2)) < 1e-13
    R = oracle_mod.rmsf(plan)
    ref = np.sin(N * phi * d) / (N * np.sin(phi * d))
    assert np.max(np.abs(R.real - ref)) < 1e-12
    assert np.max(np.abs(R.imag)) < 1e-12


# ---------------------------------------------------------------- P4: point source identity
def test_p4_point_source_identity(oracle_mod):
    """P_i = P0 exp(2i phi0 lam2_i)  =>  F(phi) = P0 exp(2i phi0 lam0^2) R(phi - phi0) for any
    weights; |F(phi0)| = |P0| with phi0 on the grid.  Catches: wrong sign of the exponent,
    Q/U swapped in Eq. 15/16, weights or K dropped, lam0^2 mis-applied."""
    rng = np.random.default_rng(3)
    nu = lofar_like(80)
    w = rand_weights(80, rng)
    phi = np.arange(-40, 41) * 0.5
    plan = oracle_mod.make_plan(nu, w, phi)
    for phi0, P0 in ((7.5, 0.8 * np.exp(0.6j)), (-3.217, 1.3 * np.exp(-2.1j))):
        P = P0 * np.exp(2j * phi0 * plan.lam2)
        # FP32 storage of the samples limits the agreement to ~1e-7
        Q = P.real.astype(np.float32)[None, :]
        U = P.imag.astype(np.float32)[None, :]
        for fn in (oracle_mod.synth_naive, oracle_mod.synth_table):
            FQ, FU = fn(plan, Q, U)
            F = FQ[0] + 1j * FU[0]
            ref = P0 * np.exp(2j * phi0 * plan.lambda0_sq) * oracle_mod.rmsf(plan, phi - phi0)
            assert np.max(np.abs(F - ref)) < 3e-7 * abs(P0)
        if phi0 == 7.5:
            k = int(np.argmax(np.abs(F)))
            assert phi[k] == phi0 and abs(abs(F[k]) - abs(P0)) < 3e-7


# ---------------------------------------------------------------- P7: FFT special case
def test_p7_reduces_to_library_fft(oracle_mod):
    """lam2_i = a + i d, phi_k = k pi/(N d): F_k = K exp(-2i phi_k (a - lam0^2)) DFT(w P)_k.
    Catches: transposed operand / wrong index pairing (i<->k), conjugation errors."""
    rng = np.random.default_rng(4)
    N, a, d = 32, 2.0, 0.05
    lam2 = a + d * np.arange(N)
    nu = C / np.sqrt(lam2)
    phi = np.arange(N) * np.pi / (N * d)
    w = rng.uniform(0.2, 1.0, N)
    plan = oracle_mod.make_plan(nu, w, phi)
    Q = rng.standard_normal((3, N)).astype(np.float32)
    U = rng.standard_normal((3, N)).astype(np.float32)
    FQ, FU = oracle_mod.synth_table(plan, Q, U)
    P = Q.astype(np.float64) + 1j * U.astype(np.float64)
    ref = plan.K * np.exp(-2j * phi * (a - plan.lambda0_sq))[None, :] * np.fft.fft(w[None, :] * P, axis=1)
    assert np.max(np.abs(FQ + 1j * FU - ref)) < 1e-12


# ---------------------------------------------------------------- P8: linearity
def test_p8_linearity(oracle_mod):
    rng = np.random.default_rng(5)
    nu, phi = lofar_like(40), np.linspace(-20, 20, 33)
    plan = oracle_mod.make_plan(nu, rand_weights(40, rng), phi)
    Q1, U1, Q2, U2 = (rng.standard_normal((4, 40)).astype(np.float32) for _ in range(4))
    a = 2.0  # exact in FP32
    F1 = oracle_mod.synth_table(plan, Q1, U1)
    F2 = oracle_mod.synth_table(plan, Q2, U2)
    # the FP32 sum Q1+a*Q2 is rounded, so feed exactly representable combinations
    Qs, Us = (Q1.astype(np.float64) + a * Q2).astype(np.float32), (U1.astype(np.float64) + a * U2).astype(np.float32)
    Fs = oracle_mod.synth_table(plan, Qs, Us)
    resid_q = np.abs(Qs.astype(np.float64) - (Q1.astype(np.float64) + a * Q2)).max()
    for j in range(2):
        assert np.max(np.abs(Fs[j] - (F1[j] + a * F2[j]))) < 1e-12 + 4 * resid_q


# ---------------------------------------------------------------- P11: brute force
def test_p11_brute_force_complex_exp(oracle_mod):
    """Eq. 11 written with the standard library's complex exp, pure Python loops, tiny cube,
    versus the real-form Eqs. 15-16 in both oracle builds.  Also |F| <= T_p (P3)."""
    import cmath
    rng = np.random.default_rng(6)
    n_pix, n_chan, n_phi = 16, 8, 9
    nu = lofar_like(n_chan, 1.0e9, 2.0e9)
    w = rng.uniform(0.0, 1.0, n_chan)
    w[2] = 0.0
    phi = np.linspace(-300, 300, n_phi)
    plan = oracle_mod.make_plan(nu, w, phi)
    Q = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    U = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    lam2 = [(C / f) ** 2 for f in nu]
    W = sum(w)
    l0 = sum(wi * l for wi, l in zip(w, lam2)) / W
    ref = np.zeros((n_pix, n_phi), dtype=complex)
    for p in range(n_pix):
        for k in range(n_phi):
            acc = 0j
            for i in range(n_chan):
                acc += w[i] * complex(float(Q[p, i]), float(U[p, i])) * cmath.exp(-2j * phi[k] * (lam2[i] - l0))
            ref[p, k] = acc / W
    assert abs(plan.K - 1 / W) < 1e-15 and abs(plan.lambda0_sq - l0) < 1e-15
    T = oracle_mod.tolerance_scale(plan, Q, U)
    for fn in (oracle_mod.synth_naive, oracle_mod.synth_table):
        FQ, FU = fn(plan, Q, U)
        assert np.max(np.abs(FQ + 1j * FU - ref)) < 1e-13
        assert np.all(np.abs(FQ + 1j * FU) <= T[:, None] * (1 + 1e-12))
    Tref = [sum(w[i] * abs(complex(float(Q[p, i]), float(U[p, i]))) for i in range(n_chan)) / W for p in range(n_pix)]
    assert np.max(np.abs(T - Tref)) < 1e-14


def test_a13_zero_weight_channels_are_removed(oracle_mod):
    """Reading A13 ("bad channels were removed before processing"): with w_i = 0 channel i is not part of the
    sums at all.  F, T_p, K and lambda_0^2 must equal those of the SHORTER problem with the flagged channels deleted,
    whatever the flagged samples hold -- NaN and Inf included.  Catches: 0 * NaN = NaN leaking into F, flagged
    channels counted in K or in the mean lambda^2."""
    rng = np.random.default_rng(9)
    n = 24
    nu = lofar_like(n, 1.0e9, 1.5e9)
    w = rng.uniform(0.2, 1.0, n)
    flagged = np.array([0, 5, 6, 17, 23])
    w[flagged] = 0.0
    phi = np.linspace(-200, 200, 11)
    Q = rng.standard_normal((6, n)).astype(np.float32)
    U = rng.standard_normal((6, n)).astype(np.float32)
    Q[0, 5] = np.nan; U[1, 17] = np.inf; Q[2, 0] = -np.inf; Q[3, flagged] = 1e30; U[4, 23] = np.nan
    keep = np.setdiff1d(np.arange(n), flagged)
    full = oracle_mod.make_plan(nu, w, phi)
    short = oracle_mod.make_plan(nu[keep], w[keep], phi)
    assert full.K == short.K and abs(full.lambda0_sq - short.lambda0_sq) < 1e-15
    for fn in (oracle_mod.synth_naive, oracle_mod.synth_table):
        a = fn(full, Q, U)
        b = fn(short, np.ascontiguousarray(Q[:, keep]), np.ascontiguousarray(U[:, keep]))
        assert np.all(np.isfinite(a[0])) and np.all(np.isfinite(a[1]))
        assert np.max(np.abs(a[0] - b[0])) < 1e-14 and np.max(np.abs(a[1] - b[1])) < 1e-14
    Ta = oracle_mod.tolerance_scale(full, Q, U)
    Tb = oracle_mod.tolerance_scale(short, np.ascontiguousarray(Q[:, keep]), np.ascontiguousarray(U[:, keep]))
    assert np.all(np.isfinite(Ta)) and np.max(np.abs(Ta - Tb)) < 1e-14
    # a non-finite sample in a channel that is NOT flagged still poisons its line of sight (and only that one)
    Q[5, 3] = np.nan
    a = oracle_mod.synth_table(full, Q, U)
    assert np.all(np.isnan(a[0][5])) and np.all(np.isfinite(a[0][:5]))


def test_naive_and_table_agree_on_config1_sample(oracle_mod):
    """oracle_table vs oracle_naive to 1e-12 T_p on real config-1 inputs."""
    import torch
    import rmsynth_inputs as ri
    cfg = ri.CONFIGS[1]
    nu, w, phi = ri.grids(cfg)
    Q, U = ri.generate_pixels(cfg, torch.arange(0, 4096, 173))
    plan = oracle_mod.make_plan(nu, w, phi)
    a = oracle_mod.synth_naive(plan, Q.numpy(), U.numpy())
    b = oracle_mod.synth_table(plan, Q.numpy(), U.numpy())
    T = oracle_mod.tolerance_scale(plan, Q.numpy(), U.numpy())
    for x, y in zip(a, b):
        assert np.max(np.abs(x - y) / T[:, None]) < 1e-12


# ---------------------------------------------------------------- P12: peaks, parabola, PA
def test_p12_parabola_exact_and_edges(oracle_mod):
    """Samples of a true parabola: vertex and height recovered exactly, uniform and
    non-uniform grids; no refinement at the edges or for a non-concave triple (A8)."""
    for phi in (np.arange(-5, 6) * 0.5, np.array([-3.0, -1.0, -0.5, 0.4, 0.9, 2.5, 4.0])):
        plan = oracle_mod.make_plan(lofar_like(8), None, phi)
        xv, h = 0.3, 30.0
        y = h - 0.7 * (phi - xv) ** 2      # amplitudes (y = |F| >= 0)
        assert np.all(y > 0)
        r = oracle_mod.peaks(plan, y[None, :], np.zeros((1, phi.size)))
        assert r["kstar"][0] == int(np.argmax(y))
        assert abs(r["peak_phi"][0] - xv) < 1e-13 and abs(r["peak_amp"][0] - h) < 1e-13
    plan = oracle_mod.make_plan(lofar_like(8), None, np.arange(5.0))
    r = oracle_mod.peaks(plan, np.array([[5.0, 4, 3, 2, 1], [1, 2, 3, 4, 5.0], [1, 3, 3, 1, 0]]), np.zeros((3, 5)))
    assert list(r["kstar"]) == [0, 4, 1]                       # edges; lowest index on ties
    assert list(r["peak_phi"][:2]) == [0.0, 4.0] and list(r["peak_amp"][:2]) == [5.0, 5.0]
    # uniform-grid closed form of A8 for a generic concave triple
    ym, y0, yp = 1.0, 3.0, 2.5
    r = oracle_mod.peaks(plan, np.array([[0, ym, y0, yp, 0.0]]), np.zeros((1, 5)))
    delta = 0.5 * (ym - yp) / (ym - 2 * y0 + yp)
    assert abs(r["peak_phi"][0] - (2.0 + delta)) < 1e-14
    assert abs(r["peak_amp"][0] - (y0 - 0.25 * (ym - yp) * delta)) < 1e-14


def test_p12_pa_recovery_for_on_grid_point_source(oracle_mod):
    """A9/A10: chi0 of a point source is recovered by pa_zero = 0.5 atan2(FU,FQ) - phi_peak lam0^2."""
    nu = lofar_like(200, 1.0e9, 2.0e9)
    phi = np.arange(-100, 101) * 2.0
    plan = oracle_mod.make_plan(nu, None, phi)
    chi0, phi0, A = 0.3, 38.0, 0.7
    P = A * np.exp(2j * (chi0 + phi0 * plan.lam2))
    FQ, FU = oracle_mod.synth_table(plan, P.real.astype(np.float32)[None], P.imag.astype(np.float32)[None])
    r = oracle_mod.peaks(plan, FQ, FU)
    assert phi[r["kstar"][0]] == phi0
    assert abs(r["peak_phi"][0] - phi0) < 1e-6 and abs(r["peak_amp"][0] - A) < 1e-6
    assert abs(r["pa_zero"][0] - chi0) < 1e-6
    assert -np.pi / 2 <= r["pa_zero"][0] < np.pi / 2


def test_p12_pa_zero_wraps_to_half_open_interval(oracle_mod):
    """Reading A9: pa_zero = pa_lambda0 - phi_peak lambda_0^2 wrapped to [-pi/2, pi/2) (polarisation angles are
    defined mod pi).  A one-depth grid makes phi_peak = phi[0], so the wrapped argument is known in closed form;
    expected values are written out as numbers on both sides of +-pi/2, after one and after several turns.
    Catches: wrapping mod 2 pi, a closed upper end, a sign error for negative arguments."""
    nu = np.array([150e6, 150e6])                      # lambda_0^2 = (c/150 MHz)^2 exactly, whatever the weights
    l0 = (C / 150e6) ** 2
    cases = [  # (pa_lambda0, rotation phi*l0, expected pa_zero)
        (0.6, 1.0, -0.4),                              # no wrap
        (-0.7, 1.0, -1.7 + np.pi),                     # below -pi/2 -> + pi  = 1.4415926535897931
        (1.5, -0.2, 1.7 - np.pi),                      # above +pi/2 -> - pi  = -1.4415926535897931
        (0.25, 10.0, 0.25 - 10.0 + 3 * np.pi),         # several turns        = -0.3252220392306207
        (-0.25, -10.0, -0.25 + 10.0 - 3 * np.pi),      #                      = 0.3252220392306207
        (0.0, -np.pi / 2, -np.pi / 2),                 # +pi/2 exactly maps to the closed lower end
    ]
    assert abs(cases[1][2] - 1.4415926535897931) < 1e-15 and abs(cases[3][2] + 0.3252220392306207) < 1e-14
    for pa, rot, want in cases:
        plan = oracle_mod.make_plan(nu, None, [rot / l0])
        assert abs(plan.lambda0_sq - l0) < 1e-15
        FQ, FU = np.array([[np.cos(2 * pa)]]), np.array([[np.sin(2 * pa)]])
        r = oracle_mod.peaks(plan, FQ, FU)
        assert abs(r["pa_lambda0"][0] - pa) < 1e-15
        assert abs(r["pa_zero"][0] - want) < 1e-13, (pa, rot, r["pa_zero"][0], want)
        assert -np.pi / 2 <= r["pa_zero"][0] < np.pi / 2
    # four-quadrant arctangent (A9 "atan2 for tan^-1(U/Q)"): Q < 0 must not fold onto Q > 0
    plan = oracle_mod.make_plan(nu, None, [0.0])
    r = oracle_mod.peaks(plan, np.array([[-1.0], [-1.0]]), np.array([[1e-9], [-1e-9]]))
    assert abs(r["pa_lambda0"][0] - np.pi / 2) < 1e-8 and abs(r["pa_lambda0"][1] + np.pi / 2) < 1e-8


def test_p12_nonfinite_line_of_sight_has_no_peak(oracle_mod):
    """Reading A17: P:L123 defines phi_peak as the depth "where |F~(phi)| is maximum"; with a NaN or Inf in |F|
    the maximum does not exist.  Non-finite samples propagate (rmsynth.h), so such a line of sight reports
    k* = -1 and NaN maps, and its finite neighbours are untouched.  Catches: a NaN silently skipped by `>`
    (the peak of the remaining samples reported as if nothing happened)."""
    plan = oracle_mod.make_plan(lofar_like(8), None, np.arange(5.0))
    FQ = np.array([[1.0, 3, 2, 1, 0], [1.0, np.nan, 2, 1, 0], [1.0, 3, 2, np.inf, 0], [0.0, 1, 5, 1, 0]])
    FU = np.zeros_like(FQ)
    FU[3, 2] = -np.inf
    r = oracle_mod.peaks(plan, FQ, FU)
    assert list(r["kstar"]) == [1, -1, -1, -1]
    for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
        assert np.isfinite(r[k][0]) and np.all(np.isnan(r[k][1:])), k


# ---------------------------------------------------------------- P13: slab generator
def test_p13_slab_signal_matches_quadrature():
    """The generator's Faraday-thick slab equals Eq. 4 integrated numerically."""
    import torch
    import rmsynth_inputs as ri
    cfg = ri.scaled(ri.CONFIGS[2], 4)
    nu, w, _ = ri.grids(cfg)
    lam2 = (C / nu) ** 2
    p = torch.arange(cfg.n_pix)
    Q, U = ri._pixel_signal(cfg, p, torch.as_tensor(lam2), w)
    u = lambda s: ri.hash_u01(cfg.seed, s, p).numpy()
    n_src = np.floor(4 * u(10)).astype(int)
    for pix in range(4):
        ref = np.zeros(cfg.n_chan, dtype=complex)
        for j in range(3):
            if n_src[pix] > j:
                A, chi, ph = 0.1 + 0.9 * u(11 + 3 * j)[pix], np.pi * u(12 + 3 * j)[pix], -80 + 160 * u(13 + 3 * j)[pix]
                ref += A * np.exp(2j * (chi + ph * lam2))
        A, chi, phc, D = 0.1 + 0.9 * u(30)[pix], np.pi * u(31)[pix], -80 + 160 * u(32)[pix], 1 + 4 * u(33)[pix]
        x = np.linspace(phc - D / 2, phc + D / 2, 20001)          # F(phi) = A e^{2i chi}/D on the slab
        integrand = (A / D) * np.exp(2j * (chi + x[None, :] * lam2[:, None]))
        ref += np.trapezoid(integrand, x, axis=1)
        got = Q[pix].numpy() + 1j * U[pix].numpy()
        assert np.max(np.abs(got - ref)) < 1e-6


def test_generator_is_counter_based_and_layout_consistent():
    import torch
    import rmsynth_inputs as ri
    cfg = ri.scaled(ri.CONFIGS[2], 8)
    Ql, Ul = ri.generate_cube(cfg, layout="los", chunk=7)
    Qf, Uf = ri.generate_cube(cfg, layout="freq", chunk=64)
    assert torch.equal(Ql, Qf.T) and torch.equal(Ul, Uf.T)
    q, u = ri.gather_los(Qf, Uf, "freq", [5, 63, 0])
    assert np.array_equal(q, Ql[[5, 63, 0]].numpy()) and np.array_equal(u, Ul[[5, 63, 0]].numpy())
    nu, w, phi = ri.grids(ri.CONFIGS[2])
    assert (w == 0).sum() == 80 and phi.size == 801 and phi[0] == -100 and phi[-1] == 100
    assert [ri.CONFIGS[i].n_phi for i in range(1, 6)] == [101, 801, 1001, 501, 401]
