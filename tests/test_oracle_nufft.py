"""Pins of the NUFFT oracle (scope row NEXT-4, the paper's "FFT instead of DFT").  CPU only.

The variant is an APPROXIMATION of Eqs. 15-16, so what pins it is (a) special cases where it must be exact whatever
the window, and (b) its distance to the exact FP64 sum (oracle_table), which must fall with the window width W and
the oversampling sigma as the theory of the Kaiser-Bessel window says (roughly a decade per unit of W at sigma = 2).
"""
import numpy as np
import pytest

C = 299792458.0


def setup(oracle_mod, n_chan=200, n_phi=257, dphi=0.8, seed=0, flag=True):
    rng = np.random.default_rng(seed)
    nu = np.linspace(1.1e9, 1.9e9, n_chan)
    w = rng.uniform(0.3, 1.0, n_chan)
    if flag:
        w[rng.random(n_chan) < 0.1] = 0.0
    phi = -90.0 + np.arange(n_phi) * dphi
    op = oracle_mod.make_plan(nu, w, phi)
    Q = rng.standard_normal((6, n_chan)).astype(np.float32)
    U = rng.standard_normal((6, n_chan)).astype(np.float32)
    return op, Q, U


def exact(oracle_mod, op, Q, U):
    FQ, FU = oracle_mod.synth_table(op, Q, U)
    return FQ + 1j * FU, oracle_mod.tolerance_scale(op, Q, U)


def test_f_single_channel(oracle_mod):
    """One channel: g = c psi(. - u), so G is the window's (aliased) transform times a phase ramp and after deapodisation
    F_k = c e^{-2 pi i (k - kc) t} up to the aliases alone: 1.4e-4, 4e-9, 1e-13 of |c| for W = 4, 8, 12 at oversampling
    ~4.  Pins the deapodisation factor, the sign of the FFT, the pre-phase at the centre depth and the mapping
    t = dphi x / pi.  Catches: missing 1/psihat, conjugated FFT, u computed from lambda^2 without lambda_0^2, an
    un-centred output band (error of order one)."""
    from oracle import nufft_oracle as nf
    nu = np.array([1.3e9, 1.7e9])
    w = np.array([1.0, 0.0])                       # the second channel is flagged: lambda_0^2 = lambda_1^2 + nothing
    phi = -40.0 + np.arange(65) * 1.25
    op = oracle_mod.make_plan(nu, w, phi, lambda0_mode=2, lambda0_in=0.01)
    Q = np.array([[0.7, 5.0]], dtype=np.float32)
    U = np.array([[-0.2, 5.0]], dtype=np.float32)
    ref, T = exact(oracle_mod, op, Q, U)
    for W, tol in ((4, 5e-4), (8, 2e-8), (12, 1e-12)):
        pl = nf.nufft_plan(op.lam2, op.w, op.phi, op.K, op.lambda0_sq, sigma=2.0, W=W)
        got = nf.nufft_synth(pl, Q, U)
        assert np.max(np.abs(got - ref)) < tol * T[0], (W, np.max(np.abs(got - ref)))


def test_f_error_falls_with_window_width_and_oversampling(oracle_mod):
    """Distance to the exact sum, relative to T_p (the north_star's scale): bounded by the table below (about 3 x the
    measured values) and strictly decreasing along W -- the stated error bound of the variant: roughly a decade per
    unit of W at oversampling 4 (sigma = 2 on this 257-depth grid gives M = 1024) and per 1.2 units at oversampling 2
    (sigma = 1.25 gives M = 512).
    Catches: a wrong beta (the error stalls around 1e-3), an off-by-one in the first spread point (error ~ 1e-1)."""
    from oracle import nufft_oracle as nf
    op, Q, U = setup(oracle_mod)
    ref, T = exact(oracle_mod, op, Q, U)
    bound = {(2.0, 4): 5e-5, (2.0, 6): 3e-7, (2.0, 8): 2e-9, (2.0, 10): 1e-11, (1.25, 4): 3e-4, (1.25, 6): 4e-6, (1.25, 8): 5e-8,
             (1.25, 12): 1e-11}
    errs = {}
    for (sigma, W), b in bound.items():
        pl = nf.nufft_plan(op.lam2, op.w, op.phi, op.K, op.lambda0_sq, sigma=sigma, W=W)
        got = nf.nufft_synth(pl, Q, U)
        errs[(sigma, W)] = float(np.max(np.abs(got - ref) / T[:, None]))
        assert errs[(sigma, W)] < b, (sigma, W, errs[(sigma, W)])
    assert errs[(2.0, 4)] > errs[(2.0, 6)] > errs[(2.0, 8)] > errs[(2.0, 10)]
    assert errs[(1.25, 4)] > errs[(1.25, 6)] > errs[(1.25, 8)] > errs[(1.25, 12)]
    assert all(errs[(1.25, W)] > errs[(2.0, W)] for W in (4, 6, 8))        # more oversampling, smaller error
    print({k: f"{v:.1e}" for k, v in errs.items()})


def test_f_grid_is_periodic_and_flags_are_skipped(oracle_mod):
    """u is taken mod M (F2): a window that straddles the end of the fine grid wraps around; flagged channels holding
    NaN do not reach the result (F6 / A13)."""
    from oracle import nufft_oracle as nf
    op, Q, U = setup(oracle_mod, seed=3)
    Q = Q.copy()
    Q[:, op.w == 0] = np.nan
    ref, T = exact(oracle_mod, op, Q, U)
    pl = nf.nufft_plan(op.lam2, op.w, op.phi, op.K, op.lambda0_sq)
    # lambda_0^2 is the weighted mean, so x_i and with it t_i changes sign across the band: some windows wrap
    assert np.any(pl["u"] < 4) and np.any(pl["u"] > pl["M"] - 4)
    got = nf.nufft_synth(pl, Q, U)
    assert np.all(np.isfinite(got)) and np.max(np.abs(got - ref) / T[:, None]) < 5e-9
    assert pl["M"] == 1024 and pl["n"] == 257


def test_f_needs_a_uniform_grid(oracle_mod):
    from oracle import nufft_oracle as nf
    op = oracle_mod.make_plan(np.linspace(1e9, 2e9, 8), None, np.array([-3.0, 0.0, 1.0, 7.0]))
    with pytest.raises(ValueError):
        nf.nufft_plan(op.lam2, op.w, op.phi, op.K, op.lambda0_sq)
