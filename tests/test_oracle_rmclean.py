"""Pins of the RM-CLEAN oracle (scope row NEXT-3).  CPU only.

The paper only names the procedure ("a procedure called RM-CLEAN (Heald 2009)", footnote 6 P:L151);
the loop is the reading C1-C8 recorded in DESIGN.md and in oracle/rmsynth_oracle.c.  What pins it is mathematics:
the decomposition identity that holds after every iteration, the closed form for an on-grid point source (a
geometric series in 1 - gain), the behaviour for two well separated sources, and the stop rules.  Each test says
which plausible mistake it catches.
"""
import numpy as np

C = 299792458.0


def make(oracle_mod, n_chan=96, n_phi=161, dphi=1.5, flag=True, seed=0):
    rng = np.random.default_rng(seed)
    nu = np.linspace(1.0e9, 1.8e9, n_chan)
    w = rng.uniform(0.3, 1.0, n_chan)
    if flag:
        w[rng.random(n_chan) < 0.15] = 0.0
    phi = (np.arange(n_phi) - n_phi // 2) * dphi
    return oracle_mod.make_plan(nu, w, phi), rng


def dirty_of_point_sources(oracle_mod, plan, comps):
    """F~(phi_k) = sum_s A_s R(phi_k - phi_s) for components ON the grid: exactly what Eq. 11 gives for
    P(lambda^2) = sum_s A_s exp(2i phi_s (lambda^2 - lambda_0^2)) (the P4 identity), formed from R itself."""
    F = np.zeros(plan.phi.size, dtype=complex)
    for k_s, A in comps:
        F += A * oracle_mod.rmsf(plan, plan.phi - plan.phi[k_s])
    return F


def convolve_with_beam(oracle_mod, plan, model):
    """sum_j m_j R(phi_k - phi_j), written as a dense matrix product (independent of the oracle's indexing of Rdw)."""
    n = plan.phi.size
    B = np.empty((n, n), dtype=complex)
    for j in range(n):
        B[:, j] = oracle_mod.rmsf(plan, plan.phi - plan.phi[j])
    return model @ B.T


def test_c_identity_model_convolved_plus_residual_is_the_dirty_spectrum(oracle_mod):
    """After ANY number of iterations  sum_j m_j R(phi_k - phi_j) + r_k = F~_k  exactly (each step moves c R from the
    residual into the model).  Random complex spectra, several gains and iteration counts.
    Catches: wrong index into the double-width RMSF (k - k* vs k* - k, off by one), conj(R), gain applied twice."""
    plan, rng = make(oracle_mod)
    F = rng.standard_normal((5, plan.phi.size)) + 1j * rng.standard_normal((5, plan.phi.size))
    for gain, iters in ((0.1, 1), (0.3, 7), (1.0, 3), (0.05, 200)):
        out = oracle_mod.rmclean(plan, F.real, F.imag, gain=gain, cutoff=0.0, max_iter=iters, restore=False)
        assert np.all(out["n_iter"] == iters)
        back = convolve_with_beam(oracle_mod, plan, out["model"]) + out["residual"]
        assert np.max(np.abs(back - F)) < 1e-12


def test_c_zero_iterations_and_cutoff_above_the_peak_are_the_identity(oracle_mod):
    """max_iter = 0, or a cutoff above max|F|: nothing is subtracted (C3 stops BEFORE subtracting)."""
    plan, rng = make(oracle_mod, seed=1)
    F = rng.standard_normal((3, plan.phi.size)) + 1j * rng.standard_normal((3, plan.phi.size))
    for kw in (dict(max_iter=0, cutoff=0.0), dict(max_iter=50, cutoff=float(np.abs(F).max()) * 1.0001)):
        out = oracle_mod.rmclean(plan, F.real, F.imag, gain=0.2, fwhm=3.0, **kw)
        assert np.all(out["n_iter"] == 0) and np.all(out["model"] == 0)
        assert np.array_equal(out["residual"], F) and np.array_equal(out["restored"], F)


def test_c_on_grid_point_source_is_a_geometric_series(oracle_mod):
    """One component of amplitude A on grid sample k0: the dirty spectrum is A R(phi - phi_k0), its maximum sits at k0
    (|R| <= 1 = R(0)), so every iteration picks k0 and after n iterations
        model_k0 = A (1 - (1 - g)^n),  all other model samples 0,  residual = (1 - g)^n F~.
    Catches: gain missing or squared, component taken from |r| instead of the complex r, residual not updated at k*."""
    plan, _ = make(oracle_mod, seed=2)
    k0, A = 47, 0.8 * np.exp(1.1j)
    F = dirty_of_point_sources(oracle_mod, plan, [(k0, A)])
    assert int(np.argmax(np.abs(F))) == k0
    for g, n in ((0.1, 25), (0.5, 6), (1.0, 1)):
        out = oracle_mod.rmclean(plan, F.real[None], F.imag[None], gain=g, cutoff=0.0, max_iter=n, restore=False)
        want = A * (1 - (1 - g) ** n)
        m = out["model"][0]
        assert abs(m[k0] - want) < 1e-13
        assert np.count_nonzero(m) == 1
        assert np.max(np.abs(out["residual"][0] - (1 - g) ** n * F)) < 1e-13
    # with a cutoff the loop stops at the first n with (1-g)^n |A| < cutoff
    g, cutoff = 0.2, 0.01
    out = oracle_mod.rmclean(plan, F.real[None], F.imag[None], gain=g, cutoff=cutoff, max_iter=1000, restore=False)
    n_expected = int(np.ceil(np.log(cutoff / abs(A)) / np.log(1 - g)))
    assert out["n_iter"][0] == n_expected
    assert abs(out["residual"][0][k0]) < cutoff <= abs(out["residual"][0][k0]) / (1 - g)


def test_c_two_separated_sources_give_two_components(oracle_mod):
    """Two on-grid components on a grid sampled at about the RMSF width (beam matrix condition number ~5, so the
    decomposition with zero residual is unique), cleaned deep: the model converges to exactly those two samples with
    their amplitudes -- sidelobe cross-talk is what CLEAN removes -- and the residual to zero.
    Catches: beam not centred on k* (components smear to neighbours), wrong sign of the subtraction (divergence)."""
    plan, _ = make(oracle_mod, n_chan=128, n_phi=25, dphi=60.0, flag=False, seed=3)
    n = plan.phi.size
    B = np.array([oracle_mod.rmsf(plan, plan.phi - plan.phi[j]) for j in range(n)]).T
    assert np.linalg.cond(B) < 10.0
    comps = [(8, 1.0 * np.exp(0.3j)), (16, 0.45 * np.exp(-2.0j))]
    F = dirty_of_point_sources(oracle_mod, plan, comps)
    out = oracle_mod.rmclean(plan, F.real[None], F.imag[None], gain=0.2, cutoff=1e-10, max_iter=5000, restore=False)
    m = out["model"][0]
    assert out["n_iter"][0] < 1000 and np.max(np.abs(out["residual"][0])) < 1e-10
    assert np.max(np.abs(convolve_with_beam(oracle_mod, plan, m[None])[0] - F)) < 2e-10
    for k_s, A in comps:
        assert abs(m[k_s] - A) < 1e-8
    assert np.max(np.abs(np.delete(m, [k for k, _ in comps]))) < 1e-8
    assert np.max(np.abs(np.linalg.solve(B, F) - m)) < 1e-8      # the unique solution of B m = F~


def test_c_restoring_beam_is_a_real_gaussian_of_the_given_fwhm(oracle_mod):
    """C5 by value: a single clean component restored with FWHM w has half its amplitude at +-w/2 and the
    component's own phase everywhere; the residual is added unchanged."""
    plan, _ = make(oracle_mod, n_phi=201, dphi=0.5, seed=4)
    k0, A, fwhm = 100, 2.0 * np.exp(0.7j), 6.0
    F = dirty_of_point_sources(oracle_mod, plan, [(k0, A)])
    out = oracle_mod.rmclean(plan, F.real[None], F.imag[None], gain=1.0, cutoff=0.0, max_iter=1, fwhm=fwhm)
    m, r, s = out["model"][0], out["residual"][0], out["restored"][0]
    assert abs(m[k0] - A) < 1e-14
    g = s - r                                     # the Gaussian part
    half = int(round(fwhm / 2 / 0.5))             # sample at +w/2
    assert abs(g[k0] - A) < 1e-13
    assert abs(g[k0 + half] - 0.5 * A) < 1e-13 and abs(g[k0 - half] - 0.5 * A) < 1e-13
    x = plan.phi - plan.phi[k0]
    sigma = fwhm / (2 * np.sqrt(2 * np.log(2)))
    assert np.max(np.abs(g - A * np.exp(-x ** 2 / (2 * sigma ** 2)))) < 1e-13


def test_c_argmax_ties_edges_and_margin(oracle_mod):
    """Lowest index wins an exact tie (as A8 for the peak maps); components at the grid edges use the one-sided part
    of the double-width beam; min_margin reports how close the decision came to a tie."""
    plan, _ = make(oracle_mod, n_phi=9, dphi=40.0, flag=False, seed=5)
    F = np.zeros((3, 9), dtype=complex)
    F[0, [2, 6]] = 1.0          # exact tie -> index 2
    F[1, 0] = 1.0               # first sample
    F[2, 8] = 1.0j              # last sample
    out = oracle_mod.rmclean(plan, F.real, F.imag, gain=0.5, cutoff=0.0, max_iter=1, restore=False)
    assert np.flatnonzero(out["model"][0]).tolist() == [2] and out["min_margin"][0] == 0.0
    assert np.flatnonzero(out["model"][1]).tolist() == [0] and np.flatnonzero(out["model"][2]).tolist() == [8]
    assert out["min_margin"][1] == 1.0
    R = oracle_mod.rmsf(plan, plan.phi - plan.phi[0])
    assert np.max(np.abs(out["residual"][1] - (F[1] - 0.5 * R))) < 1e-15


def test_c_nonfinite_line_of_sight_is_left_alone(oracle_mod):
    """Reading C7 / A17: no CLEAN of a spectrum that holds a NaN; its neighbours are cleaned as usual."""
    plan, rng = make(oracle_mod, n_phi=33, seed=6)
    F = rng.standard_normal((3, 33)) + 1j * rng.standard_normal((3, 33))
    F[1, 7] = np.nan
    out = oracle_mod.rmclean(plan, F.real, F.imag, gain=0.1, max_iter=10, fwhm=4.0)
    assert out["n_iter"].tolist() == [10, 0, 10] and np.all(out["model"][1] == 0)
    assert np.isnan(out["residual"][1][7]) and np.array_equal(out["residual"][1][:7], F[1][:7])
