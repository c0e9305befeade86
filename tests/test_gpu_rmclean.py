"""GPU parity of rmsynth_rmclean (scope row NEXT-3) against oracle_rmclean, through the C-ABI binding.

Inputs: the oracle's own dirty spectra of seeded synthetic lines of sight, rounded to FP32 (what rmsynth_execute hands
to a user) -- never anything the CUDA path produced.  Rules:
  * every line of sight: the decomposition identity  model * R + residual = dirty  holds to FP32 accuracy, iteration
    counts never exceed max_iter, and a cutoff is respected (|residual| peak < cutoff or max_iter reached);
  * lines of sight whose arg-max decisions were never within the FP32 error budget of a tie in the oracle
    (min_margin > 3 x tolerance): same number of iterations, the same component positions, model / residual /
    restored within tolerance.  Where a decision was that close, both sequences are valid CLEANs and only the
    properties are checked (the same idea as the peak-index rule of the north_star).
Tolerance (FP32 loop): each subtraction rounds to 2^-24 of |c R| and |r|, R itself to 2^-24; the components shrink
geometrically, so after n iterations the residual carries a few 2^-24 (sum |c| + max|F~|): 1e-6 max|F~| (1 + gain n / 20)
(measured: 2e-7).
A decision counts as clear of a tie when the oracle's margin |r_k*| - |r_second| exceeds 3 tolerances (15 x the measured error).
"""
import numpy as np
import pytest
import torch

import rmsynth_inputs as ri

pytestmark = pytest.mark.gpu
TOL = 1e-6


@pytest.fixture(scope="module")
def b():
    assert torch.cuda.is_available(), "gpu tests need a B200"
    from paper_1810_06250_b200 import binding
    return binding


def dirty_cube(oracle_mod, cfg_id, n_pix, n_phi=None, start=0):
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    if n_phi is not None:
        phi = phi[0] + np.arange(n_phi) * cfg.dphi
    q, u = ri.generate_pixels(cfg, torch.arange(start, start + n_pix))
    op = oracle_mod.make_plan(nu, w, phi)
    FQ, FU = oracle_mod.synth_table(op, q.numpy(), u.numpy())
    return cfg, nu, w, phi, op, FQ.astype(np.float32), FU.astype(np.float32)


def run_clean(b, plan, FQ, FU, lout, gain, cutoff, max_iter, fwhm, restore=True):
    n_pix, n_phi = FQ.shape
    layout = b.OUT_PHI_MAJOR if lout == "phi" else 0
    put = lambda a: torch.from_numpy(np.ascontiguousarray(a.T if lout == "phi" else a)).cuda()
    shape = (n_phi, n_pix) if lout == "phi" else (n_pix, n_phi)
    new = lambda: torch.full(shape, float("nan"), device="cuda")
    mq, mu, rq, ru = new(), new(), new(), new()
    sq, su = (new(), new()) if restore else (None, None)
    it = torch.full((n_pix,), -1, dtype=torch.int32, device="cuda")
    plan.rmclean(put(FQ), put(FU), n_pix, layout, gain, cutoff, max_iter, mq, mu, rq, ru, sq, su, it, fwhm=fwhm)
    torch.cuda.synchronize()
    back = lambda t: (t.cpu().numpy().T if lout == "phi" else t.cpu().numpy()).astype(np.float64)
    out = dict(model=back(mq) + 1j * back(mu), residual=back(rq) + 1j * back(ru), n_iter=it.cpu().numpy())
    out["restored"] = back(sq) + 1j * back(su) if restore else None
    return out


def check(oracle_mod, op, FQ, FU, got, ref, gain, cutoff, max_iter, what):
    F = FQ.astype(np.float64) + 1j * FU.astype(np.float64)
    n_pix, n = F.shape
    Fmax = np.abs(F).max(axis=1)
    tol = TOL * Fmax * (1 + gain * max_iter / 20)
    # properties, every line of sight
    # model * R: the beam centred on depth j is R((k - j) dphi) (reading C1) -- one RMSF call on the double-width grid, then
    # a sum over the (few) non-zero components of every line of sight
    dphi = float(op.phi[1] - op.phi[0]) if n > 1 else 1.0
    Rdw = oracle_mod.rmsf(op, dphi * (np.arange(2 * n - 1) - (n - 1)))
    back = got["residual"].copy()
    for p_, j_ in zip(*np.nonzero(got["model"])):
        back[p_] += got["model"][p_, j_] * Rdw[n - 1 - j_: 2 * n - 1 - j_]
    assert np.all(np.abs(back - F).max(axis=1) <= tol + 1e-30), f"{what}: identity broken by {np.abs(back - F).max()}"
    assert got["n_iter"].min() >= 0 and got["n_iter"].max() <= max_iter
    peak = np.abs(got["residual"]).max(axis=1)
    assert np.all((got["n_iter"] == max_iter) | (peak < cutoff + tol)), f"{what}: stopped early above the cutoff"
    # element-wise parity where the oracle's decisions were clear of a tie
    stable = ref["min_margin"] > 3 * tol
    assert stable.mean() > 0.5, f"{what}: too few decision-stable lines of sight ({stable.mean():.2f}) for a meaningful test"
    s = stable
    assert np.array_equal(got["n_iter"][s], ref["n_iter"][s]), f"{what}: iteration counts differ"
    assert np.array_equal(got["model"][s] != 0, ref["model"][s] != 0), f"{what}: component positions differ"
    for key in ("model", "residual", "restored"):
        if got[key] is None:
            continue
        err = np.abs(got[key][s] - ref[key][s]).max(axis=1)
        assert np.all(err <= tol[s]), f"{what}: {key} off by {err.max():.3e} (tol {tol[s][err.argmax()]:.3e})"
        print(f"  {what}: {key} max err / tol = {np.max(err / tol[s]):.3f}")
    return float(stable.mean())


@pytest.mark.parametrize("lout", ["los", "phi"])
@pytest.mark.parametrize("cfg_id,n_pix,n_phi,gain,max_iter,cut_frac", [(5, 203, None, 0.1, 150, 0.3), (1, 77, None, 0.2, 60, 0.02),
                                                                      (4, 64, 501, 0.1, 40, 0.08), (3, 21, 1001, 0.3, 40, 0.5),
                                                                      (2, 19, 1100, 0.2, 30, 0.1), (7, 9, None, 0.1, 40, 0.3),
                                                                      (7, 5, 9000, 0.2, 25, 0.3)])
def test_rmclean_matches_oracle(b, oracle_mod, lout, cfg_id, n_pix, n_phi, gain, max_iter, cut_frac):
    """All four warp-kernel widths (<= 128, 256, 512, 1024 depths) and the CTA kernel (1100 depths; the paper's 7000-depth
    grid with the beam in shared memory; 9000 depths with the beam read through L2 and 28 depths per thread), ragged
    pixel counts against the 8-pixel CTA batches, both cube layouts.  The cutoff is a fraction of the median dirty
    peak, chosen so that most lines of sight stop before their arg-max decisions come within FP32 rounding of a tie
    (a CLEAN run to the noise floor meets such ties in nearly every line of sight: both sequences are then valid)."""
    cfg, nu, w, phi, op, FQ, FU = dirty_cube(oracle_mod, cfg_id, n_pix, n_phi, start=4)
    cutoff = cut_frac * float(np.median(np.abs(FQ.astype(np.float64) + 1j * FU).max(axis=1)))
    fwhm = 4.0 * cfg.dphi
    ref = oracle_mod.rmclean(op, FQ, FU, gain=gain, cutoff=cutoff, max_iter=max_iter, fwhm=fwhm)
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_clean(b, plan, FQ, FU, lout, gain, cutoff, max_iter, fwhm)
    frac = check(oracle_mod, op, FQ, FU, got, ref, gain, cutoff, max_iter, f"cfg{cfg_id} {phi.size} depths {lout}")
    print(f"cfg{cfg_id} {phi.size} depths {lout}: {frac:.2f} of the lines of sight decision-stable, iterations {ref['n_iter'].min()}..{ref['n_iter'].max()}")
    plan.destroy()


@pytest.mark.parametrize("lout", ["los", "phi"])
@pytest.mark.parametrize("n_phi", [1, 2, 5, 31, 32, 33])
def test_rmclean_grids_narrower_than_a_warp(b, oracle_mod, lout, n_phi):
    """Fewer depths than lanes: the lanes without a depth must never win the arg-max (their sentinel once sorted above
    every real |r|^2 in the unsigned reduction and ended the loop before its first iteration).  1, 2, 5 and 31 depths,
    with 32 and 33 as the neighbours on the other side; band and spacing chosen so that the RMSF is a few samples
    wide.  Noise spectra plus one source, seeded here and handed to both sides."""
    nu = np.linspace(1.0e9, 1.8e9, 96)
    dphi = 25.0
    phi = (np.arange(n_phi) - n_phi // 2) * dphi
    op = oracle_mod.make_plan(nu, None, phi)
    rng = np.random.default_rng(100 + n_phi)
    n_pix = 37
    lam2 = (299792458.0 / nu) ** 2
    src = rng.uniform(phi[0], phi[-1] + 1e-9, n_pix)[:, None]
    P = np.exp(2j * src * lam2[None, :]) * rng.uniform(0.5, 2.0, (n_pix, 1)) + 0.3 * (rng.standard_normal((n_pix, 96)) + 1j * rng.standard_normal((n_pix, 96)))
    FQ, FU = oracle_mod.synth_table(op, np.ascontiguousarray(P.real, dtype=np.float32), np.ascontiguousarray(P.imag, dtype=np.float32))
    FQ, FU = FQ.astype(np.float32), FU.astype(np.float32)
    gain, max_iter, fwhm = 0.2, 30, 2.5 * dphi
    cutoff = 0.25 * float(np.median(np.abs(FQ.astype(np.float64) + 1j * FU).max(axis=1)))
    ref = oracle_mod.rmclean(op, FQ, FU, gain=gain, cutoff=cutoff, max_iter=max_iter, fwhm=fwhm)
    assert ref["n_iter"].max() > 0, "the case must iterate to test anything"
    plan = b.Plan(nu, None, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_clean(b, plan, FQ, FU, lout, gain, cutoff, max_iter, fwhm)
    check(oracle_mod, op, FQ, FU, got, ref, gain, cutoff, max_iter, f"{n_phi} depths {lout}")
    plan.destroy()


def test_rmclean_point_source_closed_form_and_edges(b, oracle_mod):
    """On-grid point source: n iterations leave (1 - g)^n of the dirty spectrum and put A (1 - (1 - g)^n) on one sample
    (the closed form that pins the oracle) -- checked on the GPU directly; max_iter = 0 and a NaN line of sight pass
    the input through (reading C7)."""
    nu = np.linspace(1.0e9, 1.8e9, 96)
    phi = (np.arange(161) - 80) * 1.5
    op = oracle_mod.make_plan(nu, None, phi)
    k0, A, g, n = 47, 0.8 * np.exp(1.1j), 0.25, 12
    F = (A * oracle_mod.rmsf(op, phi - phi[k0]))[None, :].repeat(3, axis=0)
    F[1, 5] = np.nan
    FQ, FU = F.real.astype(np.float32), F.imag.astype(np.float32)
    plan = b.Plan(nu, None, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_clean(b, plan, FQ, FU, "los", g, 0.0, n, 3.0)
    assert got["n_iter"].tolist() == [n, 0, n]
    assert abs(got["model"][0, k0] - A * (1 - (1 - g) ** n)) < 5e-6 and np.count_nonzero(got["model"][0]) == 1
    assert np.max(np.abs(got["residual"][0] - (1 - g) ** n * (FQ[0] + 1j * FU[0]))) < 5e-6
    assert np.all(got["model"][1] == 0) and np.isnan(got["residual"][1, 5]) and np.isnan(got["restored"][1, 5])
    assert np.array_equal(got["residual"][1, 6:], (FQ[1] + 1j * FU[1])[6:].astype(np.complex128))
    got0 = run_clean(b, plan, FQ, FU, "phi", g, 0.0, 0, 3.0, restore=False)
    assert got0["n_iter"].tolist() == [0, 0, 0] and np.all(got0["model"] == 0)
    assert np.array_equal(got0["residual"][0], (FQ[0] + 1j * FU[0]).astype(np.complex128))
    plan.destroy()


def test_rmclean_argument_errors(b):
    nu = np.linspace(1e9, 2e9, 16)
    t = torch.zeros(4, 5, device="cuda")
    plan = b.Plan(nu, None, np.linspace(-10, 10, 5), scheme=b.SCHEME_FP32_TABLE)
    for kw in (dict(gain=0.0), dict(gain=1.5), dict(cutoff=-1.0), dict(max_iter=-1)):
        args = dict(gain=0.1, cutoff=0.0, max_iter=3)
        args.update(kw)
        with pytest.raises(b.RmsynthError) as e:
            plan.rmclean(t, t, 4, 0, args["gain"], args["cutoff"], args["max_iter"], t, t, t, t)
        assert e.value.status == b.EINVAL
    plan.destroy()
    plan = b.Plan(nu, None, np.array([-3.0, 0.0, 1.0, 7.0, 9.0]), scheme=b.SCHEME_FP32_TABLE)   # non-uniform grid
    with pytest.raises(b.RmsynthError) as e:
        plan.rmclean(t, t, 4, 0, 0.1, 0.0, 3, t, t, t, t)
    assert e.value.status == b.EUNSUPPORTED
    plan.destroy()
