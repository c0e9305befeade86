"""GPU tests of rmsynth_execute_fft (scope row NEXT-4, the paper's "FFT instead of DFT"), through the C-ABI.

It is an approximation, so there are two comparisons: (1) against the NUFFT oracle (the same algorithm step by step in
FP64): what is left is FP32 rounding of the spreading and of the FFT, 5e-6 T_p; (2) against the EXACT oracle
(oracle_table): the error bound the header states, eps(W, sigma) T_p, which must shrink with the window width.
"""
import numpy as np
import pytest
import torch

import rmsynth_inputs as ri
from parity import oracle_reference

pytestmark = pytest.mark.gpu
LAYOUTS = [("los", "los"), ("los", "phi"), ("freq", "los"), ("freq", "phi")]


@pytest.fixture(scope="module")
def b():
    assert torch.cuda.is_available(), "gpu tests need a B200"
    from paper_1810_06250_b200 import binding
    return binding


def run_fft(b, plan, q, u, lin, lout, **kw):
    n_pix, n_phi = q.shape[0], plan.n_phi
    layout = (b.IN_FREQ_MAJOR if lin == "freq" else 0) | (b.OUT_PHI_MAJOR if lout == "phi" else 0)
    dq = torch.from_numpy(q if lin == "los" else np.ascontiguousarray(q.T)).cuda()
    du = torch.from_numpy(u if lin == "los" else np.ascontiguousarray(u.T)).cuda()
    shape = (n_pix, n_phi) if lout == "los" else (n_phi, n_pix)
    fq = torch.full(shape, float("nan"), device="cuda")
    fu = torch.full(shape, float("nan"), device="cuda")
    plan.execute_fft(dq, du, n_pix, layout, fq, fu, **kw)
    torch.cuda.synchronize()
    back = lambda t: t.cpu().numpy() if lout == "los" else t.cpu().numpy().T
    return back(fq).astype(np.float64) + 1j * back(fu)


@pytest.mark.parametrize("lin,lout", LAYOUTS)
@pytest.mark.parametrize("cfg_id,n_pix", [(1, 301), (2, 130), (5, 1031), (4, 67), (3, 75)])
def test_fft_variant_matches_nufft_oracle_and_the_exact_sum(b, oracle_mod, lin, lout, cfg_id, n_pix):
    from oracle import nufft_oracle as nf
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(5, 5 + n_pix))
    q, u = q.numpy(), u.numpy()
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    exact = FQ + 1j * FU
    approx = nf.nufft_synth(nf.nufft_plan(op.lam2, op.w, op.phi, op.K, op.lambda0_sq, sigma=2.0, W=6), q, u)
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_fft(b, plan, q, u, lin, lout)
    e_alg = np.max(np.abs(got - approx) / T[:, None])
    e_exact = np.max(np.abs(got - exact) / T[:, None])
    print(f"cfg{cfg_id} {lin}->{lout}: vs NUFFT oracle {e_alg:.2e} T_p, vs exact {e_exact:.2e} T_p")
    assert e_alg <= 5e-6 and e_exact <= 8e-6
    plan.destroy()


def test_fft_variant_error_shrinks_with_the_window(b, oracle_mod):
    """The stated bound eps(W, sigma): about a decade per unit of W until FP32 rounding (~1e-6 T_p) takes over."""
    cfg = ri.CONFIGS[2]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(0, 64))
    q, u = q.numpy(), u.numpy()
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    exact = FQ + 1j * FU
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE)
    errs = {}
    for W, bound in ((2, 3e-2), (4, 3e-4), (6, 8e-6), (8, 5e-6)):
        errs[W] = float(np.max(np.abs(run_fft(b, plan, q, u, "freq", "phi", window=W) - exact) / T[:, None]))
        assert errs[W] <= bound, (W, errs[W])
    assert errs[2] > errs[4] > errs[6]
    e_os = float(np.max(np.abs(run_fft(b, plan, q, u, "freq", "phi", window=4, oversampling=4.0) - exact) / T[:, None]))
    assert e_os < errs[4]
    print({k: f"{v:.1e}" for k, v in errs.items()}, f"W=4 at oversampling 4: {e_os:.1e}")
    plan.destroy()


def test_fft_variant_flags_nonfinite_and_errors(b, oracle_mod):
    cfg = ri.CONFIGS[2]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(0, 40))
    q, u = q.numpy().copy(), u.numpy().copy()
    q[:, w == 0] = np.nan                      # flagged channels are never read (F6 / A13)
    u[7, np.flatnonzero(w > 0)[3]] = np.inf    # an unflagged non-finite sample poisons its own line of sight only
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_fft(b, plan, q, u, "freq", "phi")
    good = np.setdiff1d(np.arange(40), [7])
    assert np.max(np.abs(got[good] - (FQ + 1j * FU)[good]) / T[good, None]) <= 8e-6
    assert not np.all(np.isfinite(got[7]))
    t = torch.zeros(4, 4, device="cuda")
    for kw in (dict(window=5), dict(window=18), dict(oversampling=1.0)):
        with pytest.raises(b.RmsynthError) as e:
            plan.execute_fft(t, t, 4, 0, t, t, **kw)
        assert e.value.status == b.EINVAL
    plan.destroy()
    plan = b.Plan(np.linspace(1e9, 2e9, 16), None, np.array([-3.0, 0.0, 1.0, 7.0, 9.0]), scheme=b.SCHEME_FP32_TABLE)
    with pytest.raises(b.RmsynthError) as e:
        plan.execute_fft(t, t, 1, 0, t, t)
    assert e.value.status == b.EUNSUPPORTED
    plan.destroy()


def test_fft_variant_on_the_7000_depth_grid(b, oracle_mod):
    """The shape the variant is for (856 channels -> 7000 depths; fine grid 16384, one line of sight per CTA batch)."""
    cfg = ri.CONFIGS[7]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(3, 3 + 37))
    q, u = q.numpy(), u.numpy()
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE)
    got = run_fft(b, plan, q, u, "freq", "phi")
    err = float(np.max(np.abs(got - (FQ + 1j * FU)) / T[:, None]))
    print(f"7000 depths: vs exact {err:.2e} T_p")
    assert err <= 8e-6
    plan.destroy()
