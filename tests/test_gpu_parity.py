"""GPU parity tests proper: every call goes through the C-ABI binding and is compared with
the FP64 oracle on the same seeded inputs (run with `-m gpu` on a B200)."""
import numpy as np
import pytest
import torch

import rmsynth_inputs as ri
from parity import TOL, check_cubes, check_peaks, oracle_reference

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    assert torch.cuda.is_available(), "gpu tests need a B200"
    from paper_1810_06250_b200 import binding
    return binding


def scheme_ids(b):
    return {"tf32x3": b.SCHEME_TF32X3, "f16x3": b.SCHEME_F16X3, "fp32_table": b.SCHEME_FP32_TABLE, "fp32_sincos": b.SCHEME_FP32_SINCOS}


SCHEMES = ["tf32x3", "f16x3", "fp32_table", "fp32_sincos"]
LAYOUTS = [("los", "los"), ("los", "phi"), ("freq", "los"), ("freq", "phi")]


def run_gpu(b, plan, q_los, u_los, lin, lout, peaks=False, cubes=True, host=False):
    """q_los/u_los: host float32 [n_pix, n_chan].  Returns LOS-major numpy outputs."""
    n_pix, n_chan = q_los.shape
    n_phi = plan.n_phi
    layout = (b.IN_FREQ_MAJOR if lin == "freq" else 0) | (b.OUT_PHI_MAJOR if lout == "phi" else 0)
    dev = "cpu" if host else "cuda"
    q = torch.from_numpy(q_los if lin == "los" else np.ascontiguousarray(q_los.T)).to(dev)
    u = torch.from_numpy(u_los if lin == "los" else np.ascontiguousarray(u_los.T)).to(dev)
    shape = (n_pix, n_phi) if lout == "los" else (n_phi, n_pix)
    FQ = torch.full(shape, float("nan"), dtype=torch.float32, device=dev) if cubes else None
    FU = torch.full(shape, float("nan"), dtype=torch.float32, device=dev) if cubes else None
    maps = {}
    if peaks:
        for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
            maps[k] = torch.full((n_pix,), float("nan"), dtype=torch.float32, device=dev)
        maps["peak_index"] = torch.full((n_pix,), -1, dtype=torch.int32, device=dev)
    if host:
        plan.execute_host(q, u, n_pix, layout, FQ, FU, **maps)
    elif peaks:
        plan.execute_peaks(q, u, n_pix, layout, FQ, FU, **maps)
        torch.cuda.synchronize()
    else:
        plan.execute(q, u, n_pix, layout, FQ, FU)
        torch.cuda.synchronize()
    out = {}
    if cubes:
        out["FQ"] = FQ.cpu().numpy() if lout == "los" else FQ.cpu().numpy().T
        out["FU"] = FU.cpu().numpy() if lout == "los" else FU.cpu().numpy().T
    if peaks:
        out["maps"] = {("kstar" if k == "peak_index" else k): v.cpu().numpy() for k, v in maps.items()}
    return out


def inputs(cfg_id, n_pix, start=0):
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(start, start + n_pix))
    return cfg, nu, w, phi, q.numpy(), u.numpy()


# ------------------------------------------------------------------ plan (rows a1-a3)
@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4, 5])
def test_plan_scalars_phase_matrix_and_rmsf(b, oracle_mod, cfg_id):
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    for mode, l0 in ((0, 0.0), (1, 0.0), (2, 0.0), (2, 1.25)):
        op = oracle_mod.make_plan(nu, w, phi, mode, l0)
        gp = b.Plan(nu, w, phi, scheme=b.SCHEME_FP32_TABLE, lambda0_mode=mode, lambda0_sq=l0)
        assert abs(gp.K - op.K) <= 1e-15 * op.K and abs(gp.lambda0_sq - op.lambda0_sq) <= 1e-14 * max(op.lambda0_sq, 1)
        R = gp.rmsf()
        assert np.max(np.abs(R - oracle_mod.rmsf(op))) < 1e-11
        pe = np.linspace(phi[0] * 1.5, phi[-1] * 1.5, 77) + 0.123
        assert np.max(np.abs(gp.rmsf(pe) - oracle_mod.rmsf(op, pe))) < 1e-11
        if mode == 0:
            c, s = gp.phase_matrix()
            th = 2.0 * phi[None, :] * (op.lam2 - op.lambda0_sq)[:, None]
            kw = (op.K * op.w)[:, None]
            scale = float(kw.max())
            assert np.max(np.abs(c - kw * np.cos(th))) <= 1.2e-7 * scale
            assert np.max(np.abs(s - kw * np.sin(th))) <= 1.2e-7 * scale
        gp.destroy()


# ------------------------------------------------------------------ cubes (rows a4-a6, a9)
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("lin,lout", LAYOUTS)
@pytest.mark.parametrize("cfg_id,n_pix", [(1, 301), (2, 257), (3, 130), (4, 200), (5, 1031)])
def test_cubes_match_oracle(b, oracle_mod, scheme, lin, lout, cfg_id, n_pix):
    """Every config's grids at a pixel count spanning several tiles plus a ragged tail, all four
    layout combinations (reading A7)."""
    cfg, nu, w, phi, q, u = inputs(cfg_id, n_pix, start=7)
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, lin, lout)
    worst = check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} cfg{cfg_id} {lin}->{lout}")
    print(f"{scheme} cfg{cfg_id} {lin}->{lout}: max err/T_p = {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_full_config1_cube(b, oracle_mod, scheme):
    """BASELINE.json configs[0] in full: 64x64 pixels, LOS-major in and out."""
    cfg = ri.CONFIGS[1]
    nu, w, phi = ri.grids(cfg)
    Q, U = ri.generate_cube(cfg, "cpu")
    q, u = Q.numpy(), U.numpy()
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, "los", "los")
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} full config 1")
    plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("n_chan,n_phi,n_pix", [(1, 1, 1), (3, 2, 5), (37, 19, 129), (8, 9, 16), (129, 257, 127),
                                                (33, 513, 3), (1000, 7, 260)])
def test_odd_shapes_and_degenerate_sizes(b, oracle_mod, scheme, n_chan, n_phi, n_pix):
    rng = np.random.default_rng(n_chan * 1000 + n_phi)
    nu = np.sort(rng.uniform(0.9e9, 1.8e9, n_chan))
    w = rng.uniform(0.0, 1.0, n_chan)
    w[0] = 0.7
    phi = np.sort(rng.uniform(-300, 300, n_phi))            # non-uniform, unsorted grids are legal
    q = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    u = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    for lin, lout in LAYOUTS:
        out = run_gpu(b, plan, q, u, lin, lout)
        check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} {n_chan}x{n_phi}x{n_pix} {lin}->{lout}")
    plan.destroy()


@pytest.mark.parametrize("scheme", ["tf32x3", "f16x3"])
@pytest.mark.parametrize("n_pix,n_chan,n_phi", [(773, 40, 2100), (17925, 8, 2100), (5000, 33, 105), (128 * 2 * 75, 16, 230), (300, 8, 8000)])
def test_work_schedule_shapes(b, oracle_mod, scheme, n_pix, n_chan, n_phi):
    """The gang schedule (tc_common.cuh: WorkIter) at shapes that exercise its corners: more depth tiles than a
    third of the CTA pairs (gangs of 17-21, left-over pairs walking depth tiles sequentially), fewer pixel-tile
    pairs than gangs, more pairs than one round, one / two / three depth tiles.  Every output must be written
    exactly once: the buffers are NaN-filled and compared in full with the oracle."""
    rng = np.random.default_rng(n_pix + n_phi)
    nu = np.linspace(1.0e9, 1.6e9, n_chan)
    phi = np.linspace(-500.0, 500.0, n_phi)
    q = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    u = rng.standard_normal((n_pix, n_chan)).astype(np.float32)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, None, phi, q, u)
    plan = b.Plan(nu, None, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, "freq" if n_pix % 2 == 0 else "los", "phi", peaks=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} schedule {n_pix}x{n_chan}x{n_phi}")
    check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], float(phi[1] - phi[0]), f"{scheme} schedule")
    plan.destroy()


def test_concurrent_streams_share_a_plan(b, oracle_mod):
    """Two streams, one plan: per-call workspace (peak records, check-in counters) is keyed by stream."""
    cfg, nu, w, phi, q, u = inputs(4, 3000)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    dq, du = torch.from_numpy(q).cuda(), torch.from_numpy(u).cuda()
    outs = []
    for rep in range(3):
        for s in streams:
            idx = torch.full((3000,), -1, dtype=torch.int32, device="cuda")
            fq = torch.full((3000, plan.n_phi), float("nan"), device="cuda")
            fu = torch.full_like(fq, float("nan"))
            s.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(s):
                plan.execute_peaks(dq, du, 3000, 0, fq, fu, peak_index=idx, stream=s.cuda_stream)
            outs.append((fq, fu, idx))
    torch.cuda.synchronize()
    y = np.sqrt(FQ ** 2 + FU ** 2)
    ko = oracle_mod.peaks(op, FQ, FU)["kstar"].astype(np.int64)
    rows = np.arange(3000)
    for fq, fu, idx in outs:
        check_cubes(fq.cpu().numpy(), fu.cpu().numpy(), FQ, FU, T, "concurrent streams")
        kg = idx.cpu().numpy().astype(np.int64)
        assert kg.min() >= 0 and kg.max() < plan.n_phi
        # the index rule of check_peaks: equal, unless the oracle's |F| at the two depths differ by <= 2e-5 T_p
        assert not ((kg != ko) & (y[rows, ko] - y[rows, kg] > 2 * TOL * T)).any()
    plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_coherent_worst_case_and_dynamic_range(b, oracle_mod, scheme):
    """All channels in phase at an on-grid depth (partial sums grow to the full norm: the worst
    case for accumulator rounding), plus pixels scaled by 1e-20 .. 1e+20."""
    cfg = ri.CONFIGS[4]
    nu, w, phi = ri.grids(cfg)
    lam2 = (ri.C_M_PER_S / nu) ** 2
    n_pix = 140
    rng = np.random.default_rng(11)
    phi0 = phi[rng.integers(0, phi.size, n_pix)]
    chi = rng.uniform(0, np.pi, n_pix)
    P = np.exp(2j * (chi[:, None] + phi0[:, None] * lam2[None, :]))
    scale = 10.0 ** rng.integers(-20, 21, n_pix)
    scale[:8] = 1.0
    q = (P.real * scale[:, None]).astype(np.float32)
    u = (P.imag * scale[:, None]).astype(np.float32)
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, "freq", "phi")
    worst = check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} coherent")
    print(f"{scheme} coherent worst case: max err/T_p = {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_very_faint_cubes(b, oracle_mod, scheme):
    """Samples far below any physical flux scale (FP32's smallest normal number is 1.2e-38): lines of sight whose largest
    sample is 1e-24, 1e-26 and 1e-28 keep the parity tolerance in every scheme.  The FP16 scheme scales every 32-channel
    chunk by its own maximum, floored at 2^(eB - 112) ~ 3e-27 so that the factor the epilogue multiplies back stays a
    normal FP32 number; a chunk under the floor is scaled by the floor's power, its hi half (a multiple of 16 after
    scaling) empties and the lo half carries it alone: accuracy falls off by a factor two per factor two, down to plain
    FP16 (2^-12 per sample) -- never flushed to zero (rmsynth.h).  Lines of sight at 1e-31 check exactly that."""
    cfg = ri.CONFIGS[5]
    nu, w, phi = ri.grids(cfg)
    q, u = ri.generate_pixels(cfg, torch.arange(7, 7 + 200))
    scale = np.repeat([1e-24, 1e-26, 1e-28, 1e-31], 50)[:, None]
    amp = np.maximum(np.abs(q.numpy()), np.abs(u.numpy())).max(axis=1, keepdims=True).astype(np.float64)   # per line of sight
    q = (q.numpy().astype(np.float64) / amp * scale).astype(np.float32)
    u = (u.numpy().astype(np.float64) / amp * scale).astype(np.float32)
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    assert T.min() > 1e-34
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, "freq", "phi")
    worst = check_cubes(out["FQ"][:150], out["FU"][:150], FQ[:150], FU[:150], T[:150], f"{scheme} faint")
    err = np.hypot(out["FQ"][150:] - FQ[150:], out["FU"][150:] - FU[150:]).max(axis=1) / T[150:]
    assert np.all(np.isfinite(err)) and err.max() <= (1e-3 if scheme == "f16x3" else TOL), f"{scheme} at 1e-31: {err.max():.2e} of T_p"
    print(f"{scheme} faint cubes: max err/T_p = {worst:.2e} (1e-24 .. 1e-28), {err.max():.2e} (1e-31)")
    plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
def test_flagged_channels_full_of_interference(b, oracle_mod, scheme):
    """Reading A13: a zero-weight channel contributes nothing, whatever (finite) garbage it holds.  Samples of
    1e30 in flagged channels next to O(1) data must neither change the result nor cost accuracy (the FP16 split
    scales each 32-channel chunk by its largest sample over the channels with w > 0 only)."""
    cfg, nu, w, phi, q, u = inputs(2, 300, start=11)
    flagged = np.flatnonzero(w == 0)
    assert flagged.size == 80
    q, u = q.copy(), u.copy()
    q[::3, flagged[::2]] = 1e30
    u[1::3, flagged[1::2]] = -3e28
    # reading A13: a flagged channel is REMOVED, so NaN-blanked / overflowed planes are as harmless as finite garbage
    q[5::7, flagged[3]] = np.nan
    u[2::5, flagged[10]] = np.inf
    q[:, flagged[20]] = -np.inf
    u[:, flagged[21]] = np.nan
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    assert np.all(np.isfinite(FQ)) and np.all(T < 10)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, "freq", "phi")
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} flagged garbage")
    out = run_gpu(b, plan, q, u, "los", "los", peaks=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"{scheme} flagged garbage los")
    assert out["maps"]["kstar"].min() >= 0 and np.all(np.isfinite(out["maps"]["peak_amp"]))
    plan.destroy()


def test_auto_scheme_choice(b):
    """AUTO = FP16X3, except when the positive weights span more than 2^18 or there are < 384 channels (then 3xTF32)."""
    phi = np.linspace(-10, 10, 9)
    assert b.Plan(np.linspace(1e9, 2e9, 383), None, phi).scheme == b.SCHEME_TF32X3
    nu = np.linspace(1e9, 2e9, 512)
    w = np.ones(512)
    assert b.Plan(nu, w, phi).scheme == b.SCHEME_F16X3
    w[5] = 0.0
    assert b.Plan(nu, w, phi).scheme == b.SCHEME_F16X3            # zero weights do not count
    w[7] = 1e-7
    assert b.Plan(nu, w, phi).scheme == b.SCHEME_TF32X3


# ------------------------------------------------------------------ peak maps (row a7)
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("lin,lout", [("freq", "phi"), ("los", "los")])
@pytest.mark.parametrize("cfg_id,n_pix", [(4, 300), (5, 517), (1, 200)])
def test_peak_maps(b, oracle_mod, scheme, lin, lout, cfg_id, n_pix):
    cfg, nu, w, phi, q, u = inputs(cfg_id, n_pix)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, lin, lout, peaks=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, "cubes with peaks")
    nd = check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], cfg.dphi, f"{scheme} cfg{cfg_id}")
    assert nd <= max(1, n_pix // 50)
    # maps only (no cubes written)
    out2 = run_gpu(b, plan, q, u, lin, lout, peaks=True, cubes=False)
    for k, v in out["maps"].items():
        assert np.array_equal(v, out2["maps"][k]), k
    plan.destroy()


def test_peak_refinement_on_nonuniform_grid_and_edges(b, oracle_mod):
    nu = np.linspace(1.0e9, 2.0e9, 64)
    phi = np.array([-90.0, -60, -45, -20, -5, 0, 12, 30, 55, 80, 120])
    lam2 = (ri.C_M_PER_S / nu) ** 2
    phi0 = np.array([-90.0, 120.0, 3.0, -50.0, 41.0, 0.0])
    P = np.exp(2j * (0.4 + phi0[:, None] * lam2[None, :]))
    q, u = P.real.astype(np.float32), P.imag.astype(np.float32)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, None, phi, q, u)
    for scheme in SCHEMES:
        plan = b.Plan(nu, None, phi, scheme=scheme_ids(b)[scheme])
        out = run_gpu(b, plan, q, u, "los", "los", peaks=True)
        check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], 5.0, scheme)
        assert out["maps"]["kstar"][0] == 0 and out["maps"]["kstar"][1] == phi.size - 1
        plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("lin,lout", LAYOUTS)
def test_abs_cube_and_maps_only(b, oracle_mod, scheme, lin, lout):
    """rmsynth_execute_ex: the |F| cube (Eq. 17) alone, with the cubes, and maps without any cube.
    Shapes chosen so that depth tiles are ragged (n_phi = 401 -> 4 tiles of 104, second warp half 40 wide)."""
    cfg, nu, w, phi, q, u = inputs(5, 389, start=3)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    Fabs = np.sqrt(FQ ** 2 + FU ** 2)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    n_pix, n_phi = q.shape[0], plan.n_phi
    layout = (b.IN_FREQ_MAJOR if lin == "freq" else 0) | (b.OUT_PHI_MAJOR if lout == "phi" else 0)
    dq = torch.from_numpy(q if lin == "los" else np.ascontiguousarray(q.T)).cuda()
    du = torch.from_numpy(u if lin == "los" else np.ascontiguousarray(u.T)).cuda()
    shape = (n_pix, n_phi) if lout == "los" else (n_phi, n_pix)
    new = lambda: torch.full(shape, float("nan"), device="cuda")
    los = lambda t: t.cpu().numpy() if lout == "los" else t.cpu().numpy().T
    fa = new()
    plan.execute_ex(dq, du, n_pix, layout, F_abs=fa)                       # |F| cube only
    torch.cuda.synchronize()
    assert np.all(np.abs(los(fa) - Fabs) <= 1.5 * TOL * T[:, None]), "F_abs alone"
    fq, fu, fa2 = new(), new(), new()
    maps = {k: torch.full((n_pix,), float("nan"), device="cuda") for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
    maps["peak_index"] = torch.full((n_pix,), -1, dtype=torch.int32, device="cuda")
    plan.execute_ex(dq, du, n_pix, layout, FQ=fq, FU=fu, F_abs=fa2, **maps)
    torch.cuda.synchronize()
    check_cubes(los(fq), los(fu), FQ, FU, T, "execute_ex cubes")
    assert torch.equal(fa, fa2)
    assert torch.equal(fa2, torch.sqrt(torch.addcmul(fu * fu, fq, fq))) or \
        float((fa2 - torch.sqrt(fq * fq + fu * fu)).abs().max()) <= 2e-7 * float(fa2.max())
    got = {("kstar" if k == "peak_index" else k): v.cpu().numpy() for k, v in maps.items()}
    check_peaks(oracle_mod, op, FQ, FU, T, got, cfg.dphi, f"execute_ex {scheme}")
    # the arg-max the fused epilogue takes must be the arg-max of the |F|^2 it could form from its own cube
    y2 = torch.addcmul(fu * fu, fq, fq) if False else (fq * fq + fu * fu)
    km = y2.argmax(1 if lout == "los" else 0).cpu().numpy()
    ymax = y2.amax(1 if lout == "los" else 0).cpu().numpy()
    ysel = (y2 if lout == "los" else y2.T)[torch.arange(n_pix), torch.as_tensor(got["kstar"], device="cuda").long()].cpu().numpy()
    assert np.all(ysel >= ymax * (1 - 3e-7)), "fused arg-max is not the maximum of the written cube"
    maps2 = {k: torch.full_like(v, -1) for k, v in maps.items()}
    plan.execute_ex(dq, du, n_pix, layout, **maps2)                        # maps only: no cube is written
    torch.cuda.synchronize()
    for k in maps:
        assert torch.equal(maps[k], maps2[k]), k
    plan.destroy()


# ------------------------------------------------------------------ host streaming + API edges
@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("lin,lout", [("freq", "phi"), ("los", "los"), ("freq", "los")])
def test_execute_host_matches_oracle(b, oracle_mod, scheme, lin, lout):
    cfg, nu, w, phi, q, u = inputs(1, 2500)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    out = run_gpu(b, plan, q, u, lin, lout, peaks=True, host=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, "execute_host")
    check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], cfg.dphi, "execute_host")
    out2 = run_gpu(b, plan, q, u, lin, lout, peaks=True, cubes=False, host=True)      # maps only: no cube crosses the bus
    for k, v in out["maps"].items():
        assert np.array_equal(v, out2["maps"][k]), k
    plan.destroy()


@pytest.mark.parametrize("scheme", ["f16x3", "tf32x3", "fp32_table"])
@pytest.mark.parametrize("lin,lout", LAYOUTS)
def test_execute_host_multi_chunk(b, oracle_mod, scheme, lin, lout):
    """The three-slot pipeline proper: 7 chunks of 148 lines of sight with a ragged last one (997 = 6 x 148 + 109;
    109 % 4 != 0 -> the repack path), slot re-use after three chunks, column-sliced 2-D copies for the FITS-order and
    phi-major layouts, map offsets -- cubes + maps, then maps only (no cube crosses the bus)."""
    cfg, nu, w, phi, q, u = inputs(4, 997, start=5)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme], host_chunk_pixels=148)
    out = run_gpu(b, plan, q, u, lin, lout, peaks=True, host=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, f"execute_host 7 chunks {scheme} {lin}->{lout}")
    check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], cfg.dphi, "execute_host 7 chunks")
    out2 = run_gpu(b, plan, q, u, lin, lout, peaks=True, cubes=False, host=True)
    check_peaks(oracle_mod, op, FQ, FU, T, out2["maps"], cfg.dphi, "execute_host 7 chunks, maps only")
    plan.destroy()


def test_execute_host_on_a_7000_depth_grid(b, oracle_mod):
    """The paper's LOFAR shape of the depth axis (856 channels -> 7000 depths): 68 depth tiles per pixel tile,
    streamed in 5 chunks through the host path."""
    cfg = ri.CONFIGS[7]
    nu, w, phi = ri.grids(cfg)
    assert phi.size == 7000 and nu.size == 856
    q, u = ri.generate_pixels(cfg, torch.arange(11, 11 + 600))
    q, u = q.numpy(), u.numpy()
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    plan = b.Plan(nu, w, phi, host_chunk_pixels=128)
    out = run_gpu(b, plan, q, u, "freq", "phi", peaks=True, host=True)
    check_cubes(out["FQ"], out["FU"], FQ, FU, T, "execute_host 7000 depths")
    check_peaks(oracle_mod, op, FQ, FU, T, out["maps"], cfg.dphi, "execute_host 7000 depths")
    plan.destroy()


@pytest.mark.parametrize("lin,lout", [("freq", "phi"), ("los", "los")])
@pytest.mark.parametrize("want", ["cubes+maps", "maps"])
def test_execute_stream_callbacks(b, oracle_mod, lin, lout, want):
    """rmsynth_execute_stream: the caller refills pinned staging chunk by chunk (the out-of-core form for cubes that
    do not fit in host memory): 6 chunks of 200 with a ragged last one, every chunk handed back exactly once
    and in order, results equal to the oracle's."""
    cfg, nu, w, phi, q, u = inputs(2, 1090, start=3)
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    n_pix, n_chan, n_phi = q.shape[0], q.shape[1], phi.size
    plan = b.Plan(nu, w, phi, host_chunk_pixels=200)
    layout = (b.IN_FREQ_MAJOR if lin == "freq" else 0) | (b.OUT_PHI_MAJOR if lout == "phi" else 0)
    got_q = np.full((n_pix, n_phi), np.nan, np.float32)
    got_u = np.full_like(got_q, np.nan)
    maps = {k: np.full(n_pix, np.nan, np.float32) for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
    maps["kstar"] = np.full(n_pix, -7, np.int32)
    order, starts = [], {}

    def fill(i, Q, U, max_pix):
        assert max_pix == 200
        p0 = i * 200
        n = max(0, min(200, n_pix - p0))
        if n:
            starts[i] = p0
            blk_q, blk_u = q[p0:p0 + n], u[p0:p0 + n]
            Q[:n * n_chan] = (blk_q.T if lin == "freq" else blk_q).ravel()
            U[:n * n_chan] = (blk_u.T if lin == "freq" else blk_u).ravel()
        return n

    def drain(i, n, out):
        order.append(i)
        p0 = starts[i]
        if want == "cubes+maps":
            shape = (n_phi, n) if lout == "phi" else (n, n_phi)
            fq, fu = out["FQ"].reshape(shape), out["FU"].reshape(shape)
            got_q[p0:p0 + n] = fq.T if lout == "phi" else fq
            got_u[p0:p0 + n] = fu.T if lout == "phi" else fu
        else:
            assert "FQ" not in out
        for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
            maps[k][p0:p0 + n] = out[k]
        maps["kstar"][p0:p0 + n] = out["peak_index"]

    done = plan.execute_stream(layout, (b.WANT_CUBES if want == "cubes+maps" else 0) | b.WANT_MAPS, fill, drain)
    assert done == n_pix and order == list(range(6))
    if want == "cubes+maps":
        check_cubes(got_q, got_u, FQ, FU, T, f"execute_stream {lin}->{lout}")
    check_peaks(oracle_mod, op, FQ, FU, T, maps, cfg.dphi, f"execute_stream {want}")
    plan.destroy()


def test_plan_device_is_honoured_and_current_device_left_alone(b):
    """A plan runs on the device it was created for and the calls leave the caller's current device as they found it."""
    nu, phi = np.linspace(1e9, 2e9, 16), np.linspace(-10, 10, 5)
    before = torch.cuda.current_device()
    plan = b.Plan(nu, None, phi, device=0)
    q = torch.randn(8, 16, device="cuda:0")
    f = torch.zeros(8, 5, device="cuda:0")
    plan.execute(q, q, 8, 0, f, f)
    plan.rmsf(np.array([0.5]))
    torch.cuda.synchronize()
    assert torch.cuda.current_device() == before and torch.isfinite(f).all()
    plan.destroy()


def test_api_edges(b):
    nu, phi = np.linspace(1e9, 2e9, 16), np.linspace(-10, 10, 5)
    for scheme in SCHEMES:
        plan = b.Plan(nu, None, phi, scheme=scheme_ids(b)[scheme])
        q = torch.zeros(4, 16, device="cuda")
        f = torch.zeros(4, 5, device="cuda")
        plan.execute(None, None, 0, 0, None, None)                 # n_pix = 0: successful no-op
        for bad in (lambda: plan.execute(q, q, -1, 0, f, f), lambda: plan.execute(q, q, 4, 4, f, f),
                    lambda: plan.execute(None, q, 4, 0, f, f), lambda: plan.execute(q, q, 4, 0, None, f),
                    lambda: plan.execute_peaks(q, q, 4, 0)):
            with pytest.raises(b.RmsynthError) as e:
                bad()
            assert e.value.status == b.EINVAL
        # runs on a caller-provided stream and does not modify its inputs
        s = torch.cuda.Stream()
        q.normal_()
        q0 = q.clone()
        with torch.cuda.stream(s):
            plan.execute(q, q, 4, 0, f, f, stream=s.cuda_stream)
        s.synchronize()
        assert torch.equal(q, q0) and torch.isfinite(f).all()
        n0 = b.rmsynth_launch_count(True)
        plan.execute(q, q, 4, 0, f, f)
        assert b.rmsynth_launch_count() >= 1 and n0 >= 1
        plan.destroy()


def test_execute_is_capturable_in_a_cuda_graph(b, oracle_mod):
    """rmsynth_execute only enqueues (kernels + one memset) once its per-stream workspace exists, so a launch-bound
    loop over small cubes can be captured in a CUDA graph and replayed."""
    cfg, nu, w, phi, q, u = inputs(1, 640)
    _, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    for scheme in ("tf32x3", "f16x3"):
        plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
        dq, du = torch.from_numpy(q).cuda(), torch.from_numpy(u).cuda()
        fq = torch.zeros(640, plan.n_phi, device="cuda")
        fu = torch.zeros_like(fq)
        idx = torch.zeros(640, dtype=torch.int32, device="cuda")
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            plan.execute_peaks(dq, du, 640, 0, fq, fu, peak_index=idx, stream=s.cuda_stream)   # first use allocates the workspace
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for _ in range(4):
                plan.execute_peaks(dq, du, 640, 0, fq, fu, peak_index=idx, stream=torch.cuda.current_stream().cuda_stream)
        fq.fill_(float("nan"))
        fu.fill_(float("nan"))
        idx.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        check_cubes(fq.cpu().numpy(), fu.cpu().numpy(), FQ, FU, T, f"graph replay {scheme}")
        assert int(idx.min()) >= 0
        # The workspace rule of rmsynth.h: a larger call on the same stream makes the workspace grow, which must not
        # invalidate the captured graph (outgrown buffers live until the plan is destroyed) ...
        big = 4 * 640
        cfg2, _, _, _, q2, u2 = inputs(1, big)
        dq2, du2 = torch.from_numpy(q2).cuda(), torch.from_numpy(u2).cuda()
        fq2 = torch.zeros(big, plan.n_phi, device="cuda")
        fu2 = torch.zeros_like(fq2)
        idx2 = torch.zeros(big, dtype=torch.int32, device="cuda")
        with torch.cuda.stream(s):
            plan.execute_peaks(dq2, du2, big, 0, fq2, fu2, peak_index=idx2, stream=s.cuda_stream)
        s.synchronize()
        fq.fill_(float("nan"))
        fu.fill_(float("nan"))
        idx.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        check_cubes(fq.cpu().numpy(), fu.cpu().numpy(), FQ, FU, T, f"graph replay after workspace growth {scheme}")
        assert int(idx.min()) >= 0
        del g
        # ... and inside a capture the workspace cannot grow: EINVAL, nothing enqueued, the capture stays usable
        bigger = 8 * 640
        cfg3, _, _, _, q3, u3 = inputs(1, bigger)
        dq3, du3 = torch.from_numpy(q3).cuda(), torch.from_numpy(u3).cuda()
        fq3 = torch.zeros(bigger, plan.n_phi, device="cuda")
        fu3 = torch.zeros_like(fq3)
        idx3 = torch.zeros(bigger, dtype=torch.int32, device="cuda")
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=s):
            with pytest.raises(b.RmsynthError) as e:
                plan.execute_peaks(dq3, du3, bigger, 0, fq3, fu3, peak_index=idx3, stream=torch.cuda.current_stream().cuda_stream)
            assert e.value.status == b.EINVAL
            plan.execute_peaks(dq, du, 640, 0, fq, fu, peak_index=idx, stream=torch.cuda.current_stream().cuda_stream)
        g2.replay()
        torch.cuda.synchronize()
        check_cubes(fq.cpu().numpy(), fu.cpu().numpy(), FQ, FU, T, f"graph after a refused call {scheme}")
        del g2
        plan.destroy()


def test_nonfinite_samples_stay_in_their_pixel(b):
    nu, phi = np.linspace(1e9, 2e9, 40), np.linspace(-100, 100, 21)
    for scheme in SCHEMES:
        plan = b.Plan(nu, None, phi, scheme=scheme_ids(b)[scheme])
        q = torch.randn(300, 40, device="cuda")
        u = torch.randn(300, 40, device="cuda")
        q[17, 3] = float("nan")
        u[150, 39] = float("inf")
        fq = torch.zeros(300, 21, device="cuda")
        fu = torch.zeros(300, 21, device="cuda")
        plan.execute(q, u, 300, 0, fq, fu)
        torch.cuda.synchronize()
        bad = ~(torch.isfinite(fq).all(1) & torch.isfinite(fu).all(1))
        assert sorted(torch.nonzero(bad).flatten().tolist()) == [17, 150], scheme
        plan.destroy()


@pytest.mark.parametrize("scheme", SCHEMES)
@pytest.mark.parametrize("lin,lout,n_pix", [("freq", "phi", 520), ("los", "los", 300), ("freq", "phi", 389)])
def test_nonfinite_lines_of_sight_in_the_peak_maps(b, oracle_mod, scheme, lin, lout, n_pix):
    """Reading A17: a line of sight with a non-finite |F| has no peak -- index -1 and NaN in every map, with the cubes
    written and in a maps-only call alike; its neighbours are untouched (520 and 300 pixels take the FP16 kernel's
    fast tile ends, 389 the scalar one)."""
    cfg, nu, w, phi, q, u = inputs(5, n_pix, start=1)
    q, u = q.copy(), u.copy()
    bad = [0, 31, 32, 127, 128, n_pix - 1, n_pix // 2]
    for j, pix in enumerate(bad):
        (q if j % 2 else u)[pix, (37 * j) % cfg.n_chan] = [np.nan, np.inf, -np.inf][j % 3]
    op, FQ, FU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    ref = oracle_mod.peaks(op, FQ, FU)
    assert sorted(np.flatnonzero(ref["kstar"] < 0).tolist()) == sorted(bad)
    plan = b.Plan(nu, w, phi, scheme=scheme_ids(b)[scheme])
    good = np.setdiff1d(np.arange(n_pix), bad)
    for cubes in (True, False):
        out = run_gpu(b, plan, q, u, lin, lout, peaks=True, cubes=cubes)
        m = out["maps"]
        assert np.all(m["kstar"][bad] == -1) and np.all(m["kstar"][good] >= 0), f"{scheme} cubes={cubes}"
        for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero"):
            assert np.all(np.isnan(m[k][bad])) and np.all(np.isfinite(m[k][good])), (scheme, cubes, k)
        check_peaks(oracle_mod, op, FQ, FU, T, m, cfg.dphi, f"{scheme} non-finite maps cubes={cubes}")
        if cubes:
            check_cubes(out["FQ"][good], out["FU"][good], FQ[good], FU[good], T[good], f"{scheme} finite neighbours")
            assert np.all(np.isnan(out["FQ"][bad]) | np.isinf(out["FQ"][bad]))
    plan.destroy()


# ------------------------------------------------------------------ full BASELINE sizes, bench launch configuration
@pytest.mark.parametrize("cfg_id,scheme", [(2, "auto"), (4, "auto"), (3, "auto"), (5, "auto"), (2, "tf32x3"), (5, "tf32x3")])
def test_full_size_cube_sampled_against_oracle(b, oracle_mod, cfg_id, scheme):
    """The cube bench.py times (same layouts, same scheme, one rmsynth_execute_peaks call over the whole
    cube), checked on lines of sight the oracle can compute one by one: every pixel of the first and last
    tile pair, tile-boundary neighbours and 16 384 random lines of sight; plus properties that hold at any
    size."""
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    Q, U = ri.generate_cube(cfg, "cuda")
    layout = (b.IN_FREQ_MAJOR if cfg.layout_in == "freq" else 0) | (b.OUT_PHI_MAJOR if cfg.layout_out == "phi" else 0)
    shape = (cfg.n_phi, cfg.n_pix) if cfg.layout_out == "phi" else (cfg.n_pix, cfg.n_phi)
    FQ = torch.full(shape, float("nan"), device="cuda")
    FU = torch.full(shape, float("nan"), device="cuda")
    maps = {k: torch.full((cfg.n_pix,), float("nan"), device="cuda") for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
    maps["peak_index"] = torch.full((cfg.n_pix,), -1, dtype=torch.int32, device="cuda")
    # default scheme = the product path; 3xTF32 = what AUTO falls back to (few channels, wide weight spans)
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_AUTO if scheme == "auto" else b.SCHEME_TF32X3)
    plan.execute_peaks(Q, U, cfg.n_pix, layout, FQ, FU, **maps)
    torch.cuda.synchronize()
    # properties at full size: every output written and finite, |F| <= T_p (triangle inequality), index in range
    assert bool(torch.isfinite(FQ).all()) and bool(torch.isfinite(FU).all())
    assert int(maps["peak_index"].min()) >= 0 and int(maps["peak_index"].max()) < cfg.n_phi
    kw = torch.as_tensor(plan.K * w, dtype=torch.float32, device="cuda")
    amp_in = torch.sqrt(Q * Q + U * U)
    T_all = (amp_in * (kw[:, None] if cfg.layout_in == "freq" else kw[None, :])).sum(0 if cfg.layout_in == "freq" else 1)
    Fmax = torch.sqrt(FQ * FQ + FU * FU).amax(0 if cfg.layout_out == "phi" else 1)
    assert bool((Fmax <= T_all * (1 + 1e-4) + 1e-30).all())
    del amp_in
    # sampled lines of sight against the oracle
    rng = np.random.default_rng(cfg_id)
    n = cfg.n_pix
    # 16 384 random lines of sight plus every pixel of the first and last tile pair (256 pixels: the FP16
    # kernel's CTA pair owns 256) and both sides of 256 tile boundaries spread over the cube
    edges = np.arange(128, n, 128)[:: max((n // 128) // 256, 1)][:256]
    pix = np.unique(np.concatenate([np.arange(0, min(256, n)), np.arange(max(n - 256, 0), n), edges - 1, edges,
                                    rng.choice(n, min(16384, n), replace=False)]))
    q, u = ri.gather_los(Q, U, cfg.layout_in, pix)
    op, oFQ, oFU, T = oracle_reference(oracle_mod, nu, w, phi, q, u)
    idx = torch.as_tensor(pix, device="cuda")
    gq = (FQ.index_select(1, idx).T if cfg.layout_out == "phi" else FQ.index_select(0, idx)).cpu().numpy()
    gu = (FU.index_select(1, idx).T if cfg.layout_out == "phi" else FU.index_select(0, idx)).cpu().numpy()
    worst = check_cubes(gq, gu, oFQ, oFU, T, f"full config {cfg_id}")
    got = {("kstar" if k == "peak_index" else k): v.index_select(0, idx).cpu().numpy() for k, v in maps.items()}
    check_peaks(oracle_mod, op, oFQ, oFU, T, got, cfg.dphi, f"full config {cfg_id}")
    print(f"full config {cfg_id}: {pix.size} sampled lines of sight, max err/T_p = {worst:.2e}")
    plan.destroy()


@pytest.mark.parametrize("cfg_id", [5, 3])
def test_full_size_cube_two_schemes_agree_everywhere(b, cfg_id):
    """A supplement to the sampled oracle comparison above, not a substitute: the FP16X3 and 3xTF32 kernels share no
    operand format, tile shape or work schedule, so a fault confined to one tile of either would show as a
    disagreement somewhere in the cube.  Every sample of the full cube (configs[4], FITS order in / phi-major out, and
    configs[2], LOS-major in and out, the largest by MACs) is compared on the device: |F_a - F_b| <= 2e-5 T_p, twice the
    oracle tolerance each of them meets on the sampled lines of sight."""
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    Q, U = ri.generate_cube(cfg, "cuda")
    layout = (b.IN_FREQ_MAJOR if cfg.layout_in == "freq" else 0) | (b.OUT_PHI_MAJOR if cfg.layout_out == "phi" else 0)
    shape = (cfg.n_phi, cfg.n_pix) if cfg.layout_out == "phi" else (cfg.n_pix, cfg.n_phi)
    out = {}
    for name, scheme in (("f16x3", b.SCHEME_F16X3), ("tf32x3", b.SCHEME_TF32X3)):
        FQ = torch.full(shape, float("nan"), device="cuda")
        FU = torch.full(shape, float("nan"), device="cuda")
        plan = b.Plan(nu, w, phi, scheme=scheme)
        plan.execute(Q, U, cfg.n_pix, layout, FQ, FU)
        torch.cuda.synchronize()
        K = plan.K
        plan.destroy()
        out[name] = (FQ, FU)
    kw = torch.as_tensor(K * w, dtype=torch.float32, device="cuda")
    amp_in = torch.sqrt(Q * Q + U * U)
    T_all = (amp_in * (kw[:, None] if cfg.layout_in == "freq" else kw[None, :])).sum(0 if cfg.layout_in == "freq" else 1)
    del amp_in, Q, U
    T_all = torch.where(T_all > 0, T_all, torch.ones_like(T_all))
    worst = 0.0
    (aq, au), (bq, bu) = out["f16x3"], out["tf32x3"]
    step = 64 if cfg.layout_out == "phi" else 1 << 18      # depth planes / lines of sight per slice: bounded temporaries
    for s0 in range(0, shape[0], step):
        d = torch.hypot(aq[s0:s0 + step] - bq[s0:s0 + step], au[s0:s0 + step] - bu[s0:s0 + step])
        d = d / (T_all[None, :] if cfg.layout_out == "phi" else T_all[s0:s0 + step, None])
        assert bool(torch.isfinite(d).all()), f"config {cfg_id}: non-finite sample in slice {s0}"
        worst = max(worst, float(d.max()))
    print(f"full config {cfg_id}: FP16X3 vs 3xTF32 over all {shape[0] * shape[1]} samples, max |dF|/T_p = {worst:.2e}")
    assert worst <= 2 * TOL
