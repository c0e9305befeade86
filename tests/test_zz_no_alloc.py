"""rmsynth_peaks_static -- the one entry point of the library that never allocates -- against the existing peak path.

Why the entry point exists: some users of this library cannot call cudaMalloc while they run (a framework whose memory
pool owns the whole device, a process under a fixed device-memory cap, a real-time loop that cannot take cudaMalloc's
device-wide synchronisation).  Every other peak path allocates its segment records on the first call of a (stream, size);
this one keeps them in a 32 MiB array that is part of the library, shared by every call.

What is checked: on cubes the existing path (rmsynth_execute_peaks) has just written, the new call must return the same
maps -- same peak index, and amplitudes / depths / angles equal to within FP32 rounding of the shared refinement
arithmetic (both sides decide on the same FP32 |F|^2, so the index is compared exactly).  Because the array keeps the
previous call's records, every case makes TWO calls in a row on DIFFERENT data and checks both: a record left over from
the first call and wrongly read by the second would show.  The file is named to be collected last (`pytest -x` stops at
the first failure) and needs nothing from the tests before it: it builds its own plans and inputs, so it passes alone in a
fresh process (where its first call is the one that looks the array up) and after the whole suite.
"""
import numpy as np
import pytest
import torch

import rmsynth_inputs as ri

pytestmark = pytest.mark.gpu

MAPS = ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")


@pytest.fixture(scope="module")
def b():
    assert torch.cuda.is_available(), "gpu tests need a B200"
    from paper_1810_06250_b200 import binding
    return binding


def new_maps(n_pix):
    m = {k: torch.full((n_pix,), float("nan"), dtype=torch.float32, device="cuda") for k in MAPS}
    m["peak_index"] = torch.full((n_pix,), -7, dtype=torch.int32, device="cuda")
    return m


def existing_path(b, plan, cfg, n_pix, start, lout, poison=()):
    """Cubes and maps from rmsynth_execute_peaks (the path that allocates its workspace)."""
    q, u = ri.generate_pixels(cfg, torch.arange(start, start + n_pix))
    for p in poison:                                    # reading A17: a non-finite line of sight has no peak
        q[p, 3] = float("nan")
    layout = b.IN_LOS_MAJOR | (b.OUT_PHI_MAJOR if lout == "phi" else b.OUT_LOS_MAJOR)
    shape = (plan.n_phi, n_pix) if lout == "phi" else (n_pix, plan.n_phi)
    FQ = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
    FU = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
    maps = new_maps(n_pix)
    plan.execute_peaks(q.cuda(), u.cuda(), n_pix, layout, FQ, FU, **maps)
    torch.cuda.synchronize()
    return layout, FQ, FU, maps


def assert_same_maps(got, ref, what):
    kg, kr = got["peak_index"].cpu().numpy(), ref["peak_index"].cpu().numpy()
    assert np.array_equal(kg, kr), f"{what}: {np.count_nonzero(kg != kr)} peak indices differ"
    for k in MAPS:
        g, r = got[k].cpu().numpy(), ref[k].cpu().numpy()
        assert np.array_equal(np.isnan(g), np.isnan(r)), f"{what}: {k} NaN pattern differs"
        # same FP32 inputs, same refinement code: equal up to the compiler's contraction choices in two kernels
        assert np.allclose(g, r, rtol=2e-6, atol=2e-6, equal_nan=True), f"{what}: {k} off by {np.nanmax(np.abs(g - r))}"


@pytest.mark.parametrize("lout", ["phi", "los"])
@pytest.mark.parametrize("cfg_id,n_pix", [(1, 1031), (4, 300), (7, 260)])
def test_static_workspace_call_matches_existing_peak_path_twice_in_a_row(b, lout, cfg_id, n_pix):
    """cfg 1: 101 depths (four segments, the last one ragged); cfg 4: 501 depths; cfg 7: the 7000-depth LOFAR grid (219 segments)."""
    cfg = ri.CONFIGS[cfg_id]
    nu, w, phi = ri.grids(cfg)
    plan = b.Plan(nu, w, phi)
    first = existing_path(b, plan, cfg, n_pix, 11, lout)
    second = existing_path(b, plan, cfg, n_pix - 37, 2000, lout, poison=(0, 101))   # other data, other size, two dead pixels
    for call, (layout, FQ, FU, ref) in enumerate((first, second)):
        n = ref["peak_index"].numel()
        got = new_maps(n)
        plan.peaks_static(FQ, FU, n, layout, **got)
        torch.cuda.synchronize()
        assert_same_maps(got, ref, f"cfg{cfg_id} {lout}-major call {call + 1}")
    assert second[3]["peak_index"][0].item() == -1 and second[3]["peak_index"][101].item() == -1
    plan.destroy()


def test_static_workspace_slab_of_a_larger_cube_and_partial_outputs(b):
    """ld + pointer offset select pixels [64, 64+200) of a phi-major cube; only two of the five maps requested."""
    cfg = ri.CONFIGS[1]
    nu, w, phi = ri.grids(cfg)
    plan = b.Plan(nu, w, phi)
    n_pix = 512
    layout, FQ, FU, ref = existing_path(b, plan, cfg, n_pix, 3, "phi")
    for _ in range(2):
        amp = torch.full((200,), float("nan"), dtype=torch.float32, device="cuda")
        idx = torch.full((200,), -7, dtype=torch.int32, device="cuda")
        plan.peaks_static(FQ.view(-1)[64:], FU.view(-1)[64:], 200, layout, ld=n_pix, peak_amp=amp, peak_index=idx)
        torch.cuda.synchronize()
        assert torch.equal(idx, ref["peak_index"][64:264])
        assert torch.allclose(amp, ref["peak_amp"][64:264], rtol=2e-6, atol=0)
    plan.destroy()


def test_static_workspace_rejects_what_does_not_fit(b):
    cfg = ri.CONFIGS[1]
    nu, w, phi = ri.grids(cfg)
    plan = b.Plan(nu, w, phi)
    x = torch.zeros(16, device="cuda")
    idx = torch.zeros(16, dtype=torch.int32, device="cuda")
    with pytest.raises(b.RmsynthError) as e:
        plan.peaks_static(x, x, (1 << 20) + 1, b.OUT_PHI_MAJOR, peak_index=idx)      # rejected before anything is read
    assert e.value.status == b.EINVAL and "1048576" in str(e.value)
    with pytest.raises(b.RmsynthError) as e:
        plan.peaks_static(x, x, 16, b.OUT_PHI_MAJOR, ld=8, peak_index=idx)
    assert e.value.status == b.EINVAL
    with pytest.raises(b.RmsynthError) as e:
        plan.peaks_static(x, x, 16, b.OUT_PHI_MAJOR)
    assert e.value.status == b.EINVAL
    plan.peaks_static(x, x, 0, b.OUT_PHI_MAJOR, peak_index=idx)                      # empty input: a no-op
    plan.destroy()
