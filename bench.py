#!/usr/bin/env python
"""Benchmark of the RM-synthesis hot path (arxiv 1810.06250) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--scheme auto] [--impl ours|reference]

A "step" is one pass of the whole hot path (staging, contraction, output store, fused peak maps) over one
synthetic cube.  The default workload is BASELINE.json configs[4], the cube the north_star states its target on
("largest cube": 2048x2048 px, 400 ch -> 401 phi, FITS order in, phi-major out, full FQ/FU output plus peak
maps); configs[1] and configs[2] (largest by MACs) are timed beside it as `secondary`.  `value` is device-resident
throughput (CUDA events on the launching stream, max over ranks); mean, median and best step are reported.
`e2e` is the same metric through rmsynth_execute_host with pinned HOST buffers (H2D + D2H inside the timed
region), next to the pinned-memcpy PCIe rates measured in the same run.  Multi-GPU: every rank processes its own
cube (independent lines of sight; no collective on the data path) -> weak scaling.
--impl reference times the FP64 oracle on host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "complex_GMAC_per_s"            # LOS x chan x phi complex multiply-accumulates per second / 1e9
TENSOR_FLOP_PER_CMAC = 24.0              # 4 real products x 3 split passes x 2
FP32_FLOP_PER_CMAC = 8.0
NCU_FILE = os.path.join(ROOT, "profiles", "r03_ncu_summary.json")


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback"


TENSOR_PATH_FILES = ("tc_gemm.cu", "tc_gemm2.cu", "tc_gemm3.cu", "tc_common.cuh", "tc_epilogue.cuh", "peak_refine.cuh", "peaks.cu",
                     "common.cuh", "execute.cu", "plan.cu")


def tensor_path_hash() -> str:
    """SHA-256 (16 hex digits) of the sources the execute path is compiled from (the tensor kernels, their epilogue, the
    peak kernels, dispatch and plan) -- what an ncu capture of that path depends on.  Edits to rmclean.cu or fft_variant.cu
    do not change it."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1810_06250_b200", "csrc")
    for name in TENSOR_PATH_FILES:
        h.update(name.encode())
        with open(os.path.join(csrc, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_evidence(config: int, scheme: str):
    """dram bytes / tensor-pipe activity of the dominant kernel from the committed ncu capture -- only if that capture
    was taken with the tensor-path sources this run uses (content hash); else None: stale evidence is no evidence."""
    try:
        with open(NCU_FILE) as f:
            d = json.load(f)
    except OSError:
        return None
    e = d.get("captures", {}).get(f"{config}:{scheme}")
    if not e or e.get("tensor_path_hash") != tensor_path_hash():
        return None
    return e


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: [self.lines.append((time.time(), l)) for l in self.proc.stdout], daemon=True).start()
        except OSError:
            self.proc = None

    def stop(self, t_begin=0.0, t_end=float("inf")):
        """Summary over the samples that arrived inside [t_begin, t_end] (the timed region)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        sm, mx, pw, reasons = [], [], [], set()
        inside = [l for t, l in self.lines if t_begin <= t <= t_end + 0.02]
        if not inside and self.lines:      # region shorter than the sampling period: nearest sample
            inside = [min(self.lines, key=lambda tl: abs(tl[0] - 0.5 * (t_begin + t_end)))[1]]
        for l in inside:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(cfg, nu, w, phi, q_los, u_los, n_threads=0, target_s=10.0):
    """FP64 oracle as it stands on a bounded sample of the workload's pixels; n_threads = 0 -> all host cores."""
    import oracle
    op = oracle.make_plan(nu, w, phi)
    n0 = min(256 if n_threads == 1 else 2048, q_los.shape[0])
    t0 = time.perf_counter()
    oracle.synth_table(op, q_los[:n0], u_los[:n0], n_threads=n_threads)
    dt = max(time.perf_counter() - t0, 1e-4)
    n = int(min(q_los.shape[0], max(n0, target_s * n0 / dt)))
    t0 = time.perf_counter()
    _, _, threads = oracle.synth_table(op, q_los[:n], u_los[:n], n_threads=n_threads, return_threads=True)
    dt = time.perf_counter() - t0
    return n * cfg.n_chan * cfg.n_phi / dt / 1e9, threads, n, dt


def workload_dict(cid, cfg):
    return {"workload": f"configs[{cid - 1}] {cfg.name}: {cfg.nx}x{cfg.ny} px, {cfg.n_chan} ch -> {cfg.n_phi} phi, "
                        f"{cfg.layout_in}-major in, {cfg.layout_out}-major out, fp32",
            "n_pix": cfg.n_pix, "n_chan": cfg.n_chan, "n_phi": cfg.n_phi}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=60)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config, 1-based (default 5 = configs[4], the target cube)")
    ap.add_argument("--scheme", default="auto", choices=["auto", "f16x3", "tf32x3", "fp32_table", "fp32_sincos"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-peaks", action="store_true", help="cubes only (default: cubes + fused peak maps, as BASELINE.json configs[4] says)")
    ap.add_argument("--no-alt", action="store_true", help="skip the side measurement of the 3xTF32 scheme")
    ap.add_argument("--no-secondary", action="store_true", help="skip configs[1] and configs[2]")
    ap.add_argument("--no-isolated", action="store_true", help="skip the launches timed alone (after an idle gap)")
    ap.add_argument("--extras", action="store_true",
                    help="also time the NEXT rows on this cube: the FFT variant (rmsynth_execute_fft) and RM-CLEAN (rmsynth_rmclean)")
    a = ap.parse_args()

    import torch
    import rmsynth_inputs as ri

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = ri.CONFIGS[a.config]
    nu, w, phi = ri.grids(cfg)
    workload = workload_dict(a.config, cfg)

    if a.impl == "reference":
        # The oracle timed on host cores; rank 0 alone runs it (others exit 0 without work).
        if rank != 0:
            return
        import oracle
        oracle.build()
        op = oracle.make_plan(nu, w, phi)
        per_pix = cfg.n_chan * cfg.n_phi
        n = int(max(16, min(4096, 2.0e9 / per_pix)))           # ~2 G complex MAC per step
        q, u = ri.generate_pixels(cfg, torch.arange(n))
        q, u = q.numpy(), u.numpy()
        threads = 0
        for _ in range(max(a.warmup, 1)):
            oracle.synth_table(op, q, u)
        t0 = time.perf_counter()
        for _ in range(a.steps):
            _, _, threads = oracle.synth_table(op, q, u, return_threads=True)
        dt = (time.perf_counter() - t0) / a.steps
        val = n * per_pix / dt / 1e9
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": "GCMAC/s", "n_gpus": a.gpus,
                          "steps": a.steps, "warmup": a.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": dict(workload, sample=f"{n} of {cfg.n_pix} lines of sight per step"),
                          "cpu_baseline": {"value": val, "unit": "GCMAC/s", "cores": threads, "kind": "oracle",
                                           "sample": f"{n} lines of sight per step, FP64 oracle_table, OpenMP"},
                          "e2e": {"value": val, "unit": "GCMAC/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}))
        return

    from paper_1810_06250_b200 import binding as b    # raises if the CUDA library is missing: no fallback
    from paper_1810_06250_b200 import build as libbuild

    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback exists)"
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    scheme_id = {"auto": b.SCHEME_AUTO, "f16x3": b.SCHEME_F16X3, "tf32x3": b.SCHEME_TF32X3, "fp32_table": b.SCHEME_FP32_TABLE,
                 "fp32_sincos": b.SCHEME_FP32_SINCOS}
    scheme_name = {v: k for k, v in scheme_id.items()}
    peaks_on = not a.no_peaks
    stream = torch.cuda.current_stream().cuda_stream

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()          # started early: nvidia-smi needs ~1 s before its first sample
    import dataclasses
    from paper_1810_06250_b200 import sharding

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    def layout_of(c):
        return (b.IN_FREQ_MAJOR if c.layout_in == "freq" else 0) | (b.OUT_PHI_MAJOR if c.layout_out == "phi" else 0)

    def alloc(c):
        # each rank owns an independent cube (weak scaling): same grids, different pixel seeds via the rank offset
        rcfg = dataclasses.replace(c, seed=sharding.rank_seed(c.seed, rank))
        Q, U = ri.generate_cube(rcfg, "cuda")
        shape = (c.n_phi, c.n_pix) if c.layout_out == "phi" else (c.n_pix, c.n_phi)
        FQ, FU = torch.empty(shape, device="cuda"), torch.empty(shape, device="cuda")
        maps = {}
        if peaks_on:
            maps = {k: torch.empty(c.n_pix, device="cuda") for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
            maps["peak_index"] = torch.empty(c.n_pix, dtype=torch.int32, device="cuda")
        return Q, U, FQ, FU, maps

    def timed(plan, c, Q, U, FQ, FU, maps, steps, warmup):
        """(per-step ms list, region ms [max over ranks], launches, wall begin, wall end) of `steps` back-to-back calls."""
        lay = layout_of(c)

        def step():
            if maps:
                plan.execute_peaks(Q, U, c.n_pix, lay, FQ, FU, stream=stream, **maps)
            else:
                plan.execute(Q, U, c.n_pix, lay, FQ, FU, stream=stream)

        for _ in range(max(warmup, 3)):
            step()
        barrier()
        b.rmsynth_launch_count(True)
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        barrier()
        t_begin = time.time()
        evs[0].record()
        for i in range(steps):
            step()
            evs[i + 1].record()
        barrier()
        t_end = time.time()
        launches = b.rmsynth_launch_count()
        total_ms = sharding.max_over_ranks(evs[0].elapsed_time(evs[-1]), "cuda")
        per_step = [evs[i].elapsed_time(evs[i + 1]) for i in range(steps)]
        return per_step, total_ms, launches, t_begin, t_end

    # ------------------------------------------------------------------ the headline workload
    Q, U, FQ, FU, maps = alloc(cfg)
    t_plan = time.perf_counter()
    plan = b.Plan(nu, w, phi, scheme=scheme_id[a.scheme])
    torch.cuda.synchronize()
    plan_create_ms = (time.perf_counter() - t_plan) * 1e3     # lambda^2, K, lambda_0^2, phase matrix, operand blobs, R(phi): once per grid
    scheme = plan.scheme                      # what "auto" resolved to
    a.scheme = scheme_name[scheme]
    per_step, total_ms, launches, t_begin, t_end = timed(plan, cfg, Q, U, FQ, FU, maps, a.steps, a.warmup)
    clocks = sampler.stop(t_begin, t_end) if rank == 0 else None
    ms_step = total_ms / a.steps
    value = sharding.whole_job_rate(cfg.cmac, ms_step * 1e-3, world) / 1e9

    # ---- the same step timed ALONE: one launch after an idle gap, so that the power governor starts from an idle chip the
    # way it does for the cuBLAS "burst" figure of MEASURED_PEAKS.json (best of ten 0.7 ms matmuls).  The headline above is K
    # back-to-back steps, i.e. a seconds-long loop under the 1 kW cap, which is what the "sustained" figure measures.
    isolated = None
    if not a.no_isolated:
        ts = []
        for _ in range(5):
            barrier()
            time.sleep(0.4)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if maps:
                plan.execute_peaks(Q, U, cfg.n_pix, layout_of(cfg), FQ, FU, stream=stream, **maps)
            else:
                plan.execute(Q, U, cfg.n_pix, layout_of(cfg), FQ, FU, stream=stream)
            e1.record()
            torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        isolated = {"ms_median": float(np.median(ts)), "ms_best": float(min(ts)), "launches": len(ts),
                    "note": "one step per launch, 0.4 s idle before each"}

    # ---- NEXT rows on the same cube (context lines; --extras)
    extras = None
    if a.extras:
        extras = {}
        def time_call(fn, k):
            for _ in range(2):
                fn()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(k):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / k
        lay = layout_of(cfg)
        k_x = max(2, min(a.steps, 5))
        try:
            ms_fft = time_call(lambda: plan.execute_fft(Q, U, cfg.n_pix, lay, FQ, FU, stream=stream), k_x)
            extras["fft_variant"] = {"ms_per_step": ms_fft, "value": cfg.cmac / (ms_fft * 1e-3) / 1e9, "unit": "GCMAC/s (equivalent: the exact sum's MAC count / time)",
                                     "params": "window 6, oversampling 2 (error <= ~2e-6 T_p)", "outputs": "FQ + FU cubes"}
        except Exception as exc:       # noqa: BLE001  (non-uniform grids are EUNSUPPORTED)
            extras["fft_variant"] = {"unavailable": str(exc)}
        plan.execute(Q, U, cfg.n_pix, lay, FQ, FU, stream=stream)       # dirty cubes for RM-CLEAN
        torch.cuda.synchronize()
        n_clean = min(cfg.n_pix, 262144)
        try:
            shape = (cfg.n_phi, n_clean) if cfg.layout_out == "phi" else (n_clean, cfg.n_phi)
            dq = FQ[:, :n_clean].contiguous() if cfg.layout_out == "phi" else FQ[:n_clean].contiguous()
            du = FU[:, :n_clean].contiguous() if cfg.layout_out == "phi" else FU[:n_clean].contiguous()
            outs = [torch.empty(shape, device="cuda") for _ in range(6)]
            nit = torch.empty(n_clean, dtype=torch.int32, device="cuda")
            cutoff = 3.0 * cfg.sigma / np.sqrt(cfg.n_chan)
            ms_cl = time_call(lambda: plan.rmclean(dq, du, n_clean, lay, 0.1, cutoff, 200, outs[0], outs[1], outs[2], outs[3],
                                                   outs[4], outs[5], n_iter=nit, stream=stream), k_x)
            extras["rmclean"] = {"ms_per_step": ms_cl, "n_pix": n_clean, "mpix_per_s": n_clean / (ms_cl * 1e-3) / 1e6,
                                 "mean_iterations": float(nit.float().mean()), "params": f"gain 0.1, cutoff 3 sigma_F = {cutoff:.3g}, max_iter 200, restored cubes written"}
            del outs, dq, du, nit
        except Exception as exc:       # noqa: BLE001
            extras["rmclean"] = {"unavailable": str(exc)}
        timed(plan, cfg, Q, U, FQ, FU, maps, 1, 0)

    # ---- side measurement: the same cube through the 3xTF32 scheme (the robust fallback of AUTO), for context
    alt = None
    tf32_peak = None
    if scheme == b.SCHEME_F16X3 and not a.no_alt:
        plan_t = b.Plan(nu, w, phi, scheme=b.SCHEME_TF32X3)
        k_alt = max(3, min(a.steps, 10))
        ps, tot, _, _, _ = timed(plan_t, cfg, Q, U, FQ, FU, maps, k_alt, 3)
        ms_alt = tot / k_alt
        alt = {"scheme": "tf32x3", "steps": k_alt, "ms_per_step": ms_alt, "ms_median": float(np.median(ps)), "ms_best": float(min(ps)),
               "value": world * cfg.cmac / (ms_alt * 1e-3) / 1e9, "unit": "GCMAC/s"}
        plan_t.destroy()
        # TF32 denominator measured the way MEASURED_PEAKS.json measures bf16: torch.matmul (cuBLAS) 8192^3, best of 10
        try:
            old = torch.backends.cuda.matmul.allow_tf32
            torch.backends.cuda.matmul.allow_tf32 = True
            x = torch.randn(8192, 8192, device="cuda"); y = torch.randn(8192, 8192, device="cuda")
            for _ in range(3):
                x @ y
            best = 1e9
            for _ in range(10):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); x @ y; e1.record(); torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            tf32_peak = 2 * 8192 ** 3 / (best * 1e-3) / 1e12
            torch.backends.cuda.matmul.allow_tf32 = old
            del x, y
        except Exception:       # noqa: BLE001  (a side measurement must not take the benchmark down)
            tf32_peak = None
        timed(plan, cfg, Q, U, FQ, FU, maps, 1, 0)      # leave FQ/FU holding the default scheme's output for the e2e comparison
        barrier()

    # ---- end-to-end through the host-buffer API (pinned memory, H2D + D2H inside the timed region)
    e2e = None
    if not a.no_e2e:
        lay = layout_of(cfg)
        hQ, hU = Q.cpu().pin_memory(), U.cpu().pin_memory()
        hFQ = torch.empty(FQ.shape, pin_memory=True)
        hFU = torch.empty(FU.shape, pin_memory=True)
        hmaps = {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True) for k, v in maps.items()}
        # PCIe rates of this box, pinned memory, one direction at a time and both at once (for the denominator)
        s2 = torch.cuda.Stream()
        n_copy = min(hQ.numel(), 1 << 28)
        src, dst = hQ.view(-1)[:n_copy], Q.view(-1)[:n_copy]
        back = hFQ.view(-1)[:min(hFQ.numel(), n_copy)]
        def rate(fn, nbytes):
            fn(); torch.cuda.synchronize()
            t0 = time.perf_counter(); fn(); torch.cuda.synchronize()
            return nbytes / (time.perf_counter() - t0) / 1e9
        saved = Q.view(-1)[:n_copy].clone()
        h2d = rate(lambda: dst.copy_(src, non_blocking=True), n_copy * 4)
        d2h = rate(lambda: back.copy_(FQ.view(-1)[:back.numel()], non_blocking=True), back.numel() * 4)
        def both():
            dst.copy_(src, non_blocking=True)
            with torch.cuda.stream(s2):
                back.copy_(FQ.view(-1)[:back.numel()], non_blocking=True)
        duplex = rate(both, (n_copy + back.numel()) * 4)
        Q.view(-1)[:n_copy].copy_(saved)
        del saved
        plan.execute_host(hQ, hU, cfg.n_pix, lay, hFQ, hFU, **hmaps)               # warm-up (allocates chunk buffers)
        barrier()
        k_e2e = max(2, min(a.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            plan.execute_host(hQ, hU, cfg.n_pix, lay, hFQ, hFU, **hmaps)
        torch.cuda.synchronize()
        dt = sharding.max_over_ranks((time.perf_counter() - t0) / k_e2e, "cuda")
        ok = True
        if scheme != b.SCHEME_FP32_SINCOS:
            ok = bool(torch.equal(hFQ.cuda(), FQ)) and bool(torch.equal(hFU.cuda(), FU))
            if maps:
                ok = ok and bool(torch.equal(hmaps["peak_index"].cuda(), maps["peak_index"]))
        h2d_bytes = 2 * hQ.numel() * 4
        d2h_bytes = 2 * hFQ.numel() * 4 + sum(v.numel() * 4 for v in hmaps.values())
        t_floor = max(h2d_bytes / (h2d * 1e9), d2h_bytes / (d2h * 1e9))
        t_duplex = (h2d_bytes + d2h_bytes) / (duplex * 1e9)      # both directions busy at once share the link's duplex rate
        e2e = {"value": world * cfg.cmac / dt / 1e9, "unit": "GCMAC/s", "h2d_bytes_per_step": h2d_bytes,
               "d2h_bytes_per_step": d2h_bytes, "ms_per_step": dt * 1e3, "steps": k_e2e,
               "matches_device_path": ok, "api": "rmsynth_execute_host (pinned host buffers, 3 slots: H2D / kernels / D2H overlap)",
               "pcie": {"h2d_gbs": h2d, "d2h_gbs": d2h, "duplex_gbs": duplex,
                        "floor_ms": t_floor * 1e3, "frac_of_floor": t_floor / dt,
                        "duplex_floor_ms": t_duplex * 1e3, "frac_of_duplex_floor": t_duplex / dt,
                        "frac_of_tighter_floor": max(t_floor, t_duplex) / dt,
                        "note": "pinned torch copies of 1 GiB measured in this run; floor = max(H2D bytes / H2D rate, D2H bytes / D2H rate); "
                                "duplex_floor = (H2D + D2H bytes) / the rate with both directions running at once (binds when the two directions carry similar bytes); "
                                "the tighter of the two is the bound"}}
        del hQ, hU, hFQ, hFU, hmaps
        if not ok:
            print("bench.py: rmsynth_execute_host disagrees with the device-resident path", file=sys.stderr)
            sys.exit(3)

    # ---- CPU baseline on this rank's own cube sample (before the cube is released)
    cpu = None
    if rank == 0 and not a.no_cpu_baseline:
        import oracle
        oracle.build()
        rng = np.random.default_rng(0)
        pix = np.sort(rng.choice(cfg.n_pix, size=min(cfg.n_pix, 131072), replace=False))
        q_los, u_los = ri.gather_los(Q, U, cfg.layout_in, pix)
        rate_all, threads, n, dt = oracle_rate(cfg, nu, w, phi, q_los, u_los)
        rate_1, _, n1, dt1 = oracle_rate(cfg, nu, w, phi, q_los, u_los, n_threads=1, target_s=6.0)
        cpu = {"value": rate_all, "unit": "GCMAC/s", "cores": threads, "kind": "oracle",
               "sample": f"{n} of {cfg.n_pix} lines of sight of the same cube, FP64 oracle_table, {dt:.1f} s",
               "single_thread": {"value": rate_1, "unit": "GCMAC/s", "cores": 1,
                                 "sample": f"{n1} lines of sight, {dt1:.1f} s; the paper's CPU figures are single-threaded (P:L242)"}}

    # ---- secondary workloads: configs[1] (the round-1 line) and configs[2] (largest by MACs), same call, fewer steps
    secondary = []
    if not a.no_secondary and a.config == 5:
        plan.destroy()
        del Q, U, FQ, FU, maps
        torch.cuda.empty_cache()
        for cid in (2, 3):
            c2 = ri.CONFIGS[cid]
            nu2, w2, phi2 = ri.grids(c2)
            Q2, U2, FQ2, FU2, maps2 = alloc(c2)
            p2 = b.Plan(nu2, w2, phi2, scheme=scheme_id["auto"])
            k2 = max(5, min(a.steps, 20))
            ps, tot, _, _, _ = timed(p2, c2, Q2, U2, FQ2, FU2, maps2, k2, 3)
            ms2 = tot / k2
            f16 = p2.scheme == b.SCHEME_F16X3
            secondary.append(dict(workload_dict(cid, c2), scheme=scheme_name[p2.scheme], peaks=peaks_on, steps=k2, ms_per_step=ms2,
                                  ms_median=float(np.median(ps)), ms_best=float(min(ps)),
                                  value=world * c2.cmac / (ms2 * 1e-3) / 1e9, unit="GCMAC/s",
                                  tensor_tflops=TENSOR_FLOP_PER_CMAC * c2.cmac / (ms2 * 1e-3) / 1e12 if f16 or p2.scheme == b.SCHEME_TF32X3 else None))
            p2.destroy()
            del Q2, U2, FQ2, FU2, maps2
            torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
        return

    peaks, peaks_src = load_peaks()
    kern_ms = float(np.mean(per_step))
    src_hash = libbuild.source_hash()
    ev = ncu_evidence(a.config, a.scheme)
    if scheme in (b.SCHEME_TF32X3, b.SCHEME_F16X3):
        achieved = TENSOR_FLOP_PER_CMAC * cfg.cmac / (kern_ms * 1e-3) / 1e12
        f16 = scheme == b.SCHEME_F16X3
        # FP16 runs at the bf16 rate; TF32: measured in this run when available, else half the bf16 rate (guide's nominal 1.1 / 2.25)
        peak = peaks["bf16_tflops"] if f16 else (tf32_peak or 0.5 * peaks["bf16_tflops"])
        sustained = peaks.get("bf16_tflops_sustained", peak) * (1.0 if f16 else 0.5)
        frac = achieved / peak
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": frac,
                "frac_above_one": frac > 1.0,
                "frac_of_sustained_peak": achieved / sustained, "peak_sustained": sustained,
                "isolated": None if not isolated else dict(isolated, achieved=TENSOR_FLOP_PER_CMAC * cfg.cmac / (isolated["ms_median"] * 1e-3) / 1e12,
                                                           frac_of_burst_peak=TENSOR_FLOP_PER_CMAC * cfg.cmac / (isolated["ms_median"] * 1e-3) / 1e12 / peak),
                "traffic": ev["dram_bytes"] if ev else None,
                "tensor_pipe_pct_of_elapsed_cycles_ncu": ev["tensor_pipe_elapsed_pct"] if ev else None,
                "tensor_pipe_pct_of_sm_active_cycles_ncu": ev["tensor_pipe_active_pct"] if ev else None,
                "peaks_gather_ncu": ev.get("peaks_gather") if ev else None,
                "kernel": "tc3_rmsynth_kernel" if f16 else "tc2_rmsynth_kernel",
                "note": f"executed split-precision tensor FLOP (3 products x 4 real x 2 = 24 per useful complex MAC) / mean CUDA-event "
                        f"step time; peak = {peaks_src} bf16 BURST {peaks['bf16_tflops']:.0f} TF ({'fp16 = bf16 rate' if f16 else 'tf32'}); the "
                        f"timed region is {a.steps} back-to-back {kern_ms:.1f} ms kernels under the 1 kW power cap (see clocks), where the same "
                        f"file's SUSTAINED figure {peaks.get('bf16_tflops_sustained', 0):.0f} TF applies: frac_of_sustained_peak; traffic and "
                        f"the tensor_pipe_* / peaks_gather_ncu fields come from profiles/r03_ncu_summary.json and are null unless that capture was taken "
                        f"with these very tensor-path sources (content hash {tensor_path_hash()}; library {src_hash})"}
    else:
        achieved = FP32_FLOP_PER_CMAC * cfg.cmac / (kern_ms * 1e-3) / 1e12
        peak = 148 * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": None, "kernel": a.scheme, "note": "8 FP32 FLOP per complex MAC; peak = 148 SM x 128 FMA lanes x 2 x max clock"}

    if alt:
        alt_peak = tf32_peak or 0.5 * peaks["bf16_tflops"]
        alt["roofline_frac"] = TENSOR_FLOP_PER_CMAC * cfg.cmac / (alt["ms_per_step"] * 1e-3) / 1e12 / alt_peak
        alt["peak"] = alt_peak
        alt["note"] = (f"3xTF32 kernel (tc2_rmsynth_kernel) on the same cube, of the TF32 peak {alt_peak:.0f} TF "
                       f"({'torch.matmul allow_tf32 8192^3, best of 10, this run' if tf32_peak else '0.5 x bf16 burst'}); "
                       "AUTO prefers the FP16 split because it finishes sooner")

    out = {"metric": METRIC, "value": value, "unit": "GCMAC/s", "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
           "ms_per_step": ms_step, "ms_median": float(np.median(per_step)), "ms_best": float(min(per_step)),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": {b.SCHEME_TF32X3: "tf32x3", b.SCHEME_F16X3: "f16x3"}.get(scheme, "f32"), "data": "synthetic",
           "config": dict(workload, scheme=a.scheme, l2="inputs and outputs larger than L2 (no flush needed)"
                          if 8 * cfg.n_pix * (cfg.n_chan + cfg.n_phi) > 126e6 else "fits in L2", peaks=peaks_on,
                          outputs="FQ + FU cubes" + (" + peak |F| / peak phi / PA maps (fused)" if peaks_on else "")),
           "mpix_per_s": world * cfg.n_pix / (ms_step * 1e-3) / 1e6, "plan_create_ms": plan_create_ms,
           "roofline": roof, "alt_scheme": alt, "secondary": secondary, "extras": extras, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
           "clocks": clocks, "library": b.rmsynth_version(),
           "paper_context": "P100 compute-only 10.6-116 GCMAC/s (Table 1, P:L302-304), other hardware: context only"}
    print(json.dumps(out))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
