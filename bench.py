#!/usr/bin/env python
"""Benchmark of the RM-synthesis hot path (arxiv 1810.06250) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--scheme tf32x3] [--impl ours|reference]

A "step" is one pass of the whole hot path (staging, contraction, output store) over one synthetic
cube of the chosen BASELINE.json config (default configs[1], LOFAR-HBA-like 512x512x800 -> 801, FITS
order in, phi-major out).  `value` is device-resident throughput (CUDA events, max over ranks);
`e2e` is the same metric through rmsynth_execute_host with pinned HOST buffers (H2D + D2H inside the
timed region).  Multi-GPU: every rank processes its own cube (independent lines of sight, P:L176;
no collective on the data path) -> weak scaling.  --impl reference times the FP64 oracle on host cores.
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
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu --set full captures
# committed under profiles/ (config, scheme) -> bytes; filled in when a capture exists
NCU_TRAFFIC = {(2, "f16x3"): 1.697770e9 + 1.644242e9,      # profiles/r01_ncu_full_tc3_cfg2.txt (algorithmic 3.358e9)
               (5, "f16x3"): 13.427832e9 + 13.411358e9,    # profiles/r01_ncu_full_tc3_cfg5.txt (algorithmic 26.877e9)
               (2, "tf32x3"): 1.942956e9 + 1.650126e9,     # profiles/r01_ncu_full_tc2_cfg2.txt
               (5, "tf32x3"): 13.432003e9 + 13.415196e9}   # profiles/r01_ncu_full_tc2_cfg5.txt


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=lambda: [self.lines.append((time.time(), l)) for l in self.proc.stdout], daemon=True).start()
        except OSError:
            self.proc = None

    def stop(self, t_begin=0.0, t_end=float("inf")):
        """Summary over the samples that arrived inside [t_begin, t_end] (the timed region)."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        inside = [l for t, l in self.lines if t_begin <= t <= t_end + 0.1]
        if not inside and self.lines:      # region shorter than the sampling period: nearest sample
            inside = [min(self.lines, key=lambda tl: abs(tl[0] - 0.5 * (t_begin + t_end)))[1]]
        for l in inside:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_rate(cfg, nu, w, phi, q_los, u_los, target_s=15.0):
    """FP64 oracle as it stands, all host cores, on a bounded sample of the workload's pixels."""
    import oracle
    op = oracle.make_plan(nu, w, phi)
    n0 = min(2048, q_los.shape[0])
    t0 = time.perf_counter()
    oracle.synth_table(op, q_los[:n0], u_los[:n0])
    dt = max(time.perf_counter() - t0, 1e-4)
    n = int(min(q_los.shape[0], max(n0, target_s * n0 / dt)))
    t0 = time.perf_counter()
    _, _, threads = oracle.synth_table(op, q_los[:n], u_los[:n], return_threads=True)
    dt = time.perf_counter() - t0
    return n * cfg.n_chan * cfg.n_phi / dt / 1e9, threads, n, dt


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (default 2 = configs[1])")
    ap.add_argument("--scheme", default="auto", choices=["auto", "f16x3", "tf32x3", "fp32_table", "fp32_sincos"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--peaks", action="store_true", help="also produce the peak maps (rmsynth_execute_peaks)")
    ap.add_argument("--no-alt", action="store_true", help="skip the side measurement of the 3xTF32 scheme")
    a = ap.parse_args()

    import torch
    import rmsynth_inputs as ri

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = ri.CONFIGS[a.config]
    nu, w, phi = ri.grids(cfg)
    workload = {"workload": f"configs[{a.config - 1}] {cfg.name}: {cfg.nx}x{cfg.ny} px, {cfg.n_chan} ch -> {cfg.n_phi} phi, "
                            f"{cfg.layout_in}-major in, {cfg.layout_out}-major out, fp32",
                "n_pix": cfg.n_pix, "n_chan": cfg.n_chan, "n_phi": cfg.n_phi}

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

    assert torch.cuda.is_available(), "bench.py needs a GPU (no CPU fallback exists)"
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    scheme = {"auto": b.SCHEME_AUTO, "f16x3": b.SCHEME_F16X3, "tf32x3": b.SCHEME_TF32X3, "fp32_table": b.SCHEME_FP32_TABLE,
              "fp32_sincos": b.SCHEME_FP32_SINCOS}[a.scheme]
    layout = (b.IN_FREQ_MAJOR if cfg.layout_in == "freq" else 0) | (b.OUT_PHI_MAJOR if cfg.layout_out == "phi" else 0)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()          # started early: nvidia-smi needs ~1 s before its first sample
    # each rank owns an independent cube (weak scaling): same grids, different pixel seeds via the rank offset
    import dataclasses
    from paper_1810_06250_b200 import sharding
    rcfg = dataclasses.replace(cfg, seed=sharding.rank_seed(cfg.seed, rank))
    Q, U = ri.generate_cube(rcfg, "cuda")
    out_shape = (cfg.n_phi, cfg.n_pix) if cfg.layout_out == "phi" else (cfg.n_pix, cfg.n_phi)
    FQ = torch.empty(out_shape, device="cuda")
    FU = torch.empty(out_shape, device="cuda")
    maps = {}
    if a.peaks:
        maps = {k: torch.empty(cfg.n_pix, device="cuda") for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
        maps["peak_index"] = torch.empty(cfg.n_pix, dtype=torch.int32, device="cuda")
    plan = b.Plan(nu, w, phi, scheme=scheme)
    scheme = plan.scheme                      # what "auto" resolved to
    a.scheme = {b.SCHEME_F16X3: "f16x3", b.SCHEME_TF32X3: "tf32x3", b.SCHEME_FP32_TABLE: "fp32_table",
                b.SCHEME_FP32_SINCOS: "fp32_sincos"}[scheme]
    stream = torch.cuda.current_stream().cuda_stream

    def step():
        if a.peaks:
            plan.execute_peaks(Q, U, cfg.n_pix, layout, FQ, FU, stream=stream, **maps)
        else:
            plan.execute(Q, U, cfg.n_pix, layout, FQ, FU, stream=stream)

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(a.warmup, 3)):
        step()
    barrier()
    b.rmsynth_launch_count(True)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(a.steps + 1)]
    barrier()
    t_begin = time.time()
    evs[0].record()
    for i in range(a.steps):
        step()
        evs[i + 1].record()
    barrier()
    t_end = time.time()
    launches = b.rmsynth_launch_count()
    clocks = sampler.stop(t_begin, t_end) if rank == 0 else None
    total_ms = sharding.max_over_ranks(evs[0].elapsed_time(evs[-1]), "cuda")
    per_step = [evs[i].elapsed_time(evs[i + 1]) for i in range(a.steps)]
    ms_step = total_ms / a.steps
    value = sharding.whole_job_rate(cfg.cmac, ms_step * 1e-3, world) / 1e9

    # ---- side measurement: the same cube through the 3xTF32 scheme (the robust fallback of AUTO), for context
    alt = None
    if scheme == b.SCHEME_F16X3 and not a.no_alt:
        plan_t = b.Plan(nu, w, phi, scheme=b.SCHEME_TF32X3)
        k_alt = max(3, min(a.steps, 10))
        for _ in range(3):
            plan_t.execute(Q, U, cfg.n_pix, layout, FQ, FU, stream=stream)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(k_alt):
            plan_t.execute(Q, U, cfg.n_pix, layout, FQ, FU, stream=stream)
        e1.record()
        barrier()
        ms_alt = sharding.max_over_ranks(e0.elapsed_time(e1) / k_alt, "cuda")
        alt = {"scheme": "tf32x3", "steps": k_alt, "ms_per_step": ms_alt, "value": world * cfg.cmac / (ms_alt * 1e-3) / 1e9,
               "unit": "GCMAC/s"}
        plan_t.destroy()
        step()                                   # leave FQ/FU holding the default scheme's output for the e2e comparison
        barrier()

    # ---- end-to-end through the host-buffer API (pinned memory, H2D + D2H inside the timed region)
    e2e = None
    if not a.no_e2e:
        hQ, hU = Q.cpu().pin_memory(), U.cpu().pin_memory()
        hFQ = torch.empty(out_shape, pin_memory=True)
        hFU = torch.empty(out_shape, pin_memory=True)
        plan.execute_host(hQ, hU, cfg.n_pix, layout, hFQ, hFU)               # warm-up (allocates chunk buffers)
        barrier()
        k_e2e = max(2, min(a.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            plan.execute_host(hQ, hU, cfg.n_pix, layout, hFQ, hFU)
        torch.cuda.synchronize()
        dt = sharding.max_over_ranks((time.perf_counter() - t0) / k_e2e, "cuda")
        ok = bool(torch.equal(hFQ.cuda(), FQ)) if scheme != b.SCHEME_FP32_SINCOS else True
        e2e = {"value": world * cfg.cmac / dt / 1e9, "unit": "GCMAC/s", "h2d_bytes_per_step": 2 * hQ.numel() * 4,
               "d2h_bytes_per_step": 2 * hFQ.numel() * 4, "ms_per_step": dt * 1e3, "steps": k_e2e,
               "matches_device_path": ok, "api": "rmsynth_execute_host (pinned host buffers)"}
        del hQ, hU, hFQ, hFU

    if rank != 0:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()
        return

    peaks, peaks_src = load_peaks()
    kern_ms = float(np.mean(per_step))
    if scheme in (b.SCHEME_TF32X3, b.SCHEME_F16X3):
        achieved = TENSOR_FLOP_PER_CMAC * cfg.cmac / (kern_ms * 1e-3) / 1e12
        f16 = scheme == b.SCHEME_F16X3
        # FP16 runs at the bf16 rate; TF32 dense = 1/2 of bf16 (guide's nominal 1.1 / 2.25 PFLOP/s)
        peak = peaks["bf16_tflops"] * (1.0 if f16 else 0.5)
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC.get((a.config, a.scheme)), "kernel": "tc3_rmsynth_kernel" if f16 else "tc2_rmsynth_kernel",
                "note": f"executed split-precision tensor FLOP (3 products x 4 real x 2 = 24 per useful complex MAC) / CUDA-event "
                        f"kernel time; peak = {'1.0' if f16 else '0.5'} x {peaks_src} bf16 burst {peaks['bf16_tflops']:.0f} TF "
                        f"({'fp16 = bf16 rate' if f16 else 'tf32 = half the bf16 rate'}); traffic = dram bytes read+written per launch "
                        f"from the committed ncu --set full capture (profiles/), null if none for this config"}
    else:
        achieved = FP32_FLOP_PER_CMAC * cfg.cmac / (kern_ms * 1e-3) / 1e12
        peak = 148 * 128 * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": None, "kernel": a.scheme, "note": "8 FP32 FLOP per complex MAC; peak = 148 SM x 128 FMA lanes x 2 x max clock"}

    if alt:
        alt_peak = 0.5 * peaks["bf16_tflops"]
        alt["roofline_frac"] = TENSOR_FLOP_PER_CMAC * cfg.cmac / (alt["ms_per_step"] * 1e-3) / 1e12 / alt_peak
        alt["note"] = (f"3xTF32 kernel (tc2_rmsynth_kernel) on the same cube, of the TF32 peak {alt_peak:.0f} TF = 0.5 x bf16; "
                       "AUTO prefers the FP16 split because it finishes sooner, not because its fraction is higher")
    cpu = None
    if not a.no_cpu_baseline:
        import oracle
        oracle.build()
        rng = np.random.default_rng(0)
        pix = np.sort(rng.choice(cfg.n_pix, size=min(cfg.n_pix, 262144), replace=False))
        q_los, u_los = ri.gather_los(Q, U, cfg.layout_in, pix)
        rate, threads, n, dt = oracle_rate(cfg, nu, w, phi, q_los, u_los)
        cpu = {"value": rate, "unit": "GCMAC/s", "cores": threads, "kind": "oracle",
               "sample": f"{n} of {cfg.n_pix} lines of sight of the same cube, FP64 oracle_table, {dt:.1f} s"}

    out = {"metric": METRIC, "value": value, "unit": "GCMAC/s", "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": {b.SCHEME_TF32X3: "tf32x3", b.SCHEME_F16X3: "f16x3"}.get(scheme, "f32"), "data": "synthetic",
           "config": dict(workload, scheme=a.scheme, l2="inputs and outputs larger than L2 (no flush needed)"
                          if 8 * cfg.n_pix * (cfg.n_chan + cfg.n_phi) > 126e6 else "fits in L2", peaks=bool(a.peaks)),
           "mpix_per_s": world * cfg.n_pix / (ms_step * 1e-3) / 1e6,
           "roofline": roof, "alt_scheme": alt, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
           "paper_context": "P100 compute-only 10.6-116 GCMAC/s (Table 1, P:L302-304), other hardware: context only"}
    print(json.dumps(out))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
