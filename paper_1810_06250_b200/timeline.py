"""Per-role timeline of the FP16 tensor kernel (tc3_rmsynth_kernel) -- debug tool, not on the product path.

    python -m paper_1810_06250_b200.timeline [--config 5] [--no-peaks] [--items 16:112]

Builds librmsynth_timeline.so (the product sources with -DRMSYNTH_TIMELINE), runs one rmsynth_execute_peaks
over a synthetic BASELINE.json cube and tabulates, per sampled CTA and warp role, where the cycles of a
work item (pixel-tile pair x depth tile) go: time blocked on each mbarrier, time in the gang check-in,
time in the tile-end store/scan.  clock64 stamps are per SM, so only differences inside one CTA are formed.
Slots (csrc/tc_gemm3.cu):
  producer   0 check-in begin | 1 check-in end | 2 last load issued | 3 sum(wait raw_empty)
  issuer     0 item begin | 1 sum(wait acc_empty, chunks >= 2) | 2 sum(wait a_ready) | 3 item end
             4 wait acc_empty, first two chunks | 5 wait a_ready, first A slot
  transform  0 item begin | 1 sum(wait raw_full, chunks >= 1) | 2 sum(wait a_empty) | 3 sum(wait b_full) | 4 item end
             5 wait raw_full, first chunk | 6 sum(loads, chunk maximum, split, TMEM store issue) | 7 sum(tcgen05.wait::st)
  epilogue   0 item begin | 1 sum(wait acc_full, chunks >= 1) | 2 last drain done | 3 tile end done
             4 wait acc_full, first chunk
"""
from __future__ import annotations

import argparse
import ctypes as C
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

TL_ITEMS, TL_SLOTS, TL_ROLES, TL_CTAS = 128, 8, 5, 8
ROLES = ["producer", "issuer", "transform", "epilogue w8", "epilogue w12"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--no-peaks", action="store_true")
    ap.add_argument("--items", default="16:112", help="first:last work item of each CTA to average over")
    a = ap.parse_args()

    from paper_1810_06250_b200 import build
    os.environ["RMSYNTH_LIB"] = build.build(timeline=True)
    import torch
    import rmsynth_inputs as ri
    from paper_1810_06250_b200 import binding as b

    cfg = ri.CONFIGS[a.config]
    nu, w, phi = ri.grids(cfg)
    Q, U = ri.generate_cube(cfg, "cuda")
    layout = (b.IN_FREQ_MAJOR if cfg.layout_in == "freq" else 0) | (b.OUT_PHI_MAJOR if cfg.layout_out == "phi" else 0)
    shape = (cfg.n_phi, cfg.n_pix) if cfg.layout_out == "phi" else (cfg.n_pix, cfg.n_phi)
    FQ, FU = torch.empty(shape, device="cuda"), torch.empty(shape, device="cuda")
    maps = {}
    if not a.no_peaks:
        maps = {k: torch.empty(cfg.n_pix, device="cuda") for k in ("peak_amp", "peak_phi", "pa_lambda0", "pa_zero")}
        maps["peak_index"] = torch.empty(cfg.n_pix, dtype=torch.int32, device="cuda")
    plan = b.Plan(nu, w, phi, scheme=b.SCHEME_F16X3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        plan.execute_peaks(Q, U, cfg.n_pix, layout, FQ, FU, **maps)
    torch.cuda.synchronize()
    e0.record()
    plan.execute_peaks(Q, U, cfg.n_pix, layout, FQ, FU, **maps)
    e1.record()
    torch.cuda.synchronize()
    n = TL_CTAS * TL_ROLES * TL_ITEMS * TL_SLOTS
    buf = np.zeros(n, dtype=np.int64)
    lib = C.CDLL(os.environ["RMSYNTH_LIB"])
    lib.rmsynth_timeline_read.argtypes = [C.c_void_p, C.c_int]
    got = lib.rmsynth_timeline_read(buf.ctypes.data, n)
    assert got == n, got
    t = buf.reshape(TL_CTAS, TL_ROLES, TL_ITEMS, TL_SLOTS).astype(np.float64)
    i0, i1 = (int(x) for x in a.items.split(":"))
    print(f"# {cfg.name}: {cfg.n_pix} px, {cfg.n_chan} ch -> {cfg.n_phi} phi, peaks={not a.no_peaks}, "
          f"sync lag {os.environ.get('RMSYNTH_SYNC_LAG', 'default')}; instrumented kernel {e0.elapsed_time(e1):.3f} ms; "
          f"cycles, mean over work items {i0}..{i1 - 1} of each sampled CTA")
    names = ["cluster0.r0", "cluster0.r1", "cluster1.r0", "cluster1.r1", "cluster3.r0", "cluster3.r1", "last.r0", "last.r1"]
    for c in range(TL_CTAS):
        P, I, T, E0, E1 = (t[c, r, i0:i1] for r in range(TL_ROLES))
        if not P[:, 1].any():
            continue
        n_items = int((t[c, TL_PRODUCER_, :, 0] > 0).sum())
        if n_items <= i0 + 2:
            continue
        i1 = min(i1, n_items - 1)
        P, I, T, E0, E1 = (t[c, r, i0:i1] for r in range(TL_ROLES))
        period = np.diff(t[c, TL_PRODUCER_, i0:i1 + 1, 0]).mean()
        print(f"{names[c]:12s} item period {period:8.0f}")
        print(f"  producer   check-in wait {np.mean(P[:, 1] - P[:, 0]):7.0f} | loads {np.mean(P[:, 2] - P[:, 1]):7.0f} "
              f"(of which blocked on raw_empty {P[:, 3].mean():7.0f})")
        if I[:, 3].any():
            print(f"  issuer     item {np.mean(I[:, 3] - I[:, 0]):7.0f} | blocked: acc_empty first two chunks {I[:, 4].mean():7.0f}, later chunks "
                  f"{I[:, 1].mean():7.0f}; a_ready first slot {I[:, 5].mean():7.0f}, later {I[:, 2].mean():7.0f}")
        print(f"  transform  item {np.mean(T[:, 4] - T[:, 0]):7.0f} | blocked: raw_full first chunk {T[:, 5].mean():7.0f}, later {T[:, 1].mean():7.0f}; "
              f"a_empty {T[:, 2].mean():7.0f}; b_full {T[:, 3].mean():7.0f} | work: load+max+split {T[:, 6].mean():7.0f}, wait::st {T[:, 7].mean():7.0f}")
        for name, E in (("epilogue w4", E0), ("epilogue w8", E1)):
            print(f"  {name} item {np.mean(E[:, 3] - E[:, 0]):7.0f} | blocked on acc_full: first chunk {E[:, 4].mean():7.0f}, later {E[:, 1].mean():7.0f} | "
                  f"drains (incl. waits) {np.mean(E[:, 2] - E[:, 0]):7.0f} | tile end (scale, store, scan) {np.mean(E[:, 3] - E[:, 2]):7.0f}")


TL_PRODUCER_ = 0

if __name__ == "__main__":
    main()
