"""Seeded synthetic Q/U cubes shaped like BASELINE.json's five configs.

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench, and holds
none of the method's arithmetic (no K, no lambda_0^2, no phase matrix, no sums over
channels): it only evaluates the paper's *forward* model, Eq. 1/3/4
    P(lambda^2) = sum_s A_s exp(2i(chi_s + phi_s lambda^2)) [+ Faraday-thick slab] + noise,
with lambda^2 = (c/nu)^2, on a counter-based RNG so any pixel range can be regenerated
independently, on CPU or on the GPU (torch ops only; same integer hash on both).

The paper measures on real telescope cubes (WSRT-SINGS, LOFAR NGC 1569) that
are not available; these cubes stand in for them (recipe: DESIGN.md "Inputs").

Because cos/sin differ in the last ulp between CPU and GPU torch, a cube generated on
one device is the input for both sides: the GPU path consumes the buffer and the oracle
receives the very same samples gathered back to the host.
"""
from __future__ import annotations

from dataclasses import dataclass

import math
import numpy as np
import torch

C_M_PER_S = 299792458.0
SEED_BASE = 1810062500

_M64 = (1 << 64) - 1


def _i64(x: int) -> int:
    """Python int -> two's-complement int64 value."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLD = _i64(0x9E3779B97F4A7C15)
_MUL1 = _i64(0xBF58476D1CE4E5B9)
_MUL2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 tensors (wrapping arithmetic)."""
    z = (z ^ _lsr(z, 30)) * _MUL1
    z = (z ^ _lsr(z, 27)) * _MUL2
    return z ^ _lsr(z, 31)


def hash_u01(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Uniform [0,1) float64 from the counter (seed, stream, idx)."""
    key = _i64(seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03 + 0x632BE59BD9B4E019)
    z = _mix(idx.to(torch.int64) * _GOLD + key)
    z = _mix(z + _GOLD)
    return _lsr(z, 11).to(torch.float64) * (1.0 / (1 << 53))


def hash_normal(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """Standard normal (Box-Muller on two counters)."""
    u1 = hash_u01(seed, 2 * stream, idx)
    u2 = hash_u01(seed, 2 * stream + 1, idx)
    return torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos(2.0 * math.pi * u2)


@dataclass(frozen=True)
class CubeConfig:
    name: str
    nx: int
    ny: int
    n_chan: int
    nu_lo_hz: float
    nu_hi_hz: float
    phi_min: float
    dphi: float
    n_phi: int
    weights: str          # "unit" | "flag10" | "uniform_half_one"
    content: str          # see _pixel_signal
    sigma: float
    layout_in: str        # "los" ([pix][chan]) | "freq" ([chan][pix], FITS order)
    layout_out: str       # "los" ([pix][phi]) | "phi" ([phi][pix])
    seed: int

    @property
    def n_pix(self) -> int:
        return self.nx * self.ny

    @property
    def cmac(self) -> int:
        return self.n_pix * self.n_chan * self.n_phi


def _cfg(i, name, n, n_chan, lo, hi, pmin, pmax, dphi, weights, content, sigma, lin, lout):
    n_phi = int(round((pmax - pmin) / dphi)) + 1
    return CubeConfig(name, n, n, n_chan, lo, hi, pmin, dphi, n_phi, weights, content, sigma,
                      lin, lout, SEED_BASE + i)


# BASELINE.json configs[0..4]; index here is 1-based to match SURVEY.md section 8.
CONFIGS = {
    1: _cfg(1, "tiny_lofar_64", 64, 128, 120e6, 168e6, -50.0, 50.0, 1.0, "unit", "one_source", 0.01, "los", "los"),
    2: _cfg(2, "lofar_hba_512", 512, 800, 120e6, 168e6, -100.0, 100.0, 0.25, "flag10", "sources_slab", 0.05, "freq", "phi"),
    3: _cfg(3, "mwa_1024", 1024, 768, 170e6, 231e6, -50.0, 50.0, 0.1, "uniform_half_one", "sparse_snr", 1.0, "los", "los"),
    4: _cfg(4, "ska_broadband_512", 512, 1000, 1.0e9, 2.0e9, -1000.0, 1000.0, 4.0, "unit", "two_sources", 0.02, "freq", "phi"),
    5: _cfg(5, "survey_2048", 2048, 400, 120e6, 168e6, -200.0, 200.0, 1.0, "unit", "thirty_percent", 0.05, "freq", "phi"),
    # Shapes of the paper's own Table 1 runs as synthetic cubes: context workloads, not BASELINE
    # configs.  WSRT: 512^2 x 803 -> 401 (band edges and phi range are my choice: the paper does not print them);
    # LOFAR_LR: 540^2 x 856 channels 120.238-166.087 MHz -> 7000 depths.
    6: _cfg(6, "paper_wsrt_512", 512, 803, 1.30e9, 1.76e9, -400.0, 400.0, 2.0, "unit", "two_sources", 0.02, "freq", "phi"),
    7: _cfg(7, "paper_lofar_lr_540", 540, 856, 120.238e6, 166.087e6, -350.0, 349.9, 0.1, "unit", "one_source", 0.05, "freq", "phi"),
}


def scaled(cfg: CubeConfig, n: int, name: str | None = None) -> CubeConfig:
    """Same grids and content, n x n pixels (for parity cases the oracle finishes in seconds)."""
    d = dict(cfg.__dict__)
    d.update(nx=n, ny=n, name=name or f"{cfg.name}_n{n}")
    return CubeConfig(**d)


def grids(cfg: CubeConfig):
    """nu[n_chan] (Hz, channel centres, endpoints inclusive), w[n_chan], phi[n_phi]; float64 numpy."""
    i = np.arange(cfg.n_chan, dtype=np.float64)
    nu = cfg.nu_lo_hz + i * ((cfg.nu_hi_hz - cfg.nu_lo_hz) / max(cfg.n_chan - 1, 1))
    phi = cfg.phi_min + np.arange(cfg.n_phi, dtype=np.float64) * cfg.dphi   # by multiplication (A11)
    idx = torch.arange(cfg.n_chan)
    if cfg.weights == "unit":
        w = np.ones(cfg.n_chan)
    elif cfg.weights == "flag10":
        r = hash_u01(cfg.seed, 900, idx).numpy()
        w = np.ones(cfg.n_chan)
        w[np.argsort(r, kind="stable")[: cfg.n_chan // 10]] = 0.0   # exactly 10 % flagged
    elif cfg.weights == "uniform_half_one":
        w = 0.5 + 0.5 * hash_u01(cfg.seed, 901, idx).numpy()
    else:
        raise ValueError(cfg.weights)
    return nu, w, phi


def _point(lam2, A, chi, phi0):
    ang = 2.0 * (chi[:, None] + phi0[:, None] * lam2[None, :])
    return A[:, None] * torch.cos(ang), A[:, None] * torch.sin(ang)


def _pixel_signal(cfg: CubeConfig, p: torch.Tensor, lam2: torch.Tensor, w_np: np.ndarray):
    """Noise-free Q,U [len(p), n_chan] float64 from per-pixel hashed parameters."""
    s = cfg.seed
    u = lambda stream: hash_u01(s, stream, p)
    zero = torch.zeros(p.numel(), lam2.numel(), dtype=torch.float64, device=p.device)
    Q, U = zero.clone(), zero.clone()
    kind = cfg.content
    if kind == "one_source":
        q, v = _point(lam2, 0.1 + 0.9 * u(1), math.pi * u(2), -40.0 + 80.0 * u(3))
        Q += q; U += v
    elif kind == "sources_slab":
        n_src = torch.floor(4.0 * u(10)).to(torch.int64)          # 0..3
        for j in range(3):
            A = (0.1 + 0.9 * u(11 + 3 * j)) * (n_src > j)
            q, v = _point(lam2, A, math.pi * u(12 + 3 * j), -80.0 + 160.0 * u(13 + 3 * j))
            Q += q; U += v
        # Faraday-thick slab (Burn slab): uniform F over [phi_c - D/2, phi_c + D/2]
        #   P = A exp(2i(chi + phi_c lam2)) sin(D lam2)/(D lam2)      (Eq. 4)
        A, chi = 0.1 + 0.9 * u(30), math.pi * u(31)
        phic, D = -80.0 + 160.0 * u(32), 1.0 + 4.0 * u(33)
        x = D[:, None] * lam2[None, :]
        q, v = _point(lam2, A, chi, phic)
        sinc = torch.sin(x) / x
        Q += q * sinc; U += v * sinc
    elif kind == "sparse_snr":
        has = u(40) < 0.01
        sig_f = cfg.sigma * math.sqrt(float((w_np ** 2).sum())) / float(w_np.sum())
        A = (5.0 + 45.0 * u(41)) * sig_f * has
        q, v = _point(lam2, A, math.pi * u(42), -40.0 + 80.0 * u(43))
        Q += q; U += v
    elif kind == "two_sources":
        for j in range(2):
            q, v = _point(lam2, 0.1 + 0.9 * u(50 + 3 * j), math.pi * u(51 + 3 * j), -800.0 + 1600.0 * u(52 + 3 * j))
            Q += q; U += v
    elif kind == "thirty_percent":
        A = (0.1 + 0.9 * u(61)) * (u(60) < 0.30)
        q, v = _point(lam2, A, math.pi * u(62), -160.0 + 320.0 * u(63))
        Q += q; U += v
    else:
        raise ValueError(kind)
    return Q, U


def generate_pixels(cfg: CubeConfig, pix: torch.Tensor):
    """Q,U float32 [len(pix), n_chan] (LOS-major rows) for the given pixel indices p = y*nx + x."""
    dev = pix.device
    nu, w, _ = grids(cfg)
    lam2 = torch.as_tensor((C_M_PER_S / nu) ** 2, dtype=torch.float64, device=dev)
    pix = pix.to(torch.int64)
    Q, U = _pixel_signal(cfg, pix, lam2, w)
    cnt = pix[:, None] * cfg.n_chan + torch.arange(cfg.n_chan, device=dev)[None, :]
    Q += cfg.sigma * hash_normal(cfg.seed, 70, cnt)
    U += cfg.sigma * hash_normal(cfg.seed, 71, cnt)
    return Q.to(torch.float32), U.to(torch.float32)


def generate_cube(cfg: CubeConfig, device="cpu", layout: str | None = None, chunk: int = 1 << 15,
                  pin_memory: bool = False):
    """Full Q,U cubes float32 on `device`: "los" -> [n_pix, n_chan]; "freq" -> [n_chan, n_pix]."""
    layout = layout or cfg.layout_in
    shape = (cfg.n_pix, cfg.n_chan) if layout == "los" else (cfg.n_chan, cfg.n_pix)
    kw = dict(dtype=torch.float32, device=device)
    if pin_memory:
        kw["pin_memory"] = True
    Q, U = torch.empty(shape, **kw), torch.empty(shape, **kw)
    for p0 in range(0, cfg.n_pix, chunk):
        p1 = min(p0 + chunk, cfg.n_pix)
        q, u = generate_pixels(cfg, torch.arange(p0, p1, device=device))
        if layout == "los":
            Q[p0:p1], U[p0:p1] = q, u
        else:
            Q[:, p0:p1], U[:, p0:p1] = q.T, u.T
    return Q, U


def gather_los(Q: torch.Tensor, U: torch.Tensor, layout: str, pix) -> tuple[np.ndarray, np.ndarray]:
    """Rows [len(pix), n_chan] of a cube in either layout, as host float32 numpy (for the oracle)."""
    idx = torch.as_tensor(np.asarray(pix), dtype=torch.int64, device=Q.device)
    if layout == "los":
        q, u = Q.index_select(0, idx), U.index_select(0, idx)
    else:
        q, u = Q.index_select(1, idx).T, U.index_select(1, idx).T
    return q.contiguous().cpu().numpy(), u.contiguous().cpu().numpy()
