"""FP64 CPU oracle of the FFT / gridded-lambda^2 approximate variant (scope row NEXT-4).  TEST INFRASTRUCTURE ONLY.

The paper only says "Further increase in speed can be achieved by using Fast Fourier Transforms (FFT) instead of
Discrete Fourier Transforms (DFT) in equations 15 and 16"; channels are not uniform in lambda^2, so
an FFT needs the samples on a uniform grid first.  The algorithm below is the standard non-uniform FFT of type 1
(non-uniform lambda^2 samples -> uniform depths; Dutt & Rokhlin 1993, Greengard & Lee 2004, Kaiser-Bessel window as in
Beatty et al. 2005), restated for this problem; its choices are readings F1-F6 of DESIGN.md section 2c.  It follows the
algorithm step by step in FP64 (numpy; np.fft.fft serves as the FFT step), shares no code with the CUDA path, and is
pinned in tests/test_oracle_nufft.py against the exact sum (oracle_table) and against closed forms.

  F1  uniform depth grid phi_k = phi_0 + k dphi, k = 0 .. N-1, centre index kc = N // 2.  With x_i = lambda_i^2 -
      lambda_0^2 and c_i = K w_i P_i exp(-2i phi_kc x_i), Eq. 11 is F_k = sum_i c_i exp(-2 pi i (k - kc) t_i),
      t_i = dphi x_i / pi: the wanted outputs are the CENTRED band k - kc in [-N/2, N/2) of the fine grid's spectrum,
      where the window's transform is largest and the aliases smallest.
  F2  fine grid of M = the smallest power of two >= sigma N points (oversampling sigma >= 1.25); channel i sits at the
      (periodic) grid coordinate u_i = M t_i mod M.
  F3  spreading: g[m] = sum_i c_i psi(m - u_i) over the W grid points nearest to u_i (periodic), psi the Kaiser-Bessel
      window psi(z) = I0(beta sqrt(1 - (2z/W)^2)) / I0(beta) for |z| <= W/2, beta = pi sqrt(W^2/s^2 (s - 1/2)^2 - 0.8),
      s = M / N the actual oversampling.
  F4  G = FFT_M(g) (forward, e^{-2 pi i k m / M}).
  F5  deapodisation: F_k = G[(k - kc) mod M] / psihat[k], psihat[k] = int psi(z) cos(2 pi (k - kc) z / M) dz evaluated by
      quadrature of the continuous window (2048-point midpoint rule, FP64): the window's Fourier transform at (k - kc)/M.
  F6  zero-weight channels are skipped (reading A13); samples are FP32 promoted to FP64.
"""
from __future__ import annotations

import numpy as np


def fine_grid_size(n_phi: int, sigma: float) -> int:
    m = 1
    while m < sigma * n_phi:
        m *= 2
    return m


def kb_beta(W: int, s: float) -> float:
    return float(np.pi * np.sqrt(W * W / (s * s) * (s - 0.5) ** 2 - 0.8))


def kb_window(z, W: int, beta: float):
    """Kaiser-Bessel window of full width W at offsets z (grid units); zero outside |z| <= W/2."""
    z = np.asarray(z, dtype=np.float64)
    a = 1.0 - (2.0 * z / W) ** 2
    inside = a >= 0.0
    return np.where(inside, np.i0(beta * np.sqrt(np.where(inside, a, 0.0))) / np.i0(beta), 0.0)


def kb_hat(n_phi: int, M: int, W: int, beta: float):
    """F5: Fourier transform of the continuous window at (k - kc) / M, k = 0 .. n_phi - 1 (midpoint rule, 2048 panels)."""
    nq = 2048
    z = (np.arange(nq) + 0.5) / nq * W - W / 2.0
    wz = kb_window(z, W, beta) * (W / nq)
    k = np.arange(n_phi, dtype=np.float64) - (n_phi // 2)
    return (wz[None, :] * np.cos(2.0 * np.pi * k[:, None] * z[None, :] / M)).sum(axis=1)


def nufft_plan(lam2, w, phi, K, lambda0_sq, sigma=2.0, W=8):
    lam2, w, phi = (np.asarray(a, dtype=np.float64) for a in (lam2, w, phi))
    n = phi.size
    dphi = (phi[-1] - phi[0]) / (n - 1) if n > 1 else 1.0
    if n > 2 and np.max(np.abs(np.diff(phi) - dphi)) > 1e-9 * abs(dphi):
        raise ValueError("the FFT variant needs a uniform depth grid (reading F1)")
    M = fine_grid_size(n, sigma)
    beta = kb_beta(W, M / n)
    x = lam2 - lambda0_sq
    t = dphi * x / np.pi
    u = np.mod(M * t, M)                                   # F2
    kc = n // 2
    return dict(n=n, M=M, W=W, beta=beta, u=u, kc=kc, pre=K * w * np.exp(-2j * phi[kc] * x), w=w, hat=kb_hat(n, M, W, beta))


def nufft_synth(plan, Q, U):
    """Approximate F [n_pix, n_phi] complex128 by F1-F6.  Q, U: float32 [n_pix, n_chan]."""
    Q, U = np.asarray(Q), np.asarray(U)
    if Q.dtype != np.float32 or U.dtype != np.float32:
        raise TypeError("Q/U cubes are FP32 (reading A12)")
    n_pix, n_chan = Q.shape
    M, W = plan["M"], plan["W"]
    g = np.zeros((n_pix, M), dtype=np.complex128)
    for i in range(n_chan):                                # F3, channel by channel
        if plan["w"][i] == 0.0:
            continue                                       # F6
        c = plan["pre"][i] * (Q[:, i].astype(np.float64) + 1j * U[:, i].astype(np.float64))
        m0 = int(np.ceil(plan["u"][i] - W / 2.0))          # first of the W grid points with |m - u| <= W/2
        for j in range(W):
            m = m0 + j
            g[:, m % M] += c * kb_window(m - plan["u"][i], W, plan["beta"])
    G = np.fft.fft(g, axis=1)                              # F4
    idx = np.mod(np.arange(plan["n"]) - plan["kc"], M)
    return G[:, idx] / plan["hat"][None, :]                # F5
