"""CPU ORACLE of the masked photometric loss L_c^M (Eq. 2).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this.  Plain numpy, fp64, the
definitions written out; it shares nothing with the CUDA library.

What the paper fixes:  L_c^M = L_c(I * M, R * M)  (Eq. 2), where "L_c is defined in Equation 7 in the 3DGS
paper" -- not reproduced in PAPER.md.  Reading S20b: that published loss is

    L_c(x, y) = (1 - lam) * mean|x - y| + lam * (1 - mean SSIM(x, y)),   lam = 0.2,

with SSIM of Wang et al. 2004 evaluated per channel on an 11 x 11 Gaussian window (sigma = 1.5, normalised to sum 1),
zero padding at the image border, C1 = 0.01^2, C2 = 0.03^2 (dynamic range 1), and both means over all 3 h w values:

    mu_x = G * x,  s_xx = G * x^2 - mu_x^2,  s_xy = G * (x y) - mu_x mu_y                       (* = windowed sum)
    SSIM = (2 mu_x mu_y + C1)(2 s_xy + C2) / ((mu_x^2 + mu_y^2 + C1)(s_xx + s_yy + C2)).

The window sum is written as the plain 121-tap double loop over shifted copies of the zero-padded image; nothing is
separated, blocked or fused.  The gradient is the chain rule through those definitions (the adjoint of a windowed sum
with a symmetric window is the same windowed sum).  Pins: tests/test_oracle_photometric.py (library correlation,
closed forms for constant / identical images, symmetry, central finite differences).
"""
from __future__ import annotations

import numpy as np

WINDOW = 11
SIGMA = 1.5
C1 = 0.01 ** 2
C2 = 0.03 ** 2
LAMBDA_DSSIM = 0.2


def gaussian_window() -> np.ndarray:
    """11 x 11 window: g[i] = exp(-(i - 5)^2 / (2 sigma^2)) normalised to sum 1, G = g g^T."""
    r = np.arange(WINDOW, dtype=np.float64) - WINDOW // 2
    g = np.exp(-(r * r) / (2.0 * SIGMA * SIGMA))
    g /= g.sum()
    return np.outer(g, g)


def window_sum(a: np.ndarray) -> np.ndarray:
    """(G * a)(p) = sum_d G[d] a(p + d) over the 11 x 11 offsets d, a = 0 outside the image.  a: [..., H, W]."""
    G = gaussian_window()
    h = WINDOW // 2
    H, W = a.shape[-2:]
    pad = np.zeros(a.shape[:-2] + (H + 2 * h, W + 2 * h), np.float64)
    pad[..., h:h + H, h:h + W] = a
    out = np.zeros(a.shape, np.float64)
    for dy in range(WINDOW):
        for dx in range(WINDOW):
            out += G[dy, dx] * pad[..., dy:dy + H, dx:dx + W]
    return out


def ssim_terms(x: np.ndarray, y: np.ndarray):
    mu_x, mu_y = window_sum(x), window_sum(y)
    s_xx = window_sum(x * x) - mu_x * mu_x
    s_yy = window_sum(y * y) - mu_y * mu_y
    s_xy = window_sum(x * y) - mu_x * mu_y
    A1, A2 = 2.0 * mu_x * mu_y + C1, 2.0 * s_xy + C2
    B1, B2 = mu_x * mu_x + mu_y * mu_y + C1, s_xx + s_yy + C2
    return mu_x, mu_y, A1, A2, B1, B2


def ssim_map(x: np.ndarray, y: np.ndarray) -> np.ndarray:
    _, _, A1, A2, B1, B2 = ssim_terms(x, y)
    return (A1 * A2) / (B1 * B2)


def photometric_loss(render: np.ndarray, target: np.ndarray, mask, lam: float = LAMBDA_DSSIM, want_grad: bool = True):
    """Eq. 2: L_c(I M, R M).  render, target: [3, H, W]; mask: [H, W] (non-zero = object) or None.
    Returns dict(loss, l1, dssim, ssim_map, grad) with grad = dL/d render ([3, H, W], fp64)."""
    R = np.asarray(render, np.float64)
    I = np.asarray(target, np.float64)
    m = np.ones(R.shape[-2:], np.float64) if mask is None else (np.asarray(mask) != 0).astype(np.float64)
    x, y = R * m, I * m
    n = float(x.size)
    l1 = np.abs(x - y).sum() / n
    mu_x, mu_y, A1, A2, B1, B2 = ssim_terms(x, y)
    S = (A1 * A2) / (B1 * B2)
    dssim = 1.0 - S.sum() / n
    out = dict(loss=(1.0 - lam) * l1 + lam * dssim, l1=l1, dssim=dssim, ssim_map=S)
    if want_grad:
        # dL/dS_p = -lam / n;  S depends on x through mu_x, G*x^2 and G*(x y):
        #   dS/dmu_x  = 2 mu_y (A2 - A1)/(B1 B2) - 2 mu_x S (1/B1 - 1/B2)      (s_xx, s_xy carry -mu_x^2, -mu_x mu_y)
        #   dS/d(G*x^2) = -S / B2,   dS/d(G*xy) = 2 A1 / (B1 B2)
        gS = -lam / n
        d_mu = gS * (2.0 * mu_y * (A2 - A1) / (B1 * B2) - 2.0 * mu_x * S * (1.0 / B1 - 1.0 / B2))
        d_xx = gS * (-S / B2)
        d_xy = gS * (2.0 * A1 / (B1 * B2))
        gx = window_sum(d_mu) + 2.0 * x * window_sum(d_xx) + y * window_sum(d_xy)
        gx += (1.0 - lam) * np.sign(x - y) / n
        out["grad"] = gx * m  # x = R M
    return out
