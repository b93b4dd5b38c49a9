"""CPU ORACLE of the two regularisers of Eq. 3.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this.  Plain numpy, fp64; shares
nothing with the CUDA library.

What the paper fixes: L = L_c^M + alpha L_d + beta L_n + gamma L_b (Eq. 3), "L_d and L_n are the
regularization terms for depth distortion and normal consistency" of 2DGS, "unchanged" and unmasked;
their formulas are not in PAPER.md.  Readings (DESIGN.md R-moments, R-Ld, R-Ln), stated on the maps the renderer returns
for one view -- alpha A = sum w_i, depth D = sum w_i z_i, normal Nrm = sum w_i n_i and the depth moments about the
per-pixel origin c = depth of the pixel's first blended pair, m1 = sum w_i (z_i - c), m2 = sum w_i (z_i - c)^2
(w_i = alpha_i T_i, n_i the camera-facing view-space normal):

  R-Ld  depth distortion, squared pairwise form:   L_d = 1/(hw) sum_p sum_{i<j} w_i w_j (z_i - z_j)^2
        which equals                               1/(hw) sum_p (A m2 - m1^2)   for ANY origin c (expand the square; pinned
        below).  Raw moments (c = 0) cancel by (z / spread of z)^2 ~ 1e3 in fp32, which is why the renderer centres them.
  R-Ln  normal consistency:                        L_n = 1/(hw) sum_p sum_i w_i (1 - n_i . Nhat) = 1/(hw) sum_p (A - Nrm . Nhat)
        with Nhat(p) the unit normal of the rendered depth surface at p: zbar = D / A (expected depth; pixels with
        A <= eps_A = 1e-4 have no surface: Nhat = 0 there and at their 4-neighbours), P = zbar * ((x - ox)/fx, (y - oy)/fy, 1)
        the back-projected point (ox = cx - 1/2: pixel-index coordinates, S2), central differences
        a = (P(x+1,y) - P(x-1,y))/2, b = (P(x,y+1) - P(x,y-1))/2, Nhat = -(a x b)/|a x b| (towards the camera, like n_i);
        Nhat = 0 on the one-pixel image border and where |a x b| = 0.

Everything is differentiated (no stop-gradient): the function returns the upstream gradients of the five maps, which
ocgs_render_bwd_reg consumes.
"""
from __future__ import annotations

import numpy as np

EPS_A = 1e-4


def distortion_map(A, m1, m2):
    """Per pixel sum_{i<j} w_i w_j (z_i - z_j)^2 = A m2 - m1^2 (R-Ld), m1, m2 the depth moments about any origin."""
    return np.asarray(A, np.float64) * np.asarray(m2, np.float64) - np.asarray(m1, np.float64) ** 2


def distortion_bruteforce(w, z):
    """The definition for ONE pixel from its blended sequence (weights w_i, depths z_i): explicit double sum over i < j."""
    w, z = np.asarray(w, np.float64), np.asarray(z, np.float64)
    tot = 0.0
    for i in range(len(w)):
        for j in range(i + 1, len(w)):
            tot += w[i] * w[j] * (z[i] - z[j]) ** 2
    return tot


def _rays(H, W, fx, fy, cx, cy):
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    return np.stack([(xs - (cx - 0.5)) / fx, (ys - (cy - 0.5)) / fy, np.ones((H, W))])


def depth_normal(A, D, fx, fy, cx, cy):
    """Nhat [3,H,W] of R-Ln, plus the intermediates the backward needs."""
    A, D = np.asarray(A, np.float64), np.asarray(D, np.float64)
    H, W = A.shape
    surf = A > EPS_A
    zbar = np.where(surf, D / np.where(surf, A, 1.0), 0.0)
    r = _rays(H, W, fx, fy, cx, cy)
    P = zbar[None] * r
    valid = np.zeros((H, W), bool)
    valid[1:-1, 1:-1] = surf[1:-1, 1:-1] & surf[1:-1, :-2] & surf[1:-1, 2:] & surf[:-2, 1:-1] & surf[2:, 1:-1]
    a = np.zeros((3, H, W)); b = np.zeros((3, H, W))
    a[:, 1:-1, 1:-1] = 0.5 * (P[:, 1:-1, 2:] - P[:, 1:-1, :-2])
    b[:, 1:-1, 1:-1] = 0.5 * (P[:, 2:, 1:-1] - P[:, :-2, 1:-1])
    c = np.cross(a, b, axis=0)
    nc = np.sqrt((c * c).sum(0))
    valid &= nc > 0
    Nhat = np.where(valid[None], -c / np.where(valid, nc, 1.0)[None], 0.0)
    return Nhat, dict(surf=surf, zbar=zbar, r=r, a=a, b=b, c=c, nc=nc, valid=valid)


def regularizers(A, D, m1, m2, Nrm, fx, fy, cx, cy, w_d=1.0, w_n=1.0):
    """Returns dict(L_d, L_n, gA, gD, gM1, gM2, gN): the two losses (each a mean over all h w pixels) and the gradients of
    w_d L_d + w_n L_n with respect to the five maps (the moments' origin held fixed: L_d does not depend on it)."""
    A, D, m1, m2, Nrm = (np.asarray(t, np.float64) for t in (A, D, m1, m2, Nrm))
    H, W = A.shape
    hw = float(H * W)
    L_d = distortion_map(A, m1, m2).sum() / hw
    Nhat, t = depth_normal(A, D, fx, fy, cx, cy)
    L_n = (A - (Nrm * Nhat).sum(0)).sum() / hw
    # distortion: d(A m2 - m1^2) = m2 dA - 2 m1 dm1 + A dm2
    gA = w_d * m2 / hw
    gM1 = -2.0 * w_d * m1 / hw
    gM2 = w_d * A / hw
    gD = np.zeros((H, W))
    # normal consistency: l = A - Nrm . Nhat
    gA = gA + w_n / hw
    gN = -w_n * Nhat / hw
    gNhat = np.where(t["valid"][None], -w_n * Nrm / hw, 0.0)
    # Nhat = -c/|c|  =>  g_c = -(g - Nhat (Nhat . g)) / |c|
    dot = (Nhat * gNhat).sum(0)
    gc = np.where(t["valid"][None], -(gNhat - Nhat * dot[None]) / np.where(t["valid"], t["nc"], 1.0)[None], 0.0)
    # c = a x b  =>  g_a = b x g_c, g_b = g_c x a
    ga = np.cross(t["b"], gc, axis=0)
    gb = np.cross(gc, t["a"], axis=0)
    # a(x,y) = (P(x+1,y) - P(x-1,y))/2, b(x,y) = (P(x,y+1) - P(x,y-1))/2
    gP = np.zeros((3, H, W))
    gP[:, 1:-1, 2:] += 0.5 * ga[:, 1:-1, 1:-1]
    gP[:, 1:-1, :-2] -= 0.5 * ga[:, 1:-1, 1:-1]
    gP[:, 2:, 1:-1] += 0.5 * gb[:, 1:-1, 1:-1]
    gP[:, :-2, 1:-1] -= 0.5 * gb[:, 1:-1, 1:-1]
    gz = (gP * t["r"]).sum(0)  # P = zbar r
    As = np.where(t["surf"], A, 1.0)
    gD = gD + np.where(t["surf"], gz / As, 0.0)  # zbar = D / A
    gA = gA - np.where(t["surf"], gz * D / (As * As), 0.0)
    return dict(L_d=L_d, L_n=L_n, gA=gA, gD=gD, gM1=gM1, gM2=gM2, gN=gN, Nhat=Nhat)
