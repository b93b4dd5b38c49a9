"""CPU ORACLE of the clone / split half of the adaptive density control ("the density of the Gaussians is
adaptively controlled", :129 "Regarding the adaptive density control, we use the same default values as 2DGS, which
correspond to the 3DGS defaults").  TEST INFRASTRUCTURE ONLY: only tests/ may import this.  Plain numpy, fp64 arithmetic
on the fp32 inputs, one step after the other; shares nothing with the CUDA library.

The paper gives no formulas (it inherits the published 3DGS procedure); reading R-densify, for 2D surfels:

  statistics over an interval (accumulate):  for every view in which surfel j passes the frustum test of O1,
      grad_accum[j] += || d_center2d_j ||_2   (d_center2d = gradient w.r.t. the projected centre, reading R-c2d)
      denom[j]      += 1
  densify:  avg_j = grad_accum_j / denom_j (0 where denom_j = 0);  selected_j = avg_j >= grad_threshold (default 2e-4);
      clone_j = selected_j and max(s_u, s_v) <= scale_threshold;  split_j = selected_j and max(s_u, s_v) > scale_threshold
      (scale_threshold = 0.01 x scene extent in the published defaults);
      output rows, in this order:
        (1) every surfel that is not split, ascending id, unchanged;
        (2) one copy of every cloned surfel, ascending id;
        (3) two children of every split surfel, ascending id, child 0 then child 1:
            position p + s_u xi[j,k,0] t_u + s_v xi[j,k,1] t_v  (a draw from the surfel's own Gaussian in its tangent plane;
            the standard-normal numbers xi [N,2,2] are INPUTS), scales (s_u, s_v) / 1.6, everything else copied;
      src[row] = id of the surfel the row comes from;  n_out = n - n_split + n_clone + 2 n_split.
"""
from __future__ import annotations

import numpy as np

SPLIT_SCALE_DIVISOR = 1.6


def accumulate(grad_accum, denom, d_center2d, in_frustum, width, height):
    """One view's contribution to the statistics (in place).  The statistic is the norm of the gradient w.r.t. the projected
    centre in NDC units (pixel = ((ndc + 1) W - 1) / 2, so d/d ndc = (W/2, H/2) d/d pixel): the unit in which the cited
    work's default threshold 2e-4 ("the same default values as 2DGS, which correspond to the 3DGS defaults")
    is calibrated; d_center2d itself is per pixel (reading R-c2d)."""
    g = np.asarray(d_center2d, np.float64)
    m = np.asarray(in_frustum).astype(bool)
    grad_accum[m] += np.sqrt((0.5 * width * g[m, 0]) ** 2 + (0.5 * height * g[m, 1]) ** 2)
    denom[m] += 1
    return grad_accum, denom


def tangents(quat):
    """t_u, t_v of R(q) (S19: polynomial in (w, x, y, z), no normalisation)."""
    q = np.asarray(quat, np.float64)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    tu = np.stack([1 - 2 * (y * y + z * z), 2 * (x * y + w * z), 2 * (x * z - w * y)], 1)
    tv = np.stack([2 * (x * y - w * z), 1 - 2 * (x * x + z * z), 2 * (y * z + w * x)], 1)
    return tu, tv


def densify(pos, scale, quat, opacity, sh, grad_accum, denom, grad_threshold, scale_threshold, xi):
    pos, scale, quat, opacity, sh = (np.asarray(a, np.float32) for a in (pos, scale, quat, opacity, sh))
    n = pos.shape[0]
    ga = np.asarray(grad_accum, np.float32).astype(np.float64)
    dn = np.asarray(denom).astype(np.float64)
    avg = np.where(dn > 0, ga / np.maximum(dn, 1.0), 0.0)
    # the decision is taken in fp32 like the kernel's (avg and the threshold rounded to fp32 first)
    selected = avg.astype(np.float32) >= np.float32(grad_threshold)
    big = np.maximum(scale[:, 0], scale[:, 1]) > np.float32(scale_threshold)
    clone = selected & ~big
    split = selected & big
    keep_ids = np.nonzero(~split)[0]
    clone_ids = np.nonzero(clone)[0]
    split_ids = np.nonzero(split)[0]
    tu, tv = tangents(quat)
    xi = np.asarray(xi, np.float32).astype(np.float64).reshape(n, 2, 2)
    out = dict(pos=[], scale=[], quat=[], opacity=[], sh=[])
    src = []

    def emit(j, p=None, s=None):
        out["pos"].append(pos[j].astype(np.float64) if p is None else p)
        out["scale"].append(scale[j].astype(np.float64) if s is None else s)
        out["quat"].append(quat[j]); out["opacity"].append(opacity[j]); out["sh"].append(sh[j])
        src.append(j)

    for j in keep_ids:
        emit(j)
    for j in clone_ids:
        emit(j)
    for j in split_ids:
        su, sv = float(scale[j, 0]), float(scale[j, 1])
        for k in range(2):
            p = pos[j].astype(np.float64) + su * xi[j, k, 0] * tu[j] + sv * xi[j, k, 1] * tv[j]
            emit(j, p=p, s=np.array([su, sv]) / SPLIT_SCALE_DIVISOR)
    res = {k: (np.stack(v) if v else np.zeros((0,) + {"pos": (3,), "scale": (2,), "quat": (4,), "opacity": (), "sh": (16, 3)}[k]))
           for k, v in out.items()}
    res.update(src=np.asarray(src, np.int32), n_out=len(src), n_keep=len(keep_ids), n_clone=len(clone_ids), n_split=len(split_ids),
               cls=np.where(split, 2, np.where(clone, 1, 0)).astype(np.uint8))
    return res
