"""Pins of the 3D-Gaussian variant of the oracle (Appendix B; reading R-3D) against things other than
itself: closed forms for on-axis Gaussians, central differences of the textbook pinhole projection (pins the Jacobian and
the covariance composition), brute force (no boxes, no tiles, exhaustive per-pixel sort), the fp64 extent of the box,
and the paper's two disqualified cases."""
import math

import numpy as np
import pytest

import oracle as orc
from paper_2501_08174_b200 import scenegen as sg

Y0 = 0.5 * math.sqrt(1.0 / math.pi)


def ident_cam(W, H, f):
    return orc.make_camera(np.eye(4, dtype=np.float32), f, f, W / 2, H / 2, W, H)


def gaussians(rows):
    """rows: (pos, scale3, quat, opacity, rgb)"""
    n = len(rows)
    sh = np.zeros((n, 16, 3), np.float32)
    for i, r in enumerate(rows):
        sh[i, 0] = (np.asarray(r[4]) - 0.5) / Y0
    return (np.asarray([r[0] for r in rows], np.float32), np.asarray([r[1] for r in rows], np.float32),
            np.asarray([r[2] for r in rows], np.float32), np.asarray([r[3] for r in rows], np.float32), sh)


def forward(P, cam, cfg, **kw):
    pre = orc.preprocess3d(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    return pre, srt, orc.render3d_fwd(pre, srt, P[3], cam, cfg, **kw)


def test_on_axis_gaussian_closed_form_and_depth_axis_independence():
    """Identity camera, Gaussian on the optical axis with axis-aligned scales (a, b, c): J's third column vanishes there, so
    Sigma' = diag((f a/z)^2, (f b/z)^2) + 0.3 I whatever c is, and alpha = o exp(-(dx^2/sxx + dy^2/syy)/2)."""
    W = H = 64
    f, z0, o = 100.0, 2.0, 0.8
    rgb = np.array([0.2, 0.5, 0.9])
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    dx, dy = xs - (W / 2 - 0.5), ys - (H / 2 - 0.5)
    ref = None
    for (a, b, c) in ((0.10, 0.16, 0.05), (0.10, 0.16, 0.30), (0.12, 0.12, 0.12)):
        P = gaussians([((0, 0, z0), (a, b, c), (1, 0, 0, 0), o, rgb)])
        pre, srt, fw = forward(P, ident_cam(W, H, f), orc.default_config(sh_degree=0))
        sxx, syy = (f * a / z0) ** 2 + 0.3, (f * b / z0) ** 2 + 0.3
        rho = dx * dx / sxx + dy * dy / syy
        expect = np.where(rho <= 9.0, o * np.exp(-0.5 * rho), 0.0)
        edge = np.abs(rho - 9.0) < 1e-4
        assert np.abs((fw["alpha"] - expect) * ~edge).max() < 1e-6
        assert np.abs((fw["color"] - expect[None] * rgb[:, None, None]) * ~edge).max() < 1e-6
        assert np.abs((fw["depth"] - expect * z0) * ~edge).max() < 1e-5  # centre depth
        # box: centre +- sqrt(rho_cut * Sigma'_xx), pixel-exact
        cx0, cy0 = W / 2 - 0.5, H / 2 - 0.5
        assert list(pre["rect"][0]) == [math.ceil(cx0 - 3 * math.sqrt(sxx)), math.ceil(cy0 - 3 * math.sqrt(syy)),
                                        math.floor(cx0 + 3 * math.sqrt(sxx)), math.floor(cy0 + 3 * math.sqrt(syy))]
        if (a, b) == (0.10, 0.16):
            ref = fw["alpha"] if ref is None else ref
            assert np.abs(fw["alpha"] - ref).max() < 1e-7  # the scale along the viewing axis does not matter on the axis


def test_rotation_about_the_view_axis_swaps_the_image_axes():
    W = H = 48
    q90 = (math.cos(math.pi / 4), 0.0, 0.0, math.sin(math.pi / 4))  # 90 degrees about z
    cfg = orc.default_config(sh_degree=0)
    _, _, f0 = forward(gaussians([((0, 0, 2.0), (0.05, 0.12, 0.02), (1, 0, 0, 0), 0.7, (0.5, 0.5, 0.5))]), ident_cam(W, H, 80.0), cfg)
    _, _, f1 = forward(gaussians([((0, 0, 2.0), (0.05, 0.12, 0.02), q90, 0.7, (0.5, 0.5, 0.5))]), ident_cam(W, H, 80.0), cfg)
    assert np.abs(f1["alpha"] - f0["alpha"].T).max() < 1e-6


def test_projected_covariance_matches_central_differences_of_the_pinhole_projection():
    """Sigma' = J W Sigma W^T J^T + 0.3 I with J the Jacobian of pi(t) = (fx tx/tz, fy ty/tz): for the three principal axes
    b_k = s_k R e_k of the Gaussian, (pi(p + eps b_k) - pi(p - eps b_k)) / (2 eps) -> J W b_k, so the sum of their outer
    products is J W Sigma W^T J^T.  Uses only the textbook projection, a generic camera pose and off-axis Gaussians."""
    sc = sg.random_scene(40, 64, 48, 60.0, seed=11, sh_degree=0)
    s3 = np.concatenate([sc.scale, 0.5 * sc.scale[:, :1]], 1).astype(np.float32)
    camn = sc.cameras[0]
    cam = orc.camera_from(camn)
    pre = orc.preprocess3d(sc.pos, s3, sc.quat, sc.opacity, sc.sh, cam, orc.default_config(sh_degree=0))
    V = camn.view.astype(np.float64)

    def pi(X):
        t = V[:3, :3] @ X + V[:3, 3]
        return np.array([camn.fx * t[0] / t[2], camn.fy * t[1] / t[2]])

    checked = 0
    for j in range(sc.n):
        if not pre["visible"][j]:
            continue
        w, x, y, z = sc.quat[j].astype(np.float64)
        R = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                      [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                      [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])
        p = sc.pos[j].astype(np.float64)
        cov = 0.3 * np.eye(2)
        for k in range(3):
            bk = s3[j, k] * R[:, k]
            eps = 1e-4
            d = (pi(p + eps * bk) - pi(p - eps * bk)) / (2 * eps)
            cov += np.outer(d, d)
        Q = np.linalg.inv(cov)
        got = pre["conic"][j].astype(np.float64)
        assert np.allclose(got, [Q[0, 0], Q[0, 1], Q[1, 1]], rtol=2e-5, atol=1e-9), (j, got, Q)
        c = pi(p) + np.array([camn.cx - 0.5, camn.cy - 0.5])
        assert np.allclose(pre["c2d"][j], c, atol=2e-4)
        checked += 1
    assert checked > 15


def _compare_bf_tiled(sc, s3, view, cfg, tol=2e-5):
    cam = orc.camera_from(sc.cameras[view])
    m = sc.mask(view)
    P = (sc.pos, s3, sc.quat, sc.opacity, sc.sh)
    pre, srt, fw = forward(P, cam, cfg, mask=m)
    bf = orc.bf3d_render(*P, cam, cfg, mask=m)
    ok = fw["fragile"] == 0
    assert ok.mean() > 0.99
    for k in ("color", "alpha", "depth"):
        scale = 1.0 if k != "depth" else np.maximum(1.0, np.abs(bf[k]))
        assert ((np.abs(fw[k] - bf[k]) / scale) * ok).max() < tol, k
    untouched = fw["fragile_touch"] == 0
    assert np.array_equal(fw["vis_count"][untouched], bf["vis_count"][untouched])
    assert np.allclose(fw["contrib_sum"][untouched], bf["contrib_sum"][untouched], rtol=1e-4, atol=1e-6)
    return fw, bf


def test_bruteforce_equals_tiled_random_scenes_and_config1():
    for seed in (1, 2):
        sc = sg.random_scene(60, 56, 40, 50.0, seed=seed, sh_degree=3)
        s3 = np.concatenate([sc.scale, 0.4 * sc.scale[:, 1:]], 1).astype(np.float32)
        _compare_bf_tiled(sc, s3, 0, orc.default_config(sh_degree=3, bg=(0.3, 0.1, 0.2)))
    sc = sg.make_scene("config1")
    s3 = np.concatenate([sc.scale, 0.2 * sc.scale[:, :1]], 1).astype(np.float32)
    fw, _ = _compare_bf_tiled(sc, s3, 1, orc.default_config(sh_degree=0))
    assert fw["alpha"].max() > 0.9


def test_box_fp32_is_conservative_at_config2_scale():
    """The integer rect of the fp32 sequence contains the fp64 extent c +- sqrt(rho_cut Sigma'_xx) of every visible Gaussian
    of full-size config 2 and exceeds it by at most one pixel."""
    sc = sg.make_scene("config2")
    s3 = np.concatenate([sc.scale, 0.3 * sc.scale[:, :1]], 1).astype(np.float32)
    camn = sc.cameras[3]
    pre = orc.preprocess3d(sc.pos, s3, sc.quat, sc.opacity, sc.sh, orc.camera_from(camn), orc.default_config(sh_degree=3))
    vis = pre["visible"] == 1
    assert vis.sum() > 100_000
    q = sc.quat.astype(np.float64)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.stack([np.stack([1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)], 1),
                  np.stack([2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)], 1),
                  np.stack([2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)], 1)], 1)  # [n,3,3]
    V = camn.view.astype(np.float64)
    Wm = V[:3, :3]
    t = sc.pos.astype(np.float64) @ Wm.T + V[:3, 3]
    B = np.einsum("ab,nbk->nak", Wm, R) * s3[:, None, :].astype(np.float64)  # W R diag(s)
    S = np.einsum("nak,nbk->nab", B, B)
    J = np.zeros((sc.n, 2, 3))
    J[:, 0, 0] = camn.fx / t[:, 2]; J[:, 0, 2] = -camn.fx * t[:, 0] / t[:, 2] ** 2
    J[:, 1, 1] = camn.fy / t[:, 2]; J[:, 1, 2] = -camn.fy * t[:, 1] / t[:, 2] ** 2
    cov = np.einsum("nak,nkl,nbl->nab", J, S, J)
    rc = np.minimum(9.0, 2 * np.log(np.maximum(sc.opacity.astype(np.float64), 1e-12) * 255.0))
    c = np.stack([camn.fx * t[:, 0] / t[:, 2] + camn.cx - 0.5, camn.fy * t[:, 1] / t[:, 2] + camn.cy - 0.5], 1)
    WH = (camn.width, camn.height)
    rect = pre["rect"][vis].astype(np.int64)
    for r in (0, 1):
        h = np.sqrt(rc * (cov[:, r, r] + 0.3))
        e0 = np.clip(np.ceil(c[vis, r] - h[vis]), 0, WH[r] - 1)
        e1 = np.clip(np.floor(c[vis, r] + h[vis]), 0, WH[r] - 1)
        assert np.all(rect[:, r] <= e0) and np.all(rect[:, 2 + r] >= e1)
        assert np.all(rect[:, r] >= e0 - 1) and np.all(rect[:, 2 + r] <= e1 + 1)


def test_occluded_and_out_of_frustum_gaussians_are_never_used():
    """PAPER.md:119 carried over to 3DGS: G_j in the frustum behind saturated pixels and G_k outside the
    frustum both end with vis_count = 0 and are pruned; the front layers stay."""
    W = H = 32
    front = [((0, 0, 1.0 + 0.1 * i), (20.0, 20.0, 0.01), (1, 0, 0, 0), 0.95, (0.3, 0.6, 0.1)) for i in range(5)]
    rows = front + [((0.02, -0.01, 2.0), (0.05, 0.05, 0.05), (1, 0, 0, 0), 0.9, (0.9, 0.1, 0.1)),
                    ((50.0, 0.0, 2.0), (0.05, 0.05, 0.05), (1, 0, 0, 0), 0.9, (0.1, 0.9, 0.1)),
                    ((0.0, 0.0, -2.0), (0.05, 0.05, 0.05), (1, 0, 0, 0), 0.9, (0.1, 0.1, 0.9))]
    P = gaussians(rows)
    pre, srt, fw = forward(P, ident_cam(W, H, 30.0), orc.default_config(sh_degree=0))
    assert pre["visible"][5] == 1 and pre["visible"][6] == 0 and pre["visible"][7] == 0
    assert np.all(fw["vis_count"][:3] == W * H) and np.all(fw["vis_count"][3:] == 0)
    po = orc.prune(fw["vis_count"], fw["contrib_sum"].astype(np.float32), P[3])
    assert list(po["prune_mask"]) == [0, 0, 0, 1, 1, 1, 1, 1]
