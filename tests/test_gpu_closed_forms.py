"""-m gpu: the CUDA path against the closed forms north_star names, directly (no oracle in between): the analytic Gaussian
footprint of a fronto-parallel surfel, exact zero contribution and exact zero gradients behind opaque front layers
(PAPER.md:119, :121), the two disqualified cases G_j / G_k of PAPER.md:119, and Eq. 1 on the rendered alpha."""
import math

import numpy as np
import pytest

from gpu_harness import GpuView
from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu

Y0 = 0.5 * math.sqrt(1.0 / math.pi)


def surfels(rows):
    """rows: (pos, scale, quat, opacity, rgb)"""
    n = len(rows)
    sh = np.zeros((n, 16, 3), np.float32)
    for i, r in enumerate(rows):
        sh[i, 0] = (np.asarray(r[4]) - 0.5) / Y0
    return (np.asarray([r[0] for r in rows], np.float32), np.asarray([r[1] for r in rows], np.float32),
            np.asarray([r[2] for r in rows], np.float32), np.asarray([r[3] for r in rows], np.float32), sh)


def ident_cam(W, H, f):
    return sg.Camera(view=np.eye(4, dtype=np.float32), fx=f, fy=f, cx=W / 2.0, cy=H / 2.0, width=W, height=H)


def test_fronto_parallel_surfel_is_the_analytic_gaussian():
    W = H = 64
    f, z0, su, sv, o = 100.0, 2.0, 0.10, 0.16, 0.8
    rgb = np.array([0.2, 0.5, 0.9])
    g = GpuView(surfels([((0, 0, z0), (su, sv), (1, 0, 0, 0), o, rgb)]), ident_cam(W, H, f), dict(sh_degree=0))
    g.preprocess(); g.bin_sort()
    m = np.zeros((H, W), np.uint8); m[:, : W // 2] = 1
    fw = g.render_fwd(mask=m)
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    u = (xs - (W / 2 - 0.5)) * z0 / (f * su)
    v = (ys - (H / 2 - 0.5)) * z0 / (f * sv)
    rho = u * u + v * v
    expect = np.where(rho <= 9.0, np.minimum(0.99, o * np.exp(-0.5 * rho)), 0.0)
    edge = np.abs(rho - 9.0) < 1e-3  # the 3-sigma cut-off is a discontinuity: skip pixels that sit on it
    assert np.abs((fw["alpha"] - expect) * ~edge).max() < 2e-6
    assert np.abs((fw["color"] - expect[None] * rgb[:, None, None]) * ~edge).max() < 2e-6
    assert np.abs((fw["depth"] - expect * z0) * ~edge).max() < 1e-5
    assert np.abs((fw["normal"][2] + expect) * ~edge).max() < 2e-6  # t_w = +z faces away: flipped to -z
    # Eq. 1: L_b = 1/(hw) sum A (1 - M), here on the analytic alpha
    assert fw["loss_bg"] == pytest.approx((expect * (1 - m)).sum() / (H * W), abs=2e-6)
    assert fw["vis_count"][0] == int((expect > 0).sum()) or abs(int(fw["vis_count"][0]) - int((expect > 0).sum())) <= int(edge.sum())
    assert fw["contrib_sum"][0] == pytest.approx(expect.sum(), rel=1e-4)


def test_opaque_front_layers_give_exact_zero_behind_and_disqualified_cases():
    """G_j inside the frustum whose every pixel saturates first, and G_k outside the frustum, are both never
    'used during the color accumulation step'; such Gaussians receive no gradient."""
    W = H = 32
    # five huge near-opaque layers: alpha = 0.95 * G with G > 0.999 over the image, so T = 0.0507, 2.6e-3, 1.3e-4 after one,
    # two, three layers and the fourth would leave 6.6e-6 < t_min = 1e-4: rendering terminates after three (S11), well
    # away from the borderline
    front = [((0, 0, 1.0 + 0.1 * i), (20.0, 20.0), (1, 0, 0, 0), 0.95, (0.3, 0.6, 0.1)) for i in range(5)]
    behind = ((0.02, -0.01, 2.0), (0.05, 0.05), (1, 0, 0, 0), 0.9, (0.9, 0.1, 0.1))      # G_j: in frustum, occluded everywhere
    outside = ((50.0, 0.0, 2.0), (0.05, 0.05), (1, 0, 0, 0), 0.9, (0.1, 0.9, 0.1))       # G_k: outside the frustum
    back = ((0.0, 0.0, -2.0), (0.05, 0.05), (1, 0, 0, 0), 0.9, (0.1, 0.1, 0.9))          # behind the camera
    g = GpuView(surfels(front + [behind, outside, back]), ident_cam(W, H, 30.0), dict(sh_degree=0))
    gp = g.preprocess()
    assert gp["tiles"][5] > 0 and gp["tiles"][6] == 0 and gp["tiles"][7] == 0
    g.bin_sort()
    fw = g.render_fwd(mask=np.zeros((H, W), np.uint8))
    assert np.all(fw["vis_count"][:3] == W * H) and np.all(fw["vis_count"][3:] == 0)
    assert np.all(fw["contrib_sum"][3:] == 0.0)
    assert np.all(fw["n_contrib"] == 3)
    assert fw["alpha"].min() > 0.9998 and fw["alpha"].max() < 0.9999  # "a threshold opacity close to 1"
    rng = np.random.default_rng(0)
    gg = g.render_bwd(gC=rng.normal(size=(3, H, W)), gA=rng.normal(size=(H, W)), gD=rng.normal(size=(H, W)), gN=rng.normal(size=(3, H, W)))
    for k in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
        assert np.all(gg[k][3:] == 0.0), k       # exact zeros for everything that was never blended
    assert np.abs(gg["d_opacity"][:3]).min() > 0.0
    # prune rule: exactly the never-blended ones go
    import torch
    from paper_2501_08174_b200 import binding as B
    mask_t = torch.empty(8, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(8, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    pws = torch.empty(B.ocgs_prune_workspace_bytes(8), dtype=torch.uint8, device="cuda")
    B.ocgs_prune_stats(g.surfels, g.vis, g.cs, g.cfg, mask_t, remap_t, None, n_out, 0, pws)
    torch.cuda.synchronize()
    assert list(mask_t.cpu().numpy()) == [0, 0, 0, 1, 1, 1, 1, 1] and int(n_out.item()) == 3
    assert list(remap_t.cpu().numpy()) == [0, 1, 2, -1, -1, -1, -1, -1]


def test_background_loss_gradient_sign_and_locality():
    """L_b 'penalizes Gaussian opacity where O is not present': with only gamma L_b active, dL/d opacity >= 0
    for every surfel and exactly 0 for surfels that only touch mask = 1 pixels."""
    sc = sg.random_scene(200, 96, 64, 70.0, seed=5, sh_degree=0)
    g = GpuView((sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh), sc.cameras[0], dict(sh_degree=0))
    gp = g.preprocess(); g.bin_sort()
    m = np.zeros((64, 96), np.uint8); m[:, :48] = 1
    g.render_fwd(mask=m)
    gg = g.render_bwd(mask=m)  # no upstream gradient: only the fused gamma (1 - M)/(hw) into dL/dA
    assert np.all(gg["d_opacity"] >= 0.0) and gg["d_opacity"].max() > 0.0
    vis = gp["tiles"] > 0
    left_only = vis & (gp["rect"][:, 2] < 48)  # pixel rect entirely inside the mask = 1 half
    assert left_only.any() and np.all(gg["d_opacity"][left_only] == 0.0)
    g.render_fwd(mask=np.ones((64, 96), np.uint8))
    gg1 = g.render_bwd(mask=np.ones((64, 96), np.uint8))
    assert all(np.all(v == 0.0) for v in gg1.values())  # M = 1 everywhere: L_b = 0 and so is its gradient
