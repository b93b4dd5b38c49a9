"""-m gpu: ocgs_photometric_loss (masked photometric loss L_c^M, Eq. 2) against
oracle/photometric.py, element by element.

Tolerances: the three loss scalars to 1e-5 absolute (north_star's 1e-4 for "the loss"
with margin); the gradient entry-wise to 1e-3 relative + 1e-3 of the largest |entry| of the image (every entry is of
order lam/(3HW), far below north_star's absolute floor of 1e-6 at any realistic size, so the floor is scaled)."""
import numpy as np
import pytest

from oracle import photometric as ph

pytestmark = pytest.mark.gpu


def run_gpu(R, I, M, lam):
    import torch
    from paper_2501_08174_b200 import binding as B
    H, W = R.shape[-2:]
    c = torch.tensor(np.ascontiguousarray(R, np.float32), device="cuda")
    t = torch.tensor(np.ascontiguousarray(I, np.float32), device="cuda")
    m = None if M is None else torch.tensor(np.ascontiguousarray(M, np.uint8), device="cuda")
    g = torch.full((3, H, W), 7.0, dtype=torch.float32, device="cuda")
    loss = torch.zeros(3, dtype=torch.float32, device="cuda")
    ws = torch.empty(B.ocgs_photometric_workspace_bytes(W, H), dtype=torch.uint8, device="cuda")
    B.ocgs_photometric_loss(c, t, m, W, H, lam, g, loss, ws)
    torch.cuda.synchronize()
    return g.cpu().numpy(), loss.cpu().numpy()


def check(R, I, M, lam):
    g, loss = run_gpu(R, I, M, lam)
    # the kernel reads fp32 images: give the oracle the same rounded inputs
    R32, I32 = np.asarray(R, np.float32), np.asarray(I, np.float32)
    o = ph.photometric_loss(R32, I32, M, lam=lam)
    assert abs(loss[0] - o["loss"]) <= 1e-5 and abs(loss[1] - o["l1"]) <= 1e-5 and abs(loss[2] - o["dssim"]) <= 1e-5, (loss, o["loss"], o["l1"], o["dssim"])
    ref = o["grad"]
    # away from the |x - y| kink (fp32 and fp64 agree on x - y exactly: both subtract the same fp32 values)
    tol = 1e-3 * np.abs(ref) + 1e-3 * np.abs(ref).max()
    assert np.all(np.abs(g - ref) <= tol), float((np.abs(g - ref) / np.abs(ref).max()).max())
    if M is not None:
        assert np.all(g[:, np.asarray(M) == 0] == 0.0)
    return loss, o


def scene_like_images(seed, H, W):
    """Smooth structure + noise + flat regions, values in [0, 1]: the statistics SSIM is sensitive to."""
    rng = np.random.default_rng(seed)
    yy, xx = np.mgrid[0:H, 0:W]
    base = np.stack([0.5 + 0.4 * np.sin(xx / (7.0 + c) + c) * np.cos(yy / (11.0 - c)) for c in range(3)])
    R = np.clip(base + rng.normal(0, 0.03, base.shape), 0, 1)
    I = np.clip(base + rng.normal(0, 0.03, base.shape) + 0.05 * np.sin(xx / 3.0), 0, 1)
    R[:, : H // 4, : W // 3] = 0.25  # flat patch: variances cancel, the hardest case for fp32 moments
    I[:, : H // 4, : W // 3] = 0.25
    M = ((xx - W / 2) ** 2 / (0.45 * W) ** 2 + (yy - H / 2) ** 2 / (0.4 * H) ** 2 < 1).astype(np.uint8)
    return R, I, M


def test_small_ragged_image_all_lambdas():
    # 70 x 45: three tile columns, two tile rows, ragged on both axes; window reaches across tile borders
    R, I, M = scene_like_images(0, 45, 70)
    for lam in (0.0, 0.2, 1.0):
        check(R, I, M, lam)
    check(R, I, None, 0.2)


def test_identical_images_and_empty_mask():
    R, _, M = scene_like_images(1, 40, 40)
    g, loss = run_gpu(R, R, M, 0.2)
    # exact answer 0; fp32 moments leave 1e-4 of the gradient scale lam / (3 H W)
    assert np.abs(loss).max() <= 1e-6 and np.abs(g).max() <= 1e-3 * 0.2 / (3 * 40 * 40)
    g, loss = run_gpu(R, 1.0 - R, np.zeros_like(M), 0.2)
    assert np.abs(loss).max() <= 1e-6 and np.all(g == 0.0)


def test_tiny_image_smaller_than_the_window():
    R, I, M = scene_like_images(2, 7, 5)
    check(R, I, None, 0.2)


def test_invalid_arguments():
    import torch
    from paper_2501_08174_b200 import binding as B
    t = torch.zeros((3, 8, 8), device="cuda")
    ws = torch.empty(B.ocgs_photometric_workspace_bytes(8, 8), dtype=torch.uint8, device="cuda")
    with pytest.raises(B.OcgsError):
        B.ocgs_photometric_loss(t, t, None, 8, 8, 1.5, t.clone(), None, ws)
    with pytest.raises(B.OcgsError):
        B.ocgs_photometric_loss(t, t, None, 0, 8, 0.2, t.clone(), None, ws)


def test_config3_size_render_vs_target():
    """1600 x 1200 (BASELINE.json configs[2]): a rendered view of the scene against the render of its perturbed copy,
    with the analytic object mask -- the images bench.py's --loss dssim step feeds the kernel."""
    import torch
    from gpu_harness import GpuView
    from paper_2501_08174_b200 import scenegen as sg
    sc = sg.make_scene("config3")
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    pert = sc.perturbed()
    imgs = []
    for S in (P, (pert.pos, pert.scale, pert.quat, pert.opacity, pert.sh)):
        g = GpuView(S, sc.cameras[0], dict(sh_degree=3), key_capacity=48 * sc.n)
        g.preprocess(); g.bin_sort(want_ids=False)
        imgs.append(g.render_fwd(mask=None, stats=False, want_loss=False)["color"])
        del g
        torch.cuda.empty_cache()
    M = sc.mask(0)
    loss, o = check(imgs[0], imgs[1], M, 0.2)
    assert 0.0 < o["dssim"] < 0.5 and o["l1"] > 0.0
