"""-m gpu: ocgs_regularizers (L_d, L_n of Eq. 3) against oracle/regularizers.py,
and the whole chain render_fwd_reg -> regularizers -> render_bwd_reg against the oracle's chain.

Tolerances: losses 1e-5 relative + 1e-7; upstream-gradient maps entry-wise 1e-3 relative + 1e-3 of the map's largest
entry (entries are O(1/hw), below north_star's absolute 1e-6 floor, so the floor is scaled as for the photometric loss);
parameter gradients through the chain by the rule of check_grads."""
import numpy as np
import pytest

from gpu_harness import GpuView, check_grads, oracle_view
from oracle import regularizers as rg
from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu


def run_gpu(A, D, mom, Nrm, cam_np, w_d, w_n):
    import torch
    from paper_2501_08174_b200 import binding as B
    H, W = A.shape
    dev = lambda a: torch.tensor(np.ascontiguousarray(a, np.float32), device="cuda")
    tA, tD, tM, tN = dev(A), dev(D), dev(mom), dev(Nrm)
    gA, gD = (torch.full((H, W), 7.0, device="cuda") for _ in range(2))
    gM = torch.full((2, H, W), 7.0, device="cuda")
    gN = torch.full((3, H, W), 7.0, device="cuda")
    loss = torch.zeros(2, device="cuda")
    ws = torch.empty(B.ocgs_regularizers_workspace_bytes(W, H), dtype=torch.uint8, device="cuda")
    B.ocgs_regularizers(tA, tD, tM, tN, B.camera_from(cam_np), w_d, w_n, gA, gD, gM, gN, loss, ws)
    torch.cuda.synchronize()
    gM = gM.cpu().numpy()
    return dict(gA=gA.cpu().numpy(), gD=gD.cpu().numpy(), gM1=gM[0], gM2=gM[1], gN=gN.cpu().numpy()), loss.cpu().numpy()


def compare(A, D, mom, Nrm, cam_np, w_d, w_n):
    A, D, mom, Nrm = (np.asarray(t, np.float32) for t in (A, D, mom, Nrm))  # both sides see the same fp32 maps
    g, loss = run_gpu(A, D, mom, Nrm, cam_np, w_d, w_n)
    o = rg.regularizers(A, D, mom[1], mom[2], Nrm, cam_np.fx, cam_np.fy, cam_np.cx, cam_np.cy, w_d=w_d, w_n=w_n)
    assert abs(loss[0] - o["L_d"]) <= 1e-5 * abs(o["L_d"]) + 1e-7, (loss[0], o["L_d"])
    assert abs(loss[1] - o["L_n"]) <= 1e-5 * abs(o["L_n"]) + 1e-7, (loss[1], o["L_n"])
    for k in ("gA", "gD", "gM1", "gM2", "gN"):
        ref = o[k]
        tol = 1e-3 * np.abs(ref) + 1e-3 * np.abs(ref).max() + 1e-30
        assert np.all(np.abs(g[k] - ref) <= tol), (k, float((np.abs(g[k] - ref) / (np.abs(ref).max() + 1e-30)).max()))
    return g, o


def synthetic_maps(seed, H, W):
    rng = np.random.default_rng(seed)
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    A = np.clip(0.55 + 0.45 * np.sin(xs / 9.0) * np.cos(ys / 7.0), 0.0, 1.0)
    A[(xs - W / 2) ** 2 + (ys - H / 3) ** 2 < 30] = 0.0  # a hole without surface
    zbar = 2.5 + 0.3 * np.sin(xs / 6.0 + 0.3) + 0.2 * np.cos(ys / 5.0) + 0.002 * rng.normal(size=(H, W))
    D = A * zbar
    mom = np.stack([zbar - 0.05, A * (0.05 + 0.02 * np.sin(xs / 4.0)), A * (0.004 + 0.003 * rng.uniform(size=(H, W)))])
    n = rng.normal(size=(3, H, W)) * 0.2 + np.array([0.1, -0.2, -0.9])[:, None, None]
    return A, D, mom, A[None] * n


def test_synthetic_maps_ragged_sizes():
    for (H, W, f) in ((37, 50, 60.0), (8, 33, 25.0), (3, 3, 4.0)):
        cam = sg.make_camera((0.0, -3.0, 0.5), W, H, f)
        A, D, mom, Nrm = synthetic_maps(H, H, W)
        for w_d, w_n in ((1.0, 0.0), (0.0, 1.0), (100.0, 0.05)):
            compare(A, D, mom, Nrm, cam, w_d, w_n)


def test_rendered_maps_and_chain_to_parameter_gradients():
    """config 2 geometry (40 k surfels, 800x600): forward with the moment map, regularisers on the rendered maps, backward
    with their four upstream gradients; the oracle runs the same chain in fp64."""
    sc = sg.make_scene("config2", n_obj=20_000, n_bg=20_000)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    camn = sc.cameras[2]
    orc, cam, cfg, pre, srt, fw = oracle_view(P, camn, dict(sh_degree=3), mask=None)
    g = GpuView(P, camn, dict(sh_degree=3))
    g.preprocess(); g.bin_sort(want_ids=False)
    gf = g.render_fwd(mask=None, moments=True)
    ok = fw["fragile"] == 0
    # (a) the regulariser kernel on the GPU's own maps against the oracle on the same maps
    w_d, w_n = 100.0, 0.05  # the weights 2DGS uses for bounded / DTU-like scenes are of this order
    gg, o = compare(gf["alpha"], gf["depth"], gf["moments"], gf["normal"], camn, w_d, w_n)
    assert o["L_d"] > 0 and 0 < o["L_n"] < 1
    # (b) the chain into the backward pass.  Both sides take the regulariser gradients of the SAME maps (the GPU's fp32
    # maps: `o` is the oracle's regulariser on them, `gg` the kernel's): finite-difference normals amplify the 1e-5
    # rounding differences between the two forward passes' depth maps by 1/(pixel footprint) ~ 250, so a comparison
    # from independent forward maps would test the conditioning of depth differencing, not the kernels.
    # Fragile pixels get zero upstream gradient on both sides (S22).
    oo = o
    # scale the upstream maps to O(1) so that parameter gradients sit well above check_grads' absolute floor
    s = float(camn.width * camn.height)
    okf = ok.astype(np.float64)
    up_o = {k: oo[k] * okf * s for k in ("gA", "gD", "gM1", "gM2", "gN")}
    up_g = {k: gg[k].astype(np.float64) * okf * s for k in ("gA", "gD", "gM1", "gM2", "gN")}
    cfg0 = orc.default_config(sh_degree=3, gamma_bg=0.0)
    og = orc.render_bwd(*P, pre, srt, cam, cfg0, mask=None, gA=up_o["gA"].astype(np.float32), gD=up_o["gD"].astype(np.float32),
                        gN=up_o["gN"].astype(np.float32), gM1=up_o["gM1"].astype(np.float32), gM2=up_o["gM2"].astype(np.float32))
    g.cfg.gamma_bg = 0.0
    gb = g.render_bwd(gA=up_g["gA"], gD=up_g["gD"], gN=up_g["gN"], gM=np.stack([up_g["gM1"], up_g["gM2"]]), mask=None)
    # absolute floor: the normal-consistency channels cancel against each other for surfels aligned with the depth normal
    # (dl/dA = 1 against dl/dNrm = -Nhat: the surfel's total is (1 - n.Nhat) of its terms) and the distortion channels are
    # differences of fp32 depths, so entries far below an array's typical scale are fp32-limited
    check_grads(gb, og, rel=2e-3, floor_frac=1e-4)  # two fp32 stages (maps, then regulariser gradients) feed this backward
