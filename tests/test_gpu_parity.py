"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element, on seeded inputs.

Tolerances (north_star / DESIGN.md "tolerances"): integer outputs bit-exact; images, alpha, depth (relative to
max(1,|D|)) and L_b to 1e-4 on non-fragile pixels; gradients per check_grads (relative 1e-3 above 1e-6).
"""
import numpy as np
import pytest

from gpu_harness import GpuView, check_grads, oracle_view
from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu

IMG_TOL = 1e-4


def arrays(sc):
    return (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)


def full_parity(sc, view, cfg_kw, rng_seed=5, max_fragile=2e-3, with_bwd=True, key_capacity=None, check_prune=False, bench_step=False,
                max_illcond_err=IMG_TOL, label=None):
    """One view through the five C-ABI calls against the oracle, EVERY output, every pixel, every surfel.

    check_prune: the prune mask, remap and compaction from this view's statistics (a5) against the oracle's rule.
    bench_step:  additionally the step bench.py times -- ocgs_render_fwd_l1 (masked L1 fused, dL/dcolor made in-kernel) + the
                 colour / alpha-only backward instance -- against the oracle fed with ITS OWN dL/dC = M sign(R - I)/(3HW),
                 target I = the oracle's render of the perturbed copy.
    Prints one line of measured numbers (fragile fraction, worst errors, strict-rule misses); pytest -s shows it."""
    P = arrays(sc)
    camn = sc.cameras[view]
    m = sc.mask(view)
    orc, cam, cfg, pre, srt, fw = oracle_view(P, camn, cfg_kw, mask=m)
    g = GpuView(P, camn, cfg_kw, key_capacity=key_capacity)
    # (1) preprocess: integer outputs bit-exact
    gp = g.preprocess()
    vis = pre["visible"] == 1
    assert np.array_equal(gp["tiles"], pre["tiles_touched"])
    assert np.array_equal(gp["depth_bits"], pre["depth_bits"])
    assert np.array_equal(gp["rect"][vis], pre["rect"][vis])
    assert np.array_equal(gp["clamp"][vis], pre["clamp"][vis])  # reading R-clamp: the decision is an fp32 sequence both sides follow
    rec = gp["rec_id"][vis]
    if vis.any():
        # record (csrc/common.cuh): c2d, rho_cut, z_j and the packed pixel rect are bit-exact (Appendix A) ...
        assert np.array_equal(rec[:, 10:12], pre["c2d"][vis]) and np.array_equal(rec[:, 12], pre["rho_cut"][vis])
        assert np.array_equal(rec[:, 13], pre["M"][vis][:, 8])
        rb = rec[:, 14:16].copy().view(np.uint32)
        assert np.array_equal(np.stack([rb[:, 0] & 0xFFFF, rb[:, 0] >> 16, rb[:, 1] & 0xFFFF, rb[:, 1] >> 16], 1), pre["rect"][vis])
        # ... P, Q, R, D0 equal their definition evaluated in fp64 from the oracle's fp32 M
        M = pre["M"][vis].astype(np.float64)
        c = pre["c2d"][vis].astype(np.float64)
        m2, a0, a1 = M[:, 6:9], M[:, 0:3] - c[:, 0:1] * M[:, 6:9], M[:, 3:6] - c[:, 1:2] * M[:, 6:9]
        Pq, Qq, Rq = np.cross(m2, a1), np.cross(a0, m2), np.cross(a0, a1)
        ref = np.concatenate([Pq, Qq, Rq, (m2 * Rq).sum(1, keepdims=True)], 1)
        # (the kernel forms them in fp64 with fused multiply-adds, numpy without: equal to an fp32 ulp of the row scale)
        assert np.all(np.abs(rec[:, 0:10] - ref) <= 2e-7 * np.abs(ref).max(1, keepdims=True))
        assert np.abs(rec[:, 17:20] - pre["rgb"][vis]).max() < 4e-6  # fp32 colour sum against the fp64 value (R-clamp bound)
        assert np.abs(rec[:, 20:23] - pre["normal"][vis]).max() < 2e-6
    # (2) bin_sort: keys, order, ranges bit-exact
    gs = g.bin_sort()
    assert gs["error"] == 0 and gs["K"] == srt["K"] and gs["n_vis"] == int(vis.sum())
    assert np.array_equal(gs["ids"], srt["ids"])
    assert np.array_equal(gs["tile_keys"], (srt["keys"] >> np.uint64(32)).astype(np.uint32))
    assert np.array_equal(gs["ranges"], srt["ranges"])
    # (3) forward: every pixel.  fragile bit 0 = a decision within its margin (the two sides may take different branches:
    # bounded by the discontinuity jump 0.02); bit 1 only = ill-conditioned pair evaluation, nothing discontinuous: the same 1e-4
    # (measured: 7e-6 at config 3); such pixels are only left out of the upstream gradients of the backward comparison
    gf = g.render_fwd(mask=m)
    ok = fw["fragile"] == 0
    illc = fw["fragile"] == 2
    frag_frac = float(1.0 - ok.mean())
    assert frag_frac <= max_fragile, f"fragile fraction {frag_frac}"
    worst = {}
    for k in ("color", "alpha", "depth", "normal"):
        scale = np.maximum(1.0, np.abs(fw[k])) if k == "depth" else 1.0
        err = np.abs(gf[k] - fw[k]) / scale
        worst[k] = float((err * ok).max())
        worst[k + "_illcond"] = float((err * illc).max())
        assert worst[k] <= IMG_TOL, (k, worst[k])
        assert worst[k + "_illcond"] <= max_illcond_err, (k, "ill-conditioned pixel", worst[k + "_illcond"])
        assert err.max() <= 0.02, (k, "fragile pixel beyond the discontinuity bound", err.max())
    assert np.array_equal(gf["n_contrib"][ok], fw["n_contrib"][ok])
    assert abs(gf["loss_bg"] - fw["loss_bg"]) <= IMG_TOL
    dv = np.abs(gf["vis_count"].astype(np.int64) - fw["vis_count"].astype(np.int64))
    assert np.all(dv <= fw["fragile_touch"])
    clean = fw["fragile_touch"] == 0
    assert np.array_equal(gf["vis_count"][clean], fw["vis_count"][clean])
    assert np.allclose(gf["contrib_sum"][clean], fw["contrib_sum"][clean], rtol=1e-4, atol=2e-6)
    info = dict(fragile=frag_frac, K=srt["K"], worst=worst, loss_bg_err=abs(gf["loss_bg"] - fw["loss_bg"]),
                vis_count_diff_surfels=int((dv != 0).sum()))
    if check_prune:
        # (3b) a5 from this view's statistics: mask / remap / count bit-exact against the oracle's rule on the same statistics,
        # and against the oracle's OWN statistics wherever no fragile pixel was involved; compaction by its definition
        import torch
        B = g.B
        n = g.n
        mask_t = torch.empty(n, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(n, dtype=torch.int32, device="cuda")
        n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
        outs = [torch.full_like(t, -7.0) for t in (g.t["pos"], g.t["scale"], g.t["quat"], g.t["opacity"], g.t["sh"])]
        om = B.ocgs_surfels_mut(*[B._ptr(t) for t in outs], n)
        pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device="cuda")
        B.ocgs_prune_stats(g.surfels, g.vis, g.cs, g.cfg, mask_t, remap_t, om, n_out, 0, pws)
        torch.cuda.synchronize()
        pm = mask_t.cpu().numpy()
        po = orc.prune(gf["vis_count"], gf["contrib_sum"], sc.opacity)
        assert np.array_equal(pm, po["prune_mask"]) and np.array_equal(remap_t.cpu().numpy(), po["remap"]) and int(n_out.item()) == po["n_out"]
        po2 = orc.prune(fw["vis_count"], fw["contrib_sum"].astype(np.float32), sc.opacity)
        assert np.array_equal(pm[clean], po2["prune_mask"][clean])
        info["prune_mask_diff"] = int((pm != po2["prune_mask"]).sum())
        assert info["prune_mask_diff"] <= max(2, int(1e-5 * n))
        comp = orc.compact(dict(pos=sc.pos, scale=sc.scale, quat=sc.quat, opacity=sc.opacity, sh=sc.sh), pm)
        for t, name in zip(outs, ("pos", "scale", "quat", "opacity", "sh")):
            got = t.cpu().numpy()
            assert np.array_equal(got[:po["n_out"]], comp[name]), name
            assert np.all(got[po["n_out"]:] == -7.0), name
        del outs, om
    rep = None
    if with_bwd:
        # (4) backward: seeded N(0,1) upstream on all four maps, zero on fragile pixels (both sides see the same inputs)
        rng = np.random.default_rng(rng_seed)
        H, W = camn.height, camn.width
        okf = ok.astype(np.float64)
        gC, gA = rng.normal(size=(3, H, W)) * okf, rng.normal(size=(H, W)) * okf
        gD, gN = rng.normal(size=(H, W)) * okf, rng.normal(size=(3, H, W)) * okf
        mm = np.where(ok, m, 1).astype(np.uint8)
        gg = g.render_bwd(gC=gC, gA=gA, gD=gD, gN=gN, mask=mm)
        og = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=gC.astype(np.float32), gA=gA.astype(np.float32),
                            gD=gD.astype(np.float32), gN=gN.astype(np.float32))
        rep = check_grads(gg, og, cond_rho=fw["cond_rho"])
        # the colour / alpha-only instance of the kernel (no upstream gradient on the depth and normal maps)
        gg2 = g.render_bwd(gC=gC, gA=gA, mask=mm)
        og2 = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=gC.astype(np.float32), gA=gA.astype(np.float32))
        rep2 = check_grads(gg2, og2, cond_rho=fw["cond_rho"])
        # surfels never blended receive exactly zero gradient
        never = gf["vis_count"] == 0
        for k in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
            assert np.all(gg[k][never] == 0.0), k
        info["grads"] = {k: (v["strict_fail_frac"], v["worst_strict_rel"], v["worst_cond_units"]) for k, v in rep.items()}
        info["grads_colour_alpha"] = {k: (v["strict_fail_frac"], v["worst_strict_rel"], v["worst_cond_units"]) for k, v in rep2.items()}
    if bench_step:
        info["bench_step"] = bench_step_parity(sc, view, g, orc, cam, cfg, pre, srt, fw, gf, m)
    print(f"PARITY {label or sc.name} n={sc.n} {camn.width}x{camn.height} view {view}: {info}")
    return dict(fragile=frag_frac, grads=rep, K=srt["K"], info=info, ranges=srt["ranges"])


def bench_step_parity(sc, view, g, orc, cam, cfg, pre, srt, fw, gf, m):
    """The step bench.py times: ocgs_render_fwd_l1 + ocgs_render_bwd with dL/dcolor only (render_bwd_kernel<false,false>)."""
    import torch
    B = g.B
    P = arrays(sc)
    H, W = g.H, g.W
    HW3 = 3.0 * H * W
    # target image (Appendix B): the oracle's render of the perturbed copy
    pt = sc.perturbed()
    _, _, _, _, _, tw = oracle_view(arrays(pt), sc.cameras[view], dict(sh_degree=sc.sh_degree), mask=m)
    target = tw["color"].astype(np.float32)
    tt = torch.tensor(target, device="cuda")
    o2 = B.alloc_outputs(W, H)
    gC_t = torch.full_like(tt, 9.0); l1 = torch.zeros(1, device="cuda")
    vis_f = torch.zeros(g.n, dtype=torch.int32, device="cuda"); cs_f = torch.zeros(g.n, device="cuda")
    B.ocgs_render_fwd_l1(g.n, g.cam, g.cfg, g.ws, g.cap, g.mask_t, tt, o2["color"], o2["alpha"], o2["depth"], o2["normal"], o2["n_contrib"],
                         o2["loss_bg"], l1, gC_t, vis_f, cs_f)
    grads = B.alloc_grads(g.n)
    B.ocgs_render_bwd(g.surfels, g.cam, g.cfg, g.ws, g.cap, g.mask_t, o2["n_contrib"], gC_t, None, None, None, grads["d_pos"], grads["d_scale"],
                      grads["d_quat"], grads["d_opacity"], grads["d_sh"], grads["d_center2d"])
    torch.cuda.synchronize()
    # the fused forward writes the same maps, statistics and L_b as the plain forward
    for k in ("color", "alpha", "depth", "normal"):
        assert np.array_equal(o2[k].cpu().numpy(), gf[k]), k
    assert float(o2["loss_bg"].item()) == gf["loss_bg"] and np.array_equal(vis_f.cpu().numpy().view(np.uint32), gf["vis_count"])
    # masked L1 (S20) against the oracle's own maps
    ok = fw["fragile"] == 0
    diff = (fw["color"] - target.astype(np.float64)) * (m[None] > 0)
    l1_o = np.abs(diff).sum() / HW3
    assert abs(float(l1.item()) - l1_o) <= 1e-4 * max(1.0, l1_o)
    gC_o = np.sign(diff) / HW3
    gC_g = gC_t.cpu().numpy().astype(np.float64)
    clear = ok[None] & (np.abs(diff) > 2e-4)  # the sign of R - I is a decision: compared where it is clear on both sides
    assert np.array_equal(np.sign(gC_g)[clear], np.sign(gC_o)[clear])
    assert np.all(np.isin(np.round(np.abs(gC_g) * HW3, 3), (0.0, 1.0)))
    # (a) the whole step: GPU-made dL/dC -> GPU backward against oracle-made dL/dC -> oracle backward.  The few pixels whose sign
    # differs (|R - I| below fp32 resolution) and the fragile pixels move an entry by O(1/(3HW)) x w, far below the 1e-6 floor
    og = orc.render_bwd(*P, pre, srt, cam, cfg, mask=m, gC=gC_o.astype(np.float32))
    gg = {k: v.cpu().numpy() for k, v in grads.items()}
    rep = check_grads(gg, og, cond_rho=fw["cond_rho"])
    # (b) every entry of this step is O(pixels / (3HW)), mostly below north_star's floor, so the colour / alpha-only instance is
    # also run on the oracle's dL/dC (zero on fragile pixels, both sides the same input) and compared with the floor at 1e-9:
    # conditioning rule asserted, strict-rule misses reported
    gC_in = (gC_o * ok[None]).astype(np.float32)
    mm = np.where(ok, m, 1).astype(np.uint8)
    gg_b = g.render_bwd(gC=gC_in, mask=mm)
    og_b = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=gC_in)
    rep9 = check_grads(gg_b, og_b, floor=1e-9, max_strict_fail=1.0, cond_rho=fw["cond_rho"])
    return dict(l1_err=abs(float(l1.item()) - l1_o), sign_unclear=int((~clear).sum()),
                strict={k: (v["strict_fail_frac"], v["worst_strict_rel"]) for k, v in rep.items()},
                floor1e9={k: (v["strict_fail_frac"], v["worst_cond_units"]) for k, v in rep9.items()})


def test_config1_all_views():
    sc = sg.make_scene("config1")
    for v in range(4):
        full_parity(sc, v, dict(sh_degree=0))


def test_random_scenes_ragged_image_sh3_background():
    # 100x70: partial tiles on both axes; random orientations; coloured background
    for seed in (3, 4):
        sc = sg.random_scene(300, 100, 70, 80.0, seed=seed, sh_degree=3)
        full_parity(sc, 0, dict(sh_degree=3, bg=(0.3, 0.1, 0.2)))


def test_subpixel_surfels_filter_branch():
    sc = sg.random_scene(400, 64, 48, 40.0, seed=9, sh_degree=1, scale_lo=0.005, scale_hi=0.05)
    full_parity(sc, 0, dict(sh_degree=1))


def test_config2_shrunk_two_views():
    # config 2's geometry and distributions at 1/5 of the surfels: 1 900 tiles, several sort blocks, SH degree 3
    sc = sg.make_scene("config2", n_obj=20_000, n_bg=20_000)
    for v in (0, 7):
        r = full_parity(sc, v, dict(sh_degree=3))
        assert r["K"] > 4096 * 3


def test_long_tile_lists_take_the_heavy_walk():
    """Tiles whose lists exceed kFwdHeavyLen (raster_fwd.cu) take the several-survivors-per-iteration walk: thousands of large,
    nearly transparent surfels over a ragged 40x24 image, so that every pixel blends of the order of a thousand pairs."""
    sc = sg.random_scene(6000, 40, 24, 40.0, seed=21, sh_degree=1, scale_lo=0.2, scale_hi=0.5, op_mu=-4.0, op_sigma=0.5)
    r = full_parity(sc, 0, dict(sh_degree=1, bg=(0.1, 0.2, 0.3)), max_fragile=0.08)
    assert r["K"] > 6 * 2048
    # the same walk with the depth moments (kMoments instance)
    P, m = arrays(sc), sc.mask(0)
    orc, cam, cfg, pre, srt, fw = oracle_view(P, sc.cameras[0], dict(sh_degree=1), mask=m)
    g = GpuView(P, sc.cameras[0], dict(sh_degree=1))
    g.preprocess(); g.bin_sort(want_ids=False)
    gf = g.render_fwd(mask=m, moments=True)
    ok = fw["fragile"] == 0
    assert np.array_equal(gf["n_contrib"][ok], fw["n_contrib"][ok])
    for i, k in enumerate(("origin", "m1", "m2")):
        err = np.abs(gf["moments"][i] - fw[k]) / np.maximum(1.0, np.abs(fw[k]))
        assert (err * ok).max() <= IMG_TOL, (k, (err * ok).max())


def test_split_heavy_tile_backward_both_instances():
    """ONE 16x16 tile whose blended list (= the surfels with vis_count > 0, by the oracle) is longer than kBwdHeavyLen = 2048
    (raster_bwd.cu): the backward pass walks it with two CTAs, one pixel per thread.  Checked for both instances of the kernel:
    upstream gradients on all four maps, and on colour + alpha only (the masked-L1 + L_b step; depth / normal terms left out)."""
    sc = sg.random_scene(6000, 16, 16, 40.0, seed=33, sh_degree=0, scale_lo=0.2, scale_hi=0.5, op_mu=-4.5, op_sigma=0.5)
    P, m = arrays(sc), sc.mask(0)
    orc, cam, cfg, pre, srt, fw = oracle_view(P, sc.cameras[0], dict(sh_degree=0), mask=m)
    assert int((fw["vis_count"] > 0).sum()) > 2048
    g = GpuView(P, sc.cameras[0], dict(sh_degree=0))
    g.preprocess(); g.bin_sort(want_ids=False)
    gf = g.render_fwd(mask=m)
    ok = fw["fragile"] == 0
    print("PARITY split-tile scene: fragile fraction %.4f" % (1 - ok.mean()))
    assert 1 - ok.mean() <= 0.2  # thousands of nearly transparent surfels over one tile: measured 0.09
    assert np.array_equal(gf["n_contrib"][ok], fw["n_contrib"][ok])
    rng = np.random.default_rng(12)
    okf = ok.astype(np.float64)
    gC, gA = rng.normal(size=(3, 16, 16)) * okf, rng.normal(size=(16, 16)) * okf
    gD, gN = rng.normal(size=(16, 16)) * okf, rng.normal(size=(3, 16, 16)) * okf
    mm = np.where(ok, m, 1).astype(np.uint8)
    f32 = lambda a: a.astype(np.float32)
    gg = g.render_bwd(gC=gC, gA=gA, gD=gD, gN=gN, mask=mm)
    og = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=f32(gC), gA=f32(gA), gD=f32(gD), gN=f32(gN))
    check_grads(gg, og, cond_rho=fw["cond_rho"])
    gg = g.render_bwd(gC=gC, gA=gA, mask=mm)
    og = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=f32(gC), gA=f32(gA))
    check_grads(gg, og, cond_rho=fw["cond_rho"])
    never = gf["vis_count"] == 0
    for k in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
        assert np.all(gg[k][never] == 0.0), k


def test_segmented_heavy_tile_clusters_forward_backward_and_visibility_pass():
    """ONE 16x16 tile under 9 000 near-transparent surfels: its list is longer than kSegLen = 6144 (raster_fwd.cu) and its blended
    list longer than kBwdSegLen = 4096 (raster_bwd.cu), so the forward pass, the backward pass AND the statistics-only visibility
    pass all take the thread-block clusters (exact segmented compositing).  Everything against the oracle
    (full_parity), then the visibility pass against the forward pass: same pairs, same stop decisions, so vis_count is identical."""
    import torch
    from paper_2501_08174_b200 import binding as B
    sc = sg.random_scene(9000, 16, 16, 40.0, seed=41, sh_degree=0, scale_lo=0.2, scale_hi=0.5, op_mu=-5.0, op_sigma=0.5)
    r = full_parity(sc, 0, dict(sh_degree=0, bg=(0.2, 0.1, 0.3)), max_fragile=0.25, check_prune=True, label="one-tile-9000")
    L = r["ranges"][:, 1] - r["ranges"][:, 0]
    assert L.max() > 6144
    P, m = arrays(sc), sc.mask(0)
    g = GpuView(P, sc.cameras[0], dict(sh_degree=0))
    g.preprocess(); g.bin_sort(want_ids=False)
    gf = g.render_fwd(mask=m)
    assert int((gf["vis_count"] > 0).sum()) > 4096  # the blended list is long enough for the backward clusters
    vis_s = torch.zeros(g.n, dtype=torch.int32, device="cuda"); cs_s = torch.zeros(g.n, device="cuda")
    B.ocgs_visibility_pass(g.surfels, g.cam, g.cfg, g.ws, g.cap, vis_s, cs_s)
    torch.cuda.synchronize()
    assert np.array_equal(vis_s.cpu().numpy().view(np.uint32), gf["vis_count"])
    assert np.allclose(cs_s.cpu().numpy(), gf["contrib_sum"], rtol=1e-5, atol=1e-7)


def test_sh_degrees():
    sc = sg.random_scene(120, 48, 48, 40.0, seed=13, sh_degree=3)
    for deg in (0, 1, 2, 3):
        full_parity(sc, 0, dict(sh_degree=deg))


def test_depth_moments_and_their_gradient():
    """SURVEY.md 8(f) f-2 / reading R-moments: ocgs_render_fwd_reg's (origin, m1, m2) and ocgs_render_bwd_reg's upstream
    gradients of m1, m2, against the oracle; the other maps must be bit-identical to the plain forward."""
    for sc, cfg_kw in ((sg.random_scene(300, 100, 70, 80.0, seed=3, sh_degree=3), dict(sh_degree=3)),
                       (sg.make_scene("config2", n_obj=20_000, n_bg=20_000), dict(sh_degree=3))):
        P = arrays(sc)
        camn = sc.cameras[0]
        m = sc.mask(0)
        orc, cam, cfg, pre, srt, fw = oracle_view(P, camn, cfg_kw, mask=m)
        g = GpuView(P, camn, cfg_kw)
        g.preprocess(); g.bin_sort(want_ids=False)
        plain = g.render_fwd(mask=m)
        gf = g.render_fwd(mask=m, moments=True)
        for k in ("color", "alpha", "depth", "normal", "n_contrib"):
            assert np.array_equal(plain[k], gf[k]), k
        ok = fw["fragile"] == 0
        for i, k in enumerate(("origin", "m1", "m2")):
            err = np.abs(gf["moments"][i] - fw[k]) / np.maximum(1.0, np.abs(fw[k]))
            assert (err * ok).max() <= IMG_TOL, (k, (err * ok).max())
        rng = np.random.default_rng(17)
        H, W = camn.height, camn.width
        okf = ok.astype(np.float64)
        gC, gD, gM = rng.normal(size=(3, H, W)) * okf, rng.normal(size=(H, W)) * okf, rng.normal(size=(2, H, W)) * okf
        mm = np.where(ok, m, 1).astype(np.uint8)
        gg = g.render_bwd(gC=gC, gD=gD, gM=gM, mask=mm)
        og = orc.render_bwd(*P, pre, srt, cam, cfg, mask=mm, gC=gC.astype(np.float32), gD=gD.astype(np.float32),
                            gM1=gM[0].astype(np.float32), gM2=gM[1].astype(np.float32))
        # dz = z_i - z_first is a difference of fp32 depths (each good to ~3e-7 at z ~ 3): for thin surfaces the terms
        # proportional to dz carry that absolute noise, so the floor is 1e-4 of each array's typical (99th percentile) scale
        check_grads(gg, og, floor_frac=1e-4, cond_rho=fw["cond_rho"])


def test_empty_and_all_culled_and_capacity():
    import torch
    from paper_2501_08174_b200 import binding as B
    sc = sg.random_scene(50, 40, 40, 30.0, seed=2, sh_degree=0)
    camn = sc.cameras[0]
    # all culled: everything behind the camera
    P = list(arrays(sc))
    P[0] = sc.pos * np.array([1, 1, -1], np.float32)
    g = GpuView(tuple(P), camn, dict(sh_degree=0, bg=(0.5, 0.25, 0.125)))
    gp = g.preprocess()
    assert np.all(gp["tiles"] == 0)
    gs = g.bin_sort()
    assert gs["K"] == 0 and gs["n_vis"] == 0 and np.all(gs["ranges"] == 0)
    gf = g.render_fwd(mask=np.zeros((40, 40), np.uint8))
    assert np.all(gf["alpha"] == 0) and gf["loss_bg"] == 0.0 and np.all(gf["n_contrib"] == 0)
    assert np.allclose(gf["color"][0], 0.5) and np.allclose(gf["color"][2], 0.125)
    gg = g.render_bwd(gC=np.ones((3, 40, 40)))
    assert all(np.all(v == 0) for v in gg.values())
    # n = 0
    z = GpuView(tuple(a[:0] for a in arrays(sc)), camn, dict(sh_degree=0))
    z.preprocess()
    zs = z.bin_sort()
    assert zs["K"] == 0
    zf = z.render_fwd()
    assert np.all(zf["alpha"] == 0)
    # capacity overflow: flagged on the device, reported by ocgs_check, later calls stay safe
    small = GpuView(arrays(sc), camn, dict(sh_degree=0), key_capacity=8)
    small.preprocess()
    s2 = small.bin_sort()
    assert s2["error"] == 1 and s2["K"] > 8
    with pytest.raises(B.OcgsError) as e:
        B.ocgs_check(small.ws)
    assert e.value.code == B.OCGS_ERR_CAPACITY
    f2 = small.render_fwd()
    assert np.all(f2["alpha"] == 0)
    # unsupported / invalid arguments
    with pytest.raises(B.OcgsError):
        B.ocgs_preprocess(small.surfels, small.cam, B.ocgs_default_config(tile=8), small.ws, small.cap)
    with pytest.raises(B.OcgsError):
        B.ocgs_preprocess(small.surfels, small.cam, B.ocgs_default_config(sh_degree=4), small.ws, small.cap)
    torch.cuda.synchronize()


def test_more_than_8192_tiles():
    # order_tiles_kernel keeps the work of the first 8 x 1024 tiles in registers and loops over the rest: 2320x1040 = 145 x 65 = 9425
    # tiles (ragged on both axes), a sparse scene so that the oracle finishes in seconds; forward and backward launch orders both
    sc = sg.random_scene(500, 2320, 1040, 1500.0, seed=11, sh_degree=0, scale_lo=0.01, scale_hi=0.1)
    full_parity(sc, 0, dict(sh_degree=0))


def test_tile_ranges_key_counts_of_every_residue_mod_4():
    # tile_ranges_kernel reads four keys per thread with one 16-byte load and the ragged end key by key: K = 1 .. and every residue of
    # K mod 4, with a key capacity that is not a multiple of four either
    seen = set()
    for n, seed in [(1, 3), (2, 4), (3, 5), (5, 6), (9, 7), (14, 8), (23, 9), (37, 10)]:
        sc = sg.random_scene(n, 48, 40, 30.0, seed=seed, sh_degree=0)
        P, camn, kw = arrays(sc), sc.cameras[0], dict(sh_degree=0)
        orc, cam, cfg, pre, srt, fw = oracle_view(P, camn, kw, mask=sc.mask(0))
        for slack in (1, 2, 3):
            g = GpuView(P, camn, kw, key_capacity=max(srt["K"], 1) + slack)
            g.preprocess()
            gs = g.bin_sort()
            assert gs["error"] == 0 and gs["K"] == srt["K"]
            assert np.array_equal(gs["tile_keys"], (srt["keys"] >> np.uint64(32)).astype(np.uint32))
            assert np.array_equal(gs["ranges"], srt["ranges"])
        seen.add(srt["K"] % 4)
    assert seen == {0, 1, 2, 3}, seen


def test_masked_l1_and_host_step_match_device_path():
    import torch
    from paper_2501_08174_b200 import binding as B
    sc = sg.make_scene("config2", n_obj=4000, n_bg=4000, width=320, height=240, f=360.0)
    camn = sc.cameras[1]
    m = sc.mask(1)
    g = GpuView(arrays(sc), camn, dict(sh_degree=3))
    g.preprocess()
    gs_nvis = g.bin_sort()["n_vis"]
    gf = g.render_fwd(mask=m)
    rng = np.random.default_rng(0)
    target = rng.uniform(0, 1, (3, 240, 320)).astype(np.float32)
    tt = torch.tensor(target, device="cuda")
    gC = torch.empty_like(tt)
    loss = torch.zeros(1, device="cuda")
    B.ocgs_masked_l1(g.out["color"], tt, g.mask_t, 320, 240, gC, loss, g.ws, g.n, g.cap)
    d = (gf["color"].astype(np.float64) - target) * (m[None] > 0)
    assert abs(float(loss.item()) - np.abs(d).sum() / (3 * 240 * 320)) < 1e-6
    assert np.array_equal(gC.cpu().numpy(), (np.sign(d) / np.float32(3 * 240 * 320)).astype(np.float32))
    gg = g.render_bwd(gC=gC.cpu().numpy())
    # the fused forward (ocgs_render_fwd_l1) = forward + masked L1 without re-reading the colour map: maps and dL/dcolor
    # bit-identical, the L1 scalar equal to fp32 rounding (different summation order)
    o2 = B.alloc_outputs(320, 240)
    gC2 = torch.full_like(tt, 9.0); l1f = torch.zeros(1, device="cuda")
    vis_f = torch.zeros(g.n, dtype=torch.int32, device="cuda"); cs_f = torch.zeros(g.n, device="cuda")
    B.ocgs_render_fwd_l1(g.n, g.cam, g.cfg, g.ws, g.cap, g.mask_t, tt, o2["color"], o2["alpha"], o2["depth"], o2["normal"], o2["n_contrib"],
                         o2["loss_bg"], l1f, gC2, vis_f, cs_f)
    torch.cuda.synchronize()
    for k in ("color", "alpha", "depth", "normal"):
        assert np.array_equal(o2[k].cpu().numpy(), gf[k]), k
    assert np.array_equal(gC2.cpu().numpy(), gC.cpu().numpy()) and float(o2["loss_bg"].item()) == gf["loss_bg"]
    assert abs(float(l1f.item()) - float(loss.item())) < 1e-7
    assert np.array_equal(vis_f.cpu().numpy().view(np.uint32), gf["vis_count"])
    g.render_fwd(mask=m)  # restore the workspace state (blended lists) the checks below rely on
    # the same step through ocgs_step_host (host buffers, copies inside)
    n, H, W = g.n, 240, 320
    hp = [torch.tensor(np.ascontiguousarray(a, np.float32)).pin_memory() for a in arrays(sc)]
    h_grads = torch.empty(58 * n).pin_memory(); h_alpha = torch.empty(H * W).pin_memory(); h_loss = torch.empty(1).pin_memory()
    d_params = torch.empty(58 * n + 16, device="cuda"); d_grads = torch.empty(58 * n + 16, device="cuda")
    d_images = torch.empty(14 * H * W, device="cuda"); d_mask = torch.empty(H * W, dtype=torch.uint8, device="cuda")
    d_nc = torch.empty(H * W, dtype=torch.int32, device="cuda"); d_lb = torch.zeros(1, device="cuda")
    vis = torch.zeros(n, dtype=torch.int32, device="cuda"); cs = torch.zeros(n, device="cuda")
    B.ocgs_step_host(hp[0], hp[1], hp[2], hp[3], hp[4], n, g.cam, g.cfg, torch.tensor(m).pin_memory(), torch.tensor(target).pin_memory(),
                     h_grads, h_alpha, h_loss, d_params, d_mask, d_images, d_nc, d_grads, vis, cs, d_lb, g.ws, g.cap)
    assert np.array_equal(h_alpha.numpy().reshape(H, W), gf["alpha"])
    assert float(h_loss.item()) == gf["loss_bg"]
    hg = h_grads.numpy()
    # float atomics: run-to-run order differs, so compare to tolerance, not bits
    for name, lo, hi in (("d_pos", 0, 3 * n), ("d_scale", 3 * n, 5 * n), ("d_quat", 5 * n, 9 * n), ("d_opacity", 9 * n, 10 * n), ("d_sh", 10 * n, 58 * n)):
        a, b = hg[lo:hi], gg[name].ravel()
        assert np.allclose(a, b, rtol=2e-3, atol=1e-6 + 1e-4 * np.abs(b).max()), name
    assert np.array_equal(vis.cpu().numpy().view(np.uint32), gf["vis_count"])
    # the training step with resident parameters (ocgs_step_view_host): only the view's target and mask come from the host,
    # uploaded on a second stream; losses come back, gradients stay on the device
    grads = B.alloc_grads(n)
    h_losses = torch.zeros(2).pin_memory(); d_losses = torch.zeros(2, device="cuda")
    vis2 = torch.zeros(n, dtype=torch.int32, device="cuda"); cs2 = torch.zeros(n, device="cuda")
    for copy_stream in (None, torch.cuda.Stream()):
        vis2.zero_(); cs2.zero_()
        B.ocgs_step_view_host(g.surfels, g.cam, g.cfg, torch.tensor(m).pin_memory(), torch.tensor(target).pin_memory(), h_losses, d_mask,
                              d_images, d_nc, grads, vis2, cs2, d_losses, g.ws, g.cap, copy_stream=copy_stream)
        assert float(h_losses[0]) == gf["loss_bg"] and abs(float(h_losses[1]) - float(loss.item())) < 1e-7
        for name in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
            a, b = grads[name].cpu().numpy().ravel(), gg[name].ravel()
            assert np.allclose(a, b, rtol=2e-3, atol=1e-6 + 1e-4 * np.abs(b).max()), name
        assert np.array_equal(vis2.cpu().numpy().view(np.uint32), gf["vis_count"])
    # the same step enqueued without synchronisation and captured into a CUDA graph (ocgs_step_view_host_enqueue): every
    # replay uploads the view's data again, so changing the pinned target between replays must change the result
    h_mask, h_target = torch.tensor(m).pin_memory(), torch.tensor(target).pin_memory()
    h_header = torch.zeros(4, dtype=torch.int32).pin_memory()
    main, side = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=main):
        B.ocgs_step_view_host_enqueue(g.surfels, g.cam, g.cfg, h_mask, h_target, h_losses, h_header, d_mask, d_images, d_nc, grads, vis2,
                                      cs2, d_losses, g.ws, g.cap, stream=main, copy_stream=side)
    for rep in range(2):
        vis2.zero_(); cs2.zero_(); h_losses.zero_(); h_header.fill_(-1)
        for name in grads:
            grads[name].fill_(7.0)
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        assert int(h_header[3]) == 0 and int(h_header[2]) == gs_nvis
        assert float(h_losses[0]) == gf["loss_bg"]
        if rep == 0:
            assert abs(float(h_losses[1]) - float(loss.item())) < 1e-7
            for name in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
                a, b = grads[name].cpu().numpy().ravel(), gg[name].ravel()
                assert np.allclose(a, b, rtol=2e-3, atol=1e-6 + 1e-4 * np.abs(b).max()), name
            assert np.array_equal(vis2.cpu().numpy().view(np.uint32), gf["vis_count"])
            h_target.add_(0.25)  # the next replay must see the new host data
        else:
            assert float(h_losses[1]) > float(loss.item()) + 0.01
    # the prefetching form (ocgs_step_view_prefetch_enqueue): this view's inputs already resident, the NEXT view's uploaded
    # meanwhile on the copy stream; fused L1.  Step A prefetches (mask, target) into the second buffers, step B runs on them.
    h_target.copy_(torch.tensor(target))
    HW = H * W
    d_img11 = torch.empty(11 * HW, device="cuda")
    bufs = [(torch.tensor(m, device="cuda"), torch.tensor(target, device="cuda") + 0.5),      # view data of step A (shifted target)
            (torch.zeros(HW, dtype=torch.uint8, device="cuda"), torch.zeros(3 * HW, device="cuda"))]  # filled by A's prefetch
    for step_i, (cur, nxt, hm, ht) in enumerate(((0, 1, h_mask, h_target), (1, 0, None, None))):
        vis2.zero_(); cs2.zero_(); h_header.fill_(-1)
        B.ocgs_step_view_prefetch_enqueue(g.surfels, g.cam, g.cfg, hm, ht, h_losses, h_header, bufs[cur][0], bufs[cur][1],
                                          bufs[nxt][0] if hm is not None else None, bufs[nxt][1] if hm is not None else None,
                                          d_img11, d_nc, grads, vis2, cs2, d_losses, g.ws, g.cap, stream=main, copy_stream=side)
        main.synchronize()
        assert int(h_header[3]) == 0 and float(h_losses[0]) == gf["loss_bg"]
        if step_i == 0:
            assert float(h_losses[1]) > float(loss.item()) + 0.01   # ran on the shifted target
            side.synchronize()
            assert torch.equal(bufs[1][0].cpu(), h_mask.view(-1)) and torch.equal(bufs[1][1].cpu(), h_target.view(-1))
        else:
            assert abs(float(h_losses[1]) - float(loss.item())) < 1e-7
            for name in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh"):
                a, b = grads[name].cpu().numpy().ravel(), gg[name].ravel()
                assert np.allclose(a, b, rtol=2e-3, atol=1e-6 + 1e-4 * np.abs(b).max()), name
            assert np.array_equal(vis2.cpu().numpy().view(np.uint32), gf["vis_count"])
