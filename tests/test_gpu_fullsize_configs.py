"""-m gpu: parity at BASELINE.json's FULL sizes for configs 2, 4 and 5 (config 3 is in test_gpu_prune_and_fullsize.py),
in the launch configuration bench.py uses.  Integer outputs (tiles, rects, depth bits, order, ranges) are compared in
full; images and gradients in full where the oracle finishes in seconds (config 2) and on sampled windows otherwise
(config 5); config 4 accumulates the visibility statistics over all 64 views, prunes and compacts."""
import numpy as np
import pytest

from gpu_harness import GpuView, check_grads
from paper_2501_08174_b200 import scenegen as sg
from test_gpu_parity import arrays, full_parity

pytestmark = pytest.mark.gpu


def test_config2_full_size_full_image():
    """200 k surfels, 800x600 (DTU's training resolution), SH degree 3: every pixel, every gradient."""
    sc = sg.make_scene("config2")
    r = full_parity(sc, 3, dict(sh_degree=3), max_fragile=3e-3)  # measured 1.06e-3
    assert r["K"] > 100_000


def windows_parity(sc, view, windows, key_capacity, rng_seed=11):
    """Integer outputs in full; forward maps and gradients on `windows` (x0, y0, x1, y1), upstream gradients non-zero
    only inside them so that the oracle walks only those pixels."""
    import oracle as orc
    P = arrays(sc)
    camn = sc.cameras[view]
    m = sc.mask(view)
    cam = orc.camera_from(camn)
    cfg = orc.default_config(sh_degree=sc.sh_degree)
    pre = orc.preprocess(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    g = GpuView(P, camn, dict(sh_degree=sc.sh_degree), key_capacity=key_capacity)
    gp = g.preprocess()
    vis = pre["visible"] == 1
    assert np.array_equal(gp["tiles"], pre["tiles_touched"]) and np.array_equal(gp["depth_bits"], pre["depth_bits"])
    assert np.array_equal(gp["rect"][vis], pre["rect"][vis]) and np.array_equal(gp["clamp"][vis], pre["clamp"][vis])
    gs = g.bin_sort()
    assert gs["error"] == 0 and gs["K"] == srt["K"] and gs["n_vis"] == int(vis.sum())
    assert np.array_equal(gs["ids"], srt["ids"]) and np.array_equal(gs["ranges"], srt["ranges"])
    gf = g.render_fwd(mask=m)
    H, W = camn.height, camn.width
    gC = np.zeros((3, H, W)); gA = np.zeros((H, W)); gD = np.zeros((H, W)); gN = np.zeros((3, H, W))
    rng = np.random.default_rng(rng_seed)
    frag_total = npix = 0
    cond_rho = np.zeros(sc.n)
    for (x0, y0, x1, y1) in windows:
        fw = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=m, window=(x0, y0, x1, y1))
        cond_rho = np.maximum(cond_rho, fw["cond_rho"])
        ok = fw["fragile"][y0:y1, x0:x1] == 0
        frag_total += int((~ok).sum()); npix += ok.size
        for k in ("color", "alpha", "depth", "normal"):
            a, b = gf[k][..., y0:y1, x0:x1], fw[k][..., y0:y1, x0:x1]
            scale = np.maximum(1.0, np.abs(b)) if k == "depth" else 1.0
            err = np.abs(a - b) / scale
            assert (err * ok).max() <= 1e-4, (k, (x0, y0), (err * ok).max())
            assert err.max() <= 0.02, (k, (x0, y0), "fragile pixel beyond the discontinuity bound")
        assert np.array_equal(gf["n_contrib"][y0:y1, x0:x1][ok], fw["n_contrib"][y0:y1, x0:x1][ok])
        okf = ok.astype(np.float64)
        gC[:, y0:y1, x0:x1] = rng.normal(size=(3, y1 - y0, x1 - x0)) * okf
        gA[y0:y1, x0:x1] = rng.normal(size=ok.shape) * okf
        gD[y0:y1, x0:x1] = rng.normal(size=ok.shape) * okf
        gN[:, y0:y1, x0:x1] = rng.normal(size=(3, y1 - y0, x1 - x0)) * okf
    assert frag_total <= 0.01 * npix
    cfg0 = orc.default_config(sh_degree=sc.sh_degree, gamma_bg=0.0)
    g.cfg.gamma_bg = 0.0
    gg = g.render_bwd(gC=gC, gA=gA, gD=gD, gN=gN, mask=m)
    og = {k: np.zeros_like(v, dtype=np.float64) for k, v in gg.items()}
    og["_abs"] = {k: np.zeros_like(v, dtype=np.float64) for k, v in gg.items()}
    for w in windows:  # gradients and their sums of |terms| are additive over disjoint sets of pixels
        part = orc.render_bwd(*P, pre, srt, cam, cfg0, mask=m, gC=gC.astype(np.float32), gA=gA.astype(np.float32),
                              gD=gD.astype(np.float32), gN=gN.astype(np.float32), window=w)
        for k in gg:
            og[k] += part[k]
            og["_abs"][k] += part["_abs"][k].reshape(og["_abs"][k].shape)
    rep = check_grads(gg, og, cond_rho=cond_rho)
    return dict(K=srt["K"], n_vis=int(vis.sum()), grads=rep, ranges=srt["ranges"])


def test_config5_full_size_full_image():
    """4 M surfels, 1920x1080: 1080 = 67.5 x 16, so the last tile row is half empty (ragged tail), tile lists of thousands of
    entries (many batches per tile), 4.3 M keys through both radix stages.  Every pixel of a view, every output (see
    full_parity), the prune mask from its statistics and the step bench.py times."""
    sc = sg.make_scene("config5")
    r = full_parity(sc, 0, dict(sh_degree=3), key_capacity=16 * sc.n, max_fragile=2.7e-3, check_prune=True, bench_step=True, label="config5")  # measured 9.2e-4
    L = r["ranges"][:, 1] - r["ranges"][:, 0]
    assert r["K"] > 2_000_000 and L.max() > 4096


def test_config5_heaviest_view_forward_and_colour_backward():
    """The view of config 5 with the longest tile list (view 7: one tile of 25 338 entries, the heavy-tile walk of both raster
    kernels): every pixel of the forward outputs and the colour / alpha-only backward instance."""
    sc = sg.make_scene("config5")
    r = full_parity(sc, 7, dict(sh_degree=3), key_capacity=16 * sc.n, max_fragile=2.4e-3, label="config5-heaviest")  # measured 7.7e-4
    L = r["ranges"][:, 1] - r["ranges"][:, 0]
    assert L.max() > 20_000
    # the statistics-only pass takes the same clusters: identical counts
    import torch
    from paper_2501_08174_b200 import binding as B
    g = GpuView(arrays(sc), sc.cameras[7], dict(sh_degree=3), key_capacity=16 * sc.n)
    g.preprocess(); g.bin_sort(want_ids=False)
    gf = g.render_fwd(mask=None, want_loss=False)
    vis_s = torch.zeros(g.n, dtype=torch.int32, device="cuda"); cs_s = torch.zeros(g.n, device="cuda")
    B.ocgs_visibility_pass(g.surfels, g.cam, g.cfg, g.ws, g.cap, vis_s, cs_s)
    torch.cuda.synchronize()
    assert np.array_equal(vis_s.cpu().numpy().view(np.uint32), gf["vis_count"])
    assert np.allclose(cs_s.cpu().numpy(), gf["contrib_sum"], rtol=1e-5, atol=1e-7)


def test_config4_full_size_all_views_prune():
    """800 k surfels (250 k near-opaque shell, 400 k interior, 150 k background), 64 views at 1024x1024: per-surfel
    statistics over all views, then the prune mask and the compaction, bit-exact against the oracle's rule; the mask
    must remove the interior and keep the shell (BASELINE.json configs[3])."""
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    sc = sg.make_scene("config4")
    P = arrays(sc)
    n = sc.n
    vis_o = np.zeros(n, np.uint32); cs_o = np.zeros(n, np.float64); touch = np.zeros(n, np.uint64)
    g = GpuView(P, sc.cameras[0], dict(sh_degree=3), key_capacity=24 * n)
    vis_g = torch.zeros(n, dtype=torch.int32, device="cuda"); cs_g = torch.zeros(n, dtype=torch.float32, device="cuda")
    vis_s = torch.zeros_like(vis_g); cs_s = torch.zeros_like(cs_g)  # the same statistics through ocgs_visibility_pass
    ocfg = orc.default_config(sh_degree=3)
    for v in range(len(sc.cameras)):
        cam = orc.camera_from(sc.cameras[v])
        pre = orc.preprocess(*P, cam, ocfg)
        srt = orc.bin_sort(pre, cam, ocfg)
        fw = orc.render_fwd(pre, srt, sc.opacity, cam, ocfg, mask=None, vis_count=vis_o, contrib_sum=cs_o)
        touch += fw["fragile_touch"]
        g.cam = B.camera_from(sc.cameras[v])
        g.preprocess()
        gs = g.bin_sort(want_ids=(v % 16 == 0))
        assert gs["K"] == srt["K"] and np.array_equal(gs["ranges"], srt["ranges"])
        if "ids" in gs:
            assert np.array_equal(gs["ids"], srt["ids"])
        gf = g.render_fwd(mask=None, vis_count=vis_g, contrib_sum=cs_g, want_loss=False)
        if v % 16 == 0:
            ok = fw["fragile"] == 0
            assert (np.abs(gf["alpha"] - fw["alpha"]) * ok).max() <= 1e-4
            assert (np.abs(gf["color"] - fw["color"]) * ok).max() <= 1e-4
        B.ocgs_visibility_pass(g.surfels, g.cam, g.cfg, g.ws, g.cap, vis_s, cs_s)
    assert torch.equal(vis_s, vis_g)
    assert np.allclose(cs_s.cpu().numpy(), cs_g.cpu().numpy(), rtol=1e-5, atol=1e-7)
    vg = vis_g.cpu().numpy().view(np.uint32)
    clean = touch == 0
    assert np.array_equal(vg[clean], vis_o[clean])
    assert np.all(np.abs(vg.astype(np.int64) - vis_o.astype(np.int64)) <= touch.astype(np.int64))
    assert np.allclose(cs_g.cpu().numpy()[clean], cs_o[clean], rtol=2e-4, atol=5e-6)
    mask_t = torch.empty(n, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(n, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    outs = [torch.full_like(t, -7.0) for t in (g.t["pos"], g.t["scale"], g.t["quat"], g.t["opacity"], g.t["sh"])]
    om = B.ocgs_surfels_mut(*[B._ptr(t) for t in outs], n)
    pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    B.ocgs_prune_stats(g.surfels, vis_g, cs_g, g.cfg, mask_t, remap_t, om, n_out, 0, pws)
    torch.cuda.synchronize()
    pm = mask_t.cpu().numpy()
    po = orc.prune(vg, cs_g.cpu().numpy(), sc.opacity)
    assert np.array_equal(pm, po["prune_mask"]) and np.array_equal(remap_t.cpu().numpy(), po["remap"]) and int(n_out.item()) == po["n_out"]
    po2 = orc.prune(vis_o, cs_o.astype(np.float32), sc.opacity)
    assert np.array_equal(pm[clean], po2["prune_mask"][clean])
    # surfels whose only blends fell on fragile pixels may legitimately differ (S22); there must be almost none
    n_diff = int((pm != po2["prune_mask"]).sum())
    print("PARITY config4: prune mask differs from the mask of the oracle's own statistics on %d of %d surfels; %d surfels touch a fragile pixel in some view"
          % (n_diff, n, int((~clean).sum())))
    assert n_diff <= 2  # measured: 0
    comp = orc.compact(dict(pos=sc.pos, scale=sc.scale, quat=sc.quat, opacity=sc.opacity, sh=sc.sh), pm)
    k = po["n_out"]
    for t, name in zip(outs, ("pos", "scale", "quat", "opacity", "sh")):
        got = t.cpu().numpy()
        assert np.array_equal(got[:k], comp[name]), name
        assert np.all(got[k:] == -7.0), name
    interior, shell = sc.group == 2, sc.group == 0
    print("config4: pruned interior %.4f, shell %.4f, background %.4f, kept %d of %d" %
          (pm[interior].mean(), pm[shell].mean(), pm[sc.group == 1].mean(), k, n))
    assert pm[interior].mean() > 0.97
    assert pm[shell].mean() < 0.5


def test_more_than_2_pow_24_keys():
    """Config 3's geometry with four times its surfels (4 M; one view): 19 M (tile, surfel) keys -- more than 2^24, so that no
    index anywhere on the path can hide in 24 bits or in an fp32 mantissa -- and mean tile lists of ~2 500 entries, so that
    most tiles take the long-list walk of the forward kernel.  Integer outputs in full, maps and gradients on three windows."""
    sc = sg.make_scene("config3", n_obj=1_200_000, n_bg=2_800_000, n_views=2)
    W, H = 1600, 1200
    windows = [(776, 576, 808, 608), (0, 0, 32, 32), (W - 32, H - 32, W, H)]
    r = windows_parity(sc, 1, windows, key_capacity=12 * sc.n)
    L = r["ranges"][:, 1] - r["ranges"][:, 0]
    assert r["K"] > (1 << 24) and np.median(L) > 2048


def test_more_than_2_pow_17_tiles_three_tile_sort_passes():
    """8192 x 4112 pixels = 512 x 257 = 131 584 tiles: tile ids need 18 bits, so the tile sort takes three radix passes (an odd
    number: the result is copied back from the alternate buffers) and its histograms come from radix_hist_all_kernel instead
    of emit_keys_kernel's two; pixel coordinates up to 8191 in the packed rects.  Integers in full, maps on windows."""
    W, H = 8192, 4112
    sc = sg.random_scene(60_000, W, H, 6000.0, seed=31, sh_degree=1, scale_lo=0.003, scale_hi=0.03)
    windows = [(0, 0, 32, 32), (W - 32, H - 32, W, H), (4080, 2040, 4112, 2072), (W - 40, 0, W, 24)]
    r = windows_parity(sc, 0, windows, key_capacity=12_000_000)
    assert r["ranges"].shape[0] == 512 * 257 and r["K"] > 5_000_000
