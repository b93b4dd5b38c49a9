"""-m gpu: (a) occlusion-aware pruning over many views (config 4's geometry), (b) parity at BASELINE.json's full size
(config 3: 1 M surfels, 1600x1200) in the launch configuration bench.py times, on every pixel of a view."""
import numpy as np
import pytest

from gpu_harness import GpuView
from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu


def arrays(sc):
    return (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)


def test_prune_stats_config4_shrunk_all_views():
    """accumulate visibility over all views, remove never-blended surfels, compact."""
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    sc = sg.make_scene("config4", n_shell=6000, n_in=9000, n_bg=3000, res=256, f=325.0, n_views=12, scale_mul=6.5)
    P = arrays(sc)
    n = sc.n
    cfg_kw = dict(sh_degree=3)
    vis_o = np.zeros(n, np.uint32); cs_o = np.zeros(n, np.float64); touch = np.zeros(n, np.uint64)
    g = GpuView(P, sc.cameras[0], cfg_kw)
    vis_g = torch.zeros(n, dtype=torch.int32, device="cuda"); cs_g = torch.zeros(n, dtype=torch.float32, device="cuda")
    ocfg = orc.default_config(sh_degree=3)
    for v in range(len(sc.cameras)):
        cam = orc.camera_from(sc.cameras[v])
        pre = orc.preprocess(*P, cam, ocfg)
        srt = orc.bin_sort(pre, cam, ocfg)
        fw = orc.render_fwd(pre, srt, sc.opacity, cam, ocfg, mask=None, vis_count=vis_o, contrib_sum=cs_o)
        touch += fw["fragile_touch"]
        g.cam = B.camera_from(sc.cameras[v])
        g.preprocess(); g.bin_sort(want_ids=False)
        g.render_fwd(mask=None, vis_count=vis_g, contrib_sum=cs_g, want_loss=False)
    vg = vis_g.cpu().numpy().view(np.uint32)
    clean = touch == 0
    assert np.array_equal(vg[clean], vis_o[clean])
    assert np.all(np.abs(vg.astype(np.int64) - vis_o.astype(np.int64)) <= touch.astype(np.int64))
    assert np.allclose(cs_g.cpu().numpy()[clean], cs_o[clean], rtol=2e-4, atol=5e-6)
    # prune + compact on the GPU
    mask_t = torch.empty(n, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(n, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    outs = [torch.full_like(t, -7.0) for t in (g.t["pos"], g.t["scale"], g.t["quat"], g.t["opacity"], g.t["sh"])]
    om = B.ocgs_surfels_mut(*[B._ptr(t) for t in outs], n)
    pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    B.ocgs_prune_stats(g.surfels, vis_g, cs_g, g.cfg, mask_t, remap_t, om, n_out, 0, pws)
    torch.cuda.synchronize()
    pm = mask_t.cpu().numpy()
    # bit-exact against the oracle's rule applied to the same statistics ...
    po = orc.prune(vg, cs_g.cpu().numpy(), sc.opacity)
    assert np.array_equal(pm, po["prune_mask"]) and np.array_equal(remap_t.cpu().numpy(), po["remap"]) and int(n_out.item()) == po["n_out"]
    # ... and against the oracle's own statistics wherever no fragile pixel was involved
    po2 = orc.prune(vis_o, cs_o.astype(np.float32), sc.opacity)
    assert np.array_equal(pm[clean], po2["prune_mask"][clean])
    assert (pm != po2["prune_mask"]).sum() <= 2
    comp = orc.compact(dict(pos=sc.pos, scale=sc.scale, quat=sc.quat, opacity=sc.opacity, sh=sc.sh), pm)
    k = po["n_out"]
    for t, name in zip(outs, ("pos", "scale", "quat", "opacity", "sh")):
        got = t.cpu().numpy()
        assert np.array_equal(got[:k], comp[name]), name
        assert np.all(got[k:] == -7.0), name  # nothing written past the survivors
    # the method's purpose: interior surfels (behind a near-opaque shell in every view) go, the visible shell stays
    interior, shell = sc.group == 2, sc.group == 0
    assert pm[interior].mean() > 0.97
    assert pm[shell].mean() < 0.35
    # tau / min_opacity extension and reset
    cfg2 = B.ocgs_default_config(sh_degree=3, tau_contrib=0.5, min_opacity=0.2)
    B.ocgs_prune_stats(g.surfels, vis_g, cs_g, cfg2, mask_t, remap_t, None, n_out, 1, pws)
    torch.cuda.synchronize()
    assert int(vis_g.abs().sum().item()) == 0 and float(cs_g.abs().sum().item()) == 0.0  # reset_stats


def test_prune_tau_and_min_opacity_rule():
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    rng = np.random.default_rng(1)
    n = 100_003  # not a multiple of the block size
    vis = rng.integers(0, 3, n).astype(np.uint32)
    cs = np.where(vis > 0, rng.uniform(0, 1, n), 0).astype(np.float32)
    sc = sg.random_scene(n, 32, 32, 30.0, seed=1, sh_degree=0)
    g = GpuView(arrays(sc), sc.cameras[0], dict(sh_degree=0), key_capacity=16)
    vt = torch.tensor(vis.view(np.int32), device="cuda"); ct = torch.tensor(cs, device="cuda")
    mask_t = torch.empty(n, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(n, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    for tau, omin in ((0.0, 0.0), (0.25, 0.1)):
        cfg = B.ocgs_default_config(sh_degree=0, tau_contrib=tau, min_opacity=omin)
        B.ocgs_prune_stats(g.surfels, vt, ct, cfg, mask_t, remap_t, None, n_out, 0, pws)
        torch.cuda.synchronize()
        po = orc.prune(vis, cs, sc.opacity, tau=tau, min_opacity=omin)
        assert np.array_equal(mask_t.cpu().numpy(), po["prune_mask"])
        assert np.array_equal(remap_t.cpu().numpy(), po["remap"]) and int(n_out.item()) == po["n_out"]


def test_posthoc_prune_driver_matches_the_oracle():
    """PAPER.md:234 (post-hoc variant): render every view with the statistics on, remove the never-blended surfels and
    carry a per-surfel side array (optimiser state) along; the driver in paper_2501_08174_b200.pruning only loops and
    marshals, so its result must equal the oracle's rule on the oracle's statistics."""
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B, pruning
    sc = sg.make_scene("config4", n_shell=3000, n_in=4000, n_bg=1500, res=192, f=245.0, n_views=8, scale_mul=8.0)
    P = arrays(sc)
    n = sc.n
    g = GpuView(P, sc.cameras[0], dict(sh_degree=3))
    out = B.alloc_outputs(g.W, g.H)
    vis = torch.zeros(n, dtype=torch.int32, device="cuda"); cs = torch.zeros(n, dtype=torch.float32, device="cuda")
    pruning.accumulate_visibility(g.surfels, n, sc.cameras, g.cfg, g.ws, g.cap, out, vis, cs)
    # the statistics-only pass (ocgs_visibility_pass: no SH colour, no maps, no blended lists) counts exactly the same pairs
    vis_s = torch.zeros_like(vis); cs_s = torch.zeros_like(cs)
    pruning.accumulate_visibility(g.surfels, n, sc.cameras, g.cfg, g.ws, g.cap, None, vis_s, cs_s)
    assert torch.equal(vis_s, vis) and int(vis.sum().item()) > 10_000
    assert np.allclose(cs_s.cpu().numpy(), cs.cpu().numpy(), rtol=1e-5, atol=1e-7)
    # ... also with two views in flight on two streams and two workspaces
    vis_s.zero_(); cs_s.zero_()
    ws2 = B.alloc_workspace(n, g.W, g.H, g.cap)
    pruning.accumulate_visibility(g.surfels, n, sc.cameras, g.cfg, g.ws, g.cap, None, vis_s, cs_s, ws2=ws2)
    torch.cuda.synchronize()
    assert torch.equal(vis_s, vis)
    assert np.allclose(cs_s.cpu().numpy(), cs.cpu().numpy(), rtol=1e-5, atol=1e-7)
    # a key capacity that only the first views exceed is still reported (the driver keeps every view's header)
    cams_mixed = list(sc.cameras[:2]) + [sc.cameras[0]] * 2
    small = B.alloc_workspace(n, g.W, g.H, 64)
    with pytest.raises(B.OcgsError) as e:
        pruning.accumulate_visibility(g.surfels, n, cams_mixed, g.cfg, small, 64, None, torch.zeros_like(vis), torch.zeros_like(cs))
    assert e.value.code == B.OCGS_ERR_CAPACITY and "key_capacity >=" in str(e.value)
    vis_o = np.zeros(n, np.uint32); cs_o = np.zeros(n, np.float64); touch = np.zeros(n, np.uint64)
    ocfg = orc.default_config(sh_degree=3)
    for camn in sc.cameras:
        cam = orc.camera_from(camn)
        pre = orc.preprocess(*P, cam, ocfg); srt = orc.bin_sort(pre, cam, ocfg)
        fw = orc.render_fwd(pre, srt, sc.opacity, cam, ocfg, mask=None, vis_count=vis_o, contrib_sum=cs_o)
        touch += fw["fragile_touch"]
    clean = touch == 0
    assert np.array_equal(vis.cpu().numpy().view(np.uint32)[clean], vis_o[clean])
    state = torch.tensor(np.random.default_rng(0).normal(size=(n, 58)).astype(np.float32), device="cuda")
    vg = vis.cpu().numpy().view(np.uint32).copy(); cg = cs.cpu().numpy().copy()
    params, extras, kept, mask, remap = pruning.prune(g.surfels, g.t, n, g.cfg, vis, cs, reset_stats=True, extra_rows=dict(adam_m=state))
    po = orc.prune(vg, cg, sc.opacity)
    assert kept == po["n_out"] and np.array_equal(mask.cpu().numpy(), po["prune_mask"]) and np.array_equal(remap.cpu().numpy(), po["remap"])
    comp = orc.compact(dict(pos=sc.pos, scale=sc.scale, quat=sc.quat, opacity=sc.opacity, sh=sc.sh, adam_m=state.cpu().numpy()), po["prune_mask"])
    for k in ("pos", "scale", "quat", "opacity", "sh"):
        assert np.array_equal(params[k].cpu().numpy(), comp[k]), k
    assert np.array_equal(extras["adam_m"].cpu().numpy(), comp["adam_m"])
    assert int(vis.abs().sum().item()) == 0  # reset for the next interval
    assert po["prune_mask"][sc.group == 2].mean() > 0.7  # most of the occluded interior goes (3 000 shell surfels leave gaps)


def test_compact_rows_follows_the_remap():
    """Optimiser state follows the parameters through a prune: by definition
    out = [row for row, pruned in zip(in, mask) if not pruned]."""
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    rng = np.random.default_rng(4)
    n = 70_001
    pm = (rng.uniform(size=n) < 0.4).astype(np.uint8)
    remap = np.where(pm == 0, np.cumsum(pm == 0) - 1, -1).astype(np.int32)
    for row in (1, 3, 48, 58):
        x = rng.normal(size=(n, row)).astype(np.float32)
        xt, rt = torch.tensor(x, device="cuda"), torch.tensor(remap, device="cuda")
        out = torch.full((n, row), -7.0, dtype=torch.float32, device="cuda")
        B.ocgs_compact_rows(xt, rt, n, row, out)
        torch.cuda.synchronize()
        ref = orc.compact(dict(x=x), pm)["x"]
        got = out.cpu().numpy()
        assert np.array_equal(got[: len(ref)], ref) and np.all(got[len(ref):] == -7.0)
    with pytest.raises(B.OcgsError):
        B.ocgs_compact_rows(xt, rt, n, 0, out)


def test_config3_full_size_full_image():
    """BASELINE.json configs[2] (the config the metric is quoted on) at full size, in bench.py's launch configuration, EVERY
    pixel and every surfel of one view: integers, the four maps, n_contrib, L_b, vis_count / contrib_sum, all six gradient
    arrays for both backward instances, the prune mask + compaction from the view's statistics, and the step bench.py times
    (ocgs_render_fwd_l1 + the colour / alpha-only backward instance)."""
    from test_gpu_parity import full_parity
    sc = sg.make_scene("config3")
    r = full_parity(sc, 0, dict(sh_degree=3), key_capacity=48 * sc.n, max_fragile=2e-2, check_prune=True, bench_step=True, label="config3")
    assert r["K"] > 4_000_000
