"""-m gpu: the 3D-Gaussian variant of the visibility statistics (Appendix B) through
the C ABI against the oracle: ocgs3d_preprocess -> ocgs_bin_sort -> ocgs3d_render_fwd over several views, then
ocgs_prune_stats + ocgs_compact_rows.  Integers bit-exact, maps to 1e-4 on non-fragile pixels, statistics exact where no
fragile pixel is involved, prune mask / remap / compaction bit-exact."""
import numpy as np
import pytest

from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu


class Gpu3D:
    def __init__(self, P, cam_np, sh_degree, key_capacity=None):
        import torch
        from paper_2501_08174_b200 import binding as B
        self.torch, self.B = torch, B
        self.t = [torch.tensor(np.ascontiguousarray(a, np.float32), device="cuda") for a in P]
        self.n = int(P[0].shape[0])
        self.W, self.H = cam_np.width, cam_np.height
        self.cfg = B.ocgs_default_config(sh_degree=sh_degree)
        self.cap = int(key_capacity if key_capacity is not None else max(1 << 16, 64 * self.n))
        self.layout = B.ocgs_workspace_layout(self.n, self.W, self.H, self.cap)
        self.ws = B.alloc_workspace(self.n, self.W, self.H, self.cap)
        self.g = B.make_gaussians3d(*self.t)
        self.out = B.alloc_outputs(self.W, self.H)

    def sec(self, name, dtype, count):
        return self.B.ws_section(self.ws, self.layout, name, dtype, count).cpu().numpy()

    def view(self, cam_np, mask=None, vis=None, cs=None, want_ids=True):
        torch, B = self.torch, self.B
        cam = B.camera_from(cam_np)
        B.ocgs3d_preprocess(self.g, cam, self.cfg, self.ws, self.cap)
        n = self.n
        pre = dict(depth_bits=self.sec("depth_bits", torch.int32, n).view(np.uint32),
                   rect=self.sec("rect", torch.int16, 4 * n).view(np.uint16).reshape(n, 4).astype(np.int32),
                   tiles=self.sec("tiles", torch.int32, n).view(np.uint32), clamp=self.sec("clamp", torch.uint8, n),
                   rec=self.sec("rec_id", torch.float32, 24 * n).reshape(n, 24))
        ids = torch.zeros(self.cap, dtype=torch.int32, device="cuda") if want_ids else None
        B.ocgs_bin_sort(n, cam, self.cfg, self.ws, self.cap, ids)
        h = B.ocgs_check(self.ws)
        K = int(h.K)
        n_tiles = ((self.W + 15) // 16) * ((self.H + 15) // 16)
        srt = dict(K=K, n_vis=int(h.n_vis), ranges=self.sec("ranges", torch.int32, 2 * n_tiles).view(np.uint32).reshape(n_tiles, 2))
        if want_ids:
            srt["ids"] = ids[:K].cpu().numpy().view(np.uint32)
        mt = None if mask is None else torch.tensor(np.ascontiguousarray(mask, np.uint8), device="cuda")
        o = self.out
        B.ocgs3d_render_fwd(n, cam, self.cfg, self.ws, self.cap, mt, o["color"], o["alpha"], o["depth"], o["n_contrib"], o["loss_bg"], vis, cs)
        torch.cuda.synchronize()
        fw = {k: o[k].cpu().numpy() for k in ("color", "alpha", "depth", "n_contrib", "loss_bg")}
        fw["n_contrib"] = fw["n_contrib"].view(np.uint32)
        fw["loss_bg"] = float(fw["loss_bg"][0])
        return pre, srt, fw


def scales3(sc, ratio):
    return np.concatenate([sc.scale, ratio * sc.scale[:, :1]], 1).astype(np.float32)


def view_parity(g, P, camn, mask, vis_g, cs_g, vis_o, cs_o, touch, max_fragile=4e-3):
    import oracle as orc
    cam = orc.camera_from(camn)
    cfg = orc.default_config(sh_degree=int(g.cfg.sh_degree))
    pre = orc.preprocess3d(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    fw = orc.render3d_fwd(pre, srt, P[3], cam, cfg, mask=mask, vis_count=vis_o, contrib_sum=cs_o)
    touch += fw["fragile_touch"]
    gp, gs, gf = g.view(camn, mask=mask, vis=vis_g, cs=cs_g)
    v = pre["visible"] == 1
    assert np.array_equal(gp["tiles"], pre["tiles_touched"]) and np.array_equal(gp["depth_bits"], pre["depth_bits"])
    assert np.array_equal(gp["rect"][v], pre["rect"][v]) and np.array_equal(gp["clamp"][v], pre["clamp"][v])
    if v.any():
        rec = gp["rec"][v]
        assert np.array_equal(rec[:, 0:3], pre["conic"][v]) and np.array_equal(rec[:, 10:12], pre["c2d"][v])
        assert np.array_equal(rec[:, 12], pre["rho_cut"][v])
        assert np.abs(rec[:, 17:20] - pre["rgb"][v]).max() < 2e-5
    assert gs["K"] == srt["K"] and gs["n_vis"] == int(v.sum())
    assert np.array_equal(gs["ids"], srt["ids"]) and np.array_equal(gs["ranges"], srt["ranges"])
    ok = fw["fragile"] == 0
    assert 1.0 - ok.mean() <= max_fragile
    for k in ("color", "alpha", "depth"):
        scale = np.maximum(1.0, np.abs(fw[k])) if k == "depth" else 1.0
        err = np.abs(gf[k] - fw[k]) / scale
        assert (err * ok).max() <= 1e-4, (k, (err * ok).max())
        assert err.max() <= 0.05, (k, "fragile pixel beyond the discontinuity bound", err.max())
    assert np.array_equal(gf["n_contrib"][ok], fw["n_contrib"][ok])
    assert abs(gf["loss_bg"] - fw["loss_bg"]) <= 1e-4
    return srt["K"]


def run_scene(sc, s3, views, sh_degree, with_masks=True):
    import torch
    import oracle as orc
    from paper_2501_08174_b200 import binding as B
    P = (sc.pos, s3, sc.quat, sc.opacity, sc.sh)
    n = sc.n
    g = Gpu3D(P, sc.cameras[views[0]], sh_degree)
    vis_g = torch.zeros(n, dtype=torch.int32, device="cuda"); cs_g = torch.zeros(n, dtype=torch.float32, device="cuda")
    vis_o = np.zeros(n, np.uint32); cs_o = np.zeros(n, np.float64); touch = np.zeros(n, np.uint64)
    Ks = [view_parity(g, P, sc.cameras[v], sc.mask(v) if with_masks else None, vis_g, cs_g, vis_o, cs_o, touch) for v in views]
    # the statistics-only pass (ocgs3d_visibility_pass) counts exactly the same pairs as the forward pass
    vis_s = torch.zeros_like(vis_g); cs_s = torch.zeros_like(cs_g)
    for v in views:
        B.ocgs3d_visibility_pass(g.g, B.camera_from(sc.cameras[v]), g.cfg, g.ws, g.cap, vis_s, cs_s)
    assert torch.equal(vis_s, vis_g)
    assert np.allclose(cs_s.cpu().numpy(), cs_g.cpu().numpy(), rtol=1e-5, atol=1e-7)
    vg = vis_g.cpu().numpy().view(np.uint32)
    clean = touch == 0
    assert np.array_equal(vg[clean], vis_o[clean])
    assert np.all(np.abs(vg.astype(np.int64) - vis_o.astype(np.int64)) <= touch.astype(np.int64))
    assert np.allclose(cs_g.cpu().numpy()[clean], cs_o[clean], rtol=2e-4, atol=5e-6)
    # prune (PAPER.md:119 rule on the accumulated statistics) and compaction of every parameter array
    mask_t = torch.empty(n, dtype=torch.uint8, device="cuda"); remap_t = torch.empty(n, dtype=torch.int32, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int32, device="cuda")
    pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device="cuda")
    only_opacity = B.ocgs_surfels(None, None, None, B._ptr(g.t[3]), None, n)
    B.ocgs_prune_stats(only_opacity, vis_g, cs_g, g.cfg, mask_t, remap_t, None, n_out, 0, pws)
    torch.cuda.synchronize()
    po = orc.prune(vg, cs_g.cpu().numpy(), sc.opacity)
    pm = mask_t.cpu().numpy()
    assert np.array_equal(pm, po["prune_mask"]) and np.array_equal(remap_t.cpu().numpy(), po["remap"]) and int(n_out.item()) == po["n_out"]
    comp = orc.compact(dict(pos=sc.pos, scale=s3, quat=sc.quat, opacity=sc.opacity, sh=sc.sh), pm)
    for t, name, row in zip(g.t, ("pos", "scale", "quat", "opacity", "sh"), (3, 3, 4, 1, 48)):
        out = torch.full_like(t, -7.0)
        B.ocgs_compact_rows(t, remap_t, n, row, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.array_equal(got[: po["n_out"]], comp[name]), name
    return Ks, pm


def test_random_scenes_ragged_image():
    for seed in (3, 4):
        sc = sg.random_scene(300, 100, 70, 80.0, seed=seed, sh_degree=3)
        run_scene(sc, scales3(sc, 0.5), [0], 3)


def test_config1_all_views():
    sc = sg.make_scene("config1")
    run_scene(sc, scales3(sc, 0.2), [0, 1, 2, 3], 0)


def test_config4_geometry_occluded_interior_is_pruned():
    """The paper's Appendix-B experiment in miniature: Gaussians inside a near-opaque shell are never used in any view and go."""
    sc = sg.make_scene("config4", n_shell=6000, n_in=9000, n_bg=3000, res=256, f=325.0, n_views=12, scale_mul=6.5)
    Ks, pm = run_scene(sc, scales3(sc, 0.15), list(range(12)), 3, with_masks=False)
    assert pm[sc.group == 2].mean() > 0.9 and pm[sc.group == 0].mean() < 0.5


def test_config2_full_size_one_view():
    sc = sg.make_scene("config2")
    Ks, _ = run_scene(sc, scales3(sc, 0.3), [5], 3)
    assert Ks[0] > 100_000
