"""Shared helpers of the -m gpu parity tests: run one view through the C ABI (via the thin binding) and through the oracle
on the same seeded inputs.  No arithmetic of the method lives here."""
from __future__ import annotations

import numpy as np


def gpu_modules():
    import torch
    from paper_2501_08174_b200 import binding as B
    return torch, B


class GpuView:
    """preprocess -> bin_sort -> render_fwd (-> render_bwd) of one view through the C ABI."""

    def __init__(self, scene_arrays, cam_np, cfg_kw, key_capacity=None, ws=None):
        torch, B = gpu_modules()
        self.torch, self.B = torch, B
        pos, scale, quat, opacity, sh = scene_arrays
        dev = "cuda"
        self.t = dict(pos=torch.tensor(np.ascontiguousarray(pos, np.float32), device=dev),
                      scale=torch.tensor(np.ascontiguousarray(scale, np.float32), device=dev),
                      quat=torch.tensor(np.ascontiguousarray(quat, np.float32), device=dev),
                      opacity=torch.tensor(np.ascontiguousarray(opacity, np.float32), device=dev),
                      sh=torch.tensor(np.ascontiguousarray(sh, np.float32), device=dev))
        self.n = int(pos.shape[0])
        self.cam = B.camera_from(cam_np)
        self.W, self.H = cam_np.width, cam_np.height
        self.cfg = B.ocgs_default_config(**cfg_kw)
        self.cap = int(key_capacity if key_capacity is not None else max(1 << 16, 64 * self.n))
        self.layout = B.ocgs_workspace_layout(self.n, self.W, self.H, self.cap)
        self.ws = ws if ws is not None else B.alloc_workspace(self.n, self.W, self.H, self.cap)
        self.surfels = B.make_surfels(self.t["pos"], self.t["scale"], self.t["quat"], self.t["opacity"], self.t["sh"])
        self.out = None
        self.mask_t = None

    def sec(self, name, dtype, count):
        return self.B.ws_section(self.ws, self.layout, name, dtype, count).cpu().numpy()

    def preprocess(self):
        self.B.ocgs_preprocess(self.surfels, self.cam, self.cfg, self.ws, self.cap)
        torch = self.torch
        n = self.n
        return dict(depth_bits=self.sec("depth_bits", torch.int32, n).view(np.uint32),
                    rect=self.sec("rect", torch.int16, 4 * n).view(np.uint16).reshape(n, 4).astype(np.int32),
                    tiles=self.sec("tiles", torch.int32, n).view(np.uint32), clamp=self.sec("clamp", torch.uint8, n),
                    rec_id=self.sec("rec_id", torch.float32, 24 * n).reshape(n, 24))

    def bin_sort(self, want_ids=True):
        torch = self.torch
        ids = torch.zeros(self.cap, dtype=torch.int32, device="cuda") if want_ids else None
        self.B.ocgs_bin_sort(self.n, self.cam, self.cfg, self.ws, self.cap, ids)
        h = self.B.ocgs_check(self.ws, raise_on_error=False)
        K = int(h.K)
        n_tiles = ((self.W + 15) // 16) * ((self.H + 15) // 16)
        res = dict(K=K, n_vis=int(h.n_vis), error=int(h.error),
                   ranges=self.sec("ranges", torch.int32, 2 * n_tiles).view(np.uint32).reshape(n_tiles, 2))
        if want_ids and not h.error:
            res["ids"] = ids[:K].cpu().numpy().view(np.uint32)
            res["tile_keys"] = self.sec("tile_keys", torch.int32, max(K, 1)).view(np.uint32)[:K]
        return res

    def render_fwd(self, mask=None, stats=True, vis_count=None, contrib_sum=None, want_loss=True, moments=False):
        torch, B = self.torch, self.B
        self.out = B.alloc_outputs(self.W, self.H)
        self.mask_t = None if mask is None else torch.tensor(np.ascontiguousarray(mask, np.uint8), device="cuda")
        if stats:
            self.vis = vis_count if vis_count is not None else torch.zeros(self.n, dtype=torch.int32, device="cuda")
            self.cs = contrib_sum if contrib_sum is not None else torch.zeros(self.n, dtype=torch.float32, device="cuda")
        else:
            self.vis = self.cs = None
        o = self.out
        if moments:  # forward with the depth moments (origin, m1, m2)
            o["moments"] = torch.zeros((3, self.H, self.W), dtype=torch.float32, device="cuda")
            B.ocgs_render_fwd_reg(self.n, self.cam, self.cfg, self.ws, self.cap, self.mask_t, o["color"], o["alpha"], o["depth"], o["normal"],
                                  o["n_contrib"], o["loss_bg"] if want_loss else None, self.vis, self.cs, o["moments"])
        else:
            B.ocgs_render_fwd(self.n, self.cam, self.cfg, self.ws, self.cap, self.mask_t, o["color"], o["alpha"], o["depth"], o["normal"],
                              o["n_contrib"], o["loss_bg"] if want_loss else None, self.vis, self.cs)
        torch.cuda.synchronize()
        res = {k: v.cpu().numpy() for k, v in o.items()}
        res["n_contrib"] = res["n_contrib"].view(np.uint32)
        res["loss_bg"] = float(res["loss_bg"][0])
        if stats:
            res["vis_count"] = self.vis.cpu().numpy().view(np.uint32)
            res["contrib_sum"] = self.cs.cpu().numpy()
        return res

    def render_bwd(self, gC=None, gA=None, gD=None, gN=None, mask="same", gM=None):
        torch, B = self.torch, self.B
        g = B.alloc_grads(self.n)
        for v in g.values():  # every row must be WRITTEN by the call (culled surfels: zeros), not found clean
            v.fill_(float("nan"))

        def dev(a):
            return None if a is None else torch.tensor(np.ascontiguousarray(a, np.float32), device="cuda")
        m = self.mask_t if isinstance(mask, str) else (None if mask is None else torch.tensor(np.ascontiguousarray(mask, np.uint8), device="cuda"))
        if gM is not None:  # [2,H,W]: upstream of m1, m2; the origin map is the forward's
            B.ocgs_render_bwd_reg(self.surfels, self.cam, self.cfg, self.ws, self.cap, m, self.out["n_contrib"], dev(gC), dev(gA), dev(gD),
                                  dev(gN), self.out["moments"], dev(gM), g["d_pos"], g["d_scale"], g["d_quat"], g["d_opacity"], g["d_sh"], g["d_center2d"])
        else:
            B.ocgs_render_bwd(self.surfels, self.cam, self.cfg, self.ws, self.cap, m, self.out["n_contrib"], dev(gC), dev(gA), dev(gD), dev(gN),
                              g["d_pos"], g["d_scale"], g["d_quat"], g["d_opacity"], g["d_sh"], g["d_center2d"])
        torch.cuda.synchronize()
        return {k: v.cpu().numpy() for k, v in g.items()}


def oracle_view(scene_arrays, cam_np, cfg_kw, mask=None):
    import oracle as orc
    kw = dict(cfg_kw)
    cfg = orc.default_config(sh_degree=kw.pop("sh_degree", 3), bg=kw.pop("bg", (0.0, 0.0, 0.0)), gamma_bg=kw.pop("gamma_bg", 0.5), **kw)
    cam = orc.camera_from(cam_np)
    pre, srt, fwd = orc.forward_view(*scene_arrays, cam, cfg, mask=mask)
    return orc, cam, cfg, pre, srt, fwd


GROUPS = ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh", "d_center2d")


def check_grads(gpu, ora, rel=1e-3, floor=1e-6, sum_eps=1e-5, floor_frac=None, max_strict_fail=1e-3, cond_rho=None):
    """Gradient parity rule (north_star: relative error 1e-3 on entries above 1e-6).

    STRICT rule, per entry: |gpu - oracle| <= rel*|oracle| + floor.  The number of entries of each array that miss it is
    ASSERTED to be at most max(3, max_strict_fail x size) (1e-3 of the entries; measured: 5e-5 at configs 3 and 5), and every
    entry that misses it must be explained by the fp32 arithmetic it comes from, in one of two ways:
    (a) cancellation: the kernel accumulates the record gradients in its own basis (P, Q, R of the centred homography) and maps
        them to the parameters afterwards, so an entry that is small beside the other entries of its surfel's block inherits
        their rounding error: |err| <= rel x max|oracle| over the block (d_pos and d_scale, both per world length and made from
        the same homography gradient, form ONE block: the scale gradient of a sub-pixel-thin surfel is a single well-conditioned
        term -2 v^2 g_rho / s_v that the homography basis reaches only as a difference of large ones; d_opacity: sum_eps x the
        sum of |terms|);
    (b) ill-conditioned pair evaluation: |err| <= (sum_eps + 16 cond_rho[j]) x (sum of the |terms| of that entry, reported by the
        oracle as ora["_abs"]), cond_rho[j] (oracle forward, per surfel) being the first-order fp32 error estimate of rho
        over the surfel's blended pairs -- for the few surfels seen almost edge-on (q_z cancels)
        every term carries that relative error (x16: a gradient term is a derivative of the value the estimate is made for; the largest ratio measured at configs 3 and 5 is 9); sum_eps = 1e-5 = 84 units of fp32 roundoff covers the summation itself.
    Returns, per array: entries, number and fraction missing the strict rule, the worst strict relative error
    (|err| / (|oracle| + floor/rel)) and the worst error in units of sum|terms|; raises AssertionError naming the first failing
    entry.  floor_frac (optional): the absolute floor of each array is raised to floor_frac x the 99th percentile of its
    per-surfel block scales (for upstream gradients whose per-pair terms are differences of nearly equal fp32 depths: their
    absolute noise is set by the depth, not by the entry)."""
    report = {}
    floor0 = floor
    for k in GROUPS:
        a = gpu[k].astype(np.float64).reshape(gpu[k].shape[0], -1)
        b = ora[k].reshape(a.shape)
        cond = ora["_abs"][k].reshape(a.shape)
        err = np.abs(a - b)
        floor = floor0
        if floor_frac is not None and a.size:
            bs = np.abs(b).max(1)
            if (bs > 0).any():
                floor = max(floor0, floor_frac * float(np.percentile(bs[bs > 0], 99)))
        strict = err <= rel * np.abs(b) + floor
        slack = sum_eps if cond_rho is None else (sum_eps + 16.0 * np.asarray(cond_rho, np.float64))[:, None]
        if k == "d_opacity":
            block = cond * (sum_eps / rel)
        elif k in ("d_pos", "d_scale"):  # both are gradients w.r.t. world lengths made from the same homography gradient: one block
            block = np.maximum(np.abs(ora["d_pos"]).reshape(a.shape[0], -1).max(1), np.abs(ora["d_scale"]).reshape(a.shape[0], -1).max(1))[:, None]
        else:
            block = np.abs(b).max(1, keepdims=True)
        ok = strict | (err <= rel * block + floor) | (err <= slack * cond + floor)
        n_strict_fail = int((~strict).sum())
        big = np.abs(b) > floor
        report[k] = dict(n=int(a.size), strict_fail=n_strict_fail, strict_fail_frac=n_strict_fail / max(1, a.size), fail=int((~ok).sum()),
                         worst_strict_rel=float((err / (np.abs(b) + floor / rel)).max()) if a.size else 0.0,
                         worst_cond_units=float((err / np.maximum(cond, 1e-300))[big & (cond > 0)].max()) if (big & (cond > 0)).any() else 0.0)
        if not ok.all():
            j, c = np.argwhere(~ok)[0]
            raise AssertionError(f"{k}[{j},{c}]: gpu {a[j, c]:.8e} oracle {b[j, c]:.8e} sum|terms| {cond[j, c]:.3e}; {report[k]}")
        assert n_strict_fail <= max(3, max_strict_fail * a.size), f"{k}: {n_strict_fail} of {a.size} entries miss the strict rule; {report[k]}"
    return report
