"""Occlusion-aware pruning drivers: orchestration only -- every step runs in the CUDA
library; this module loops over views and marshals arguments.

* accumulate_visibility: render the given views with the statistics switched on ("Inside the renderer, we save which
  Gaussians are used during the color accumulation step"); `vis_count` / `contrib_sum` accumulate.
* prune: "remove all Gaussians that are not visible in any training view" (the post-hoc variant; the same
  call serves the in-training variant every 100 / 600 iterations) -- mask, remap, compacted parameters.
"""
from __future__ import annotations

from typing import Dict, Optional, Sequence

import torch

from . import binding as B


def accumulate_visibility(surfels: B.ocgs_surfels, n: int, cameras: Sequence, cfg: B.ocgs_config, ws: torch.Tensor, key_capacity: int,
                          out: Optional[Dict[str, torch.Tensor]], vis_count: torch.Tensor, contrib_sum: torch.Tensor, stream=None,
                          ws2: Optional[torch.Tensor] = None) -> None:
    """Forward-only pass over `cameras` (scene cameras or ocgs_camera structs); the per-surfel statistics accumulate.
    out = None: the statistics-only pass (ocgs_visibility_pass: no images, no SH colour); otherwise the full forward pass,
    the images in `out` overwritten per view.  ws2 (statistics-only pass): a second workspace of the same size; views then
    alternate between two streams.  One host synchronisation, at the end; raises OcgsError if any view overflowed the key capacity."""
    cams = [cam if isinstance(cam, B.ocgs_camera) else B.camera_from(cam) for cam in cameras]
    cur = torch.cuda.current_stream() if stream is None else stream
    # every view's workspace header (K, n_vis, error word; the next view's preprocess clears it) is kept on the device and
    # checked once at the end, so that a key-capacity overflow in ANY view is reported without a per-view synchronisation
    headers = torch.zeros((max(len(cams), 1), 4), dtype=torch.int32, device=ws.device)

    def keep_header(i, w, st):
        with torch.cuda.stream(st):
            headers[i].copy_(w[:16].view(torch.int32), non_blocking=True)

    if out is None and ws2 is not None:
        # two views in flight: the short sort kernels and the tail of one view's walk (a few long tile lists on a few SMs)
        # overlap the other view's work; both streams add into the same statistics with atomics
        lanes = [(ws, torch.cuda.Stream()), (ws2, torch.cuda.Stream())]
        for _, st in lanes:
            st.wait_stream(cur)
        for i, c in enumerate(cams):
            w, st = lanes[i % 2]
            B.ocgs_visibility_pass(surfels, c, cfg, w, key_capacity, vis_count, contrib_sum, st)
            keep_header(i, w, st)
        for _, st in lanes:
            cur.wait_stream(st)
    else:
        for i, c in enumerate(cams):
            if out is None:
                B.ocgs_visibility_pass(surfels, c, cfg, ws, key_capacity, vis_count, contrib_sum, cur)
            else:
                B.ocgs_preprocess(surfels, c, cfg, ws, key_capacity, cur)
                B.ocgs_bin_sort(n, c, cfg, ws, key_capacity, None, cur)
                B.ocgs_render_fwd(n, c, cfg, ws, key_capacity, None, out["color"], out["alpha"], out["depth"], out["normal"], out["n_contrib"],
                                  None, vis_count, contrib_sum, cur)
            keep_header(i, ws, cur)
    cur.synchronize()
    err = headers[:, 3].cpu()
    if int((err & 1).sum()) > 0:
        bad = int(torch.nonzero(err & 1)[0])
        need = int(headers[bad, :2].cpu().numpy().view("uint64")[0])
        raise B.OcgsError(f"accumulate_visibility: view {bad} needs key_capacity >= {need}", B.OCGS_ERR_CAPACITY)
    if int((err & 2).sum()) > 0:
        raise B.OcgsError("accumulate_visibility: a tile list exceeds 2^24 entries", B.OCGS_ERR_UNSUPPORTED)


def prune(surfels: B.ocgs_surfels, params: Dict[str, torch.Tensor], n: int, cfg: B.ocgs_config, vis_count: torch.Tensor,
          contrib_sum: torch.Tensor, reset_stats: bool = True, extra_rows: Optional[Dict[str, torch.Tensor]] = None, stream=None):
    """Prune mask from the statistics, stable compaction of the five parameter arrays and of any `extra_rows` (per-surfel
    [n, k] float arrays such as optimiser moments).  Returns (compacted params, compacted extras, n_kept, prune_mask, remap)."""
    dev = vis_count.device
    mask = torch.empty(n, dtype=torch.uint8, device=dev)
    remap = torch.empty(n, dtype=torch.int32, device=dev)
    n_out = torch.zeros(1, dtype=torch.int32, device=dev)
    outs = {k: torch.empty_like(params[k]) for k in ("pos", "scale", "quat", "opacity", "sh")}
    om = B.ocgs_surfels_mut(*[B._ptr(outs[k]) for k in ("pos", "scale", "quat", "opacity", "sh")], n)
    pws = torch.empty(B.ocgs_prune_workspace_bytes(n), dtype=torch.uint8, device=dev)
    B.ocgs_prune_stats(surfels, vis_count, contrib_sum, cfg, mask, remap, om, n_out, 1 if reset_stats else 0, pws, stream)
    extras = {}
    for k, t in (extra_rows or {}).items():
        o = torch.empty_like(t)
        B.ocgs_compact_rows(t, remap, n, int(t.numel() // max(n, 1)), o, stream)
        extras[k] = o
    kept = int(n_out.item())  # the one host read of the pass
    return {k: v[:kept] for k, v in outs.items()}, {k: v[:kept] for k, v in extras.items()}, kept, mask, remap
