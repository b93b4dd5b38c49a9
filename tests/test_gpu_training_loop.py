"""-m gpu: the pieces used together the way the paper's training loop uses them ("pick a view, render, losses,
backpropagate", :129 pruning every interval from the statistics gathered inside the renderer, Eq. 3's gamma L_b): Adam steps
on perturbed parameters with the library's gradients must bring the library's loss down on every view, through a prune +
clone/split in the middle that changes N.  An integration check of signs and scales; element-wise parity is elsewhere."""
import numpy as np
import pytest

from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu


def test_adam_on_library_gradients_reduces_the_loss_through_a_prune_and_densify():
    import torch
    from paper_2501_08174_b200 import binding as B, pruning
    sc = sg.make_scene("config1")
    dev = "cuda"
    W, H = sc.cameras[0].width, sc.cameras[0].height
    cams = [B.camera_from(c) for c in sc.cameras]
    masks = [torch.tensor(sc.mask(v), device=dev) for v in range(len(cams))]
    cfg = B.ocgs_default_config(sh_degree=0)
    out = B.alloc_outputs(W, H)
    gC = torch.empty((3, H, W), device=dev)
    l1 = torch.zeros(1, device=dev)

    def setup(params):
        n = params["pos"].shape[0]
        cap = max(1 << 16, 64 * n)
        return dict(n=n, cap=cap, ws=B.alloc_workspace(n, W, H, cap), grads=B.alloc_grads(n),
                    surfels=B.make_surfels(params["pos"], params["scale"], params["quat"], params["opacity"], params["sh"]),
                    vis=torch.zeros(n, dtype=torch.int32, device=dev), cs=torch.zeros(n, device=dev),
                    gacc=torch.zeros(n, device=dev), den=torch.zeros(n, dtype=torch.int32, device=dev))

    def render_loss_grads(params, st, v, target, backward=True):
        B.ocgs_preprocess(st["surfels"], cams[v], cfg, st["ws"], st["cap"])
        B.ocgs_bin_sort(st["n"], cams[v], cfg, st["ws"], st["cap"])
        B.ocgs_render_fwd_l1(st["n"], cams[v], cfg, st["ws"], st["cap"], masks[v], target, out["color"], out["alpha"], out["depth"],
                             out["normal"], out["n_contrib"], out["loss_bg"], l1, gC, st["vis"], st["cs"])
        if backward:
            g = st["grads"]
            B.ocgs_render_bwd(st["surfels"], cams[v], cfg, st["ws"], st["cap"], masks[v], out["n_contrib"], gC, None, None, None,
                              g["d_pos"], g["d_scale"], g["d_quat"], g["d_opacity"], g["d_sh"], g["d_center2d"])
            B.ocgs_densify_accumulate(st["ws"], st["n"], W, H, st["cap"], g["d_center2d"], st["gacc"], st["den"])
        return float(l1.item()) + cfg.gamma_bg * float(out["loss_bg"].item())

    # targets: renders of the reference scene
    ref = {k: torch.tensor(np.ascontiguousarray(getattr(sc, k), np.float32), device=dev) for k in ("pos", "scale", "quat", "opacity", "sh")}
    st = setup(ref)
    targets = []
    for v in range(len(cams)):
        render_loss_grads(ref, st, v, torch.zeros((3, H, W), device=dev), backward=False)
        targets.append(out["color"].clone())
    # start: positions, colours and opacities perturbed
    rng = np.random.default_rng(0)
    params = {k: t.clone() for k, t in ref.items()}
    params["pos"] += torch.tensor(rng.normal(0, 0.02, sc.pos.shape).astype(np.float32), device=dev)
    params["sh"][:, 0] += torch.tensor(rng.normal(0, 0.5, (sc.n, 3)).astype(np.float32), device=dev)
    params["opacity"] = (params["opacity"] * 0.7).contiguous()
    st = setup(params)

    def total_loss(params, st):
        return [render_loss_grads(params, st, v, targets[v], backward=False) for v in range(len(cams))]

    def make_opt(params):
        return torch.optim.Adam([dict(params=[params["pos"]], lr=2e-3), dict(params=[params["sh"]], lr=2e-2),
                                 dict(params=[params["opacity"]], lr=1e-2)])

    def train(params, st, steps, opt):
        for it in range(steps):
            v = it % len(cams)
            render_loss_grads(params, st, v, targets[v])
            g = st["grads"]
            params["pos"].grad, params["sh"].grad, params["opacity"].grad = g["d_pos"], g["d_sh"], g["d_opacity"]
            opt.step()
            with torch.no_grad():
                params["opacity"].clamp_(0.01, 0.99)  # activated values are what the library takes

    start = total_loss(params, st)
    train(params, st, 60, make_opt(params))
    mid = total_loss(params, st)
    assert all(m < 0.8 * s for m, s in zip(mid, start)), (start, mid)
    # prune on the statistics gathered inside the renderer during those steps, then clone / split; N changes
    n0 = st["n"]
    new_params, _, kept, mask, remap = pruning.prune(st["surfels"], params, n0, cfg, st["vis"], st["cs"], reset_stats=True)
    assert 0 < kept < n0
    gacc = torch.empty(kept, device=dev); den = torch.empty(kept, dtype=torch.int32, device=dev)
    B.ocgs_compact_rows(st["gacc"], remap, n0, 1, gacc)
    B.ocgs_compact_rows(st["den"].view(torch.float32), remap, n0, 1, den.view(torch.float32))
    p2 = {k: new_params[k][:kept].contiguous() for k in new_params}
    surf2 = B.make_surfels(p2["pos"], p2["scale"], p2["quat"], p2["opacity"], p2["sh"])
    cap_rows = 2 * kept
    outs = {k: torch.empty((cap_rows,) + tuple(p2[k].shape[1:]), device=dev) for k in p2}
    om = B.ocgs_surfels_mut(*[B._ptr(outs[k]) for k in ("pos", "scale", "quat", "opacity", "sh")], cap_rows)
    counts = torch.zeros(4, dtype=torch.int32, device=dev)
    src = torch.empty(cap_rows, dtype=torch.int32, device=dev)
    xi = torch.tensor(rng.normal(size=(kept, 2, 2)).astype(np.float32), device=dev)
    dws = torch.empty(max(B.ocgs_densify_workspace_bytes(kept), 16), dtype=torch.uint8, device=dev)
    # the statistic is per NDC unit, so the cited work's DEFAULT threshold 2e-4 is of the order of the
    # statistic of a scene that is still 30 % away from its targets (measured: median 9e-4, 94 % selected on this small, badly
    # perturbed scene); in pixel units the statistic would sit W/2 times lower and the default would select nothing
    avg = (gacc / den.clamp(min=1)).float()
    frac_default = float((avg >= 2e-4).float().mean().item())
    print("PARITY densify: share of surfels selected at the default grad_threshold 2e-4: %.4f (median statistic %.3e)" % (frac_default, float(avg.median().item())))
    assert frac_default > 0.005 and 2e-5 < float(avg.median().item()) < 2e-2, frac_default  # the statistic lives in the decade of the default
    B.ocgs_densify(surf2, gacc, den, 2e-4, float(p2["scale"].max(1).values.median().item()), xi, om, src, counts, dws)
    assert int(counts[2].item()) + int(counts[3].item()) == int((avg >= 2e-4).sum().item())
    tau = float(torch.quantile(avg, 0.9).item())  # densify the top tenth
    B.ocgs_densify(surf2, gacc, den, tau, float(p2["scale"].max(1).values.median().item()), xi, om, src, counts, dws)
    n_out = int(counts[0].item())
    assert kept < n_out <= cap_rows and int(counts[2].item()) + int(counts[3].item()) > 0
    params = {k: outs[k][:n_out].contiguous() for k in outs}
    st = setup(params)
    after_edit = total_loss(params, st)
    train(params, st, 60, make_opt(params))
    end = total_loss(params, st)
    assert all(e < a for e, a in zip(end, after_edit)), (after_edit, end)
    assert all(e < 0.7 * s for e, s in zip(end, start)), (start, end)
