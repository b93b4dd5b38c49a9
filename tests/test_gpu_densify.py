"""-m gpu: ocgs_densify_accumulate / ocgs_densify (clone / split of the adaptive density control, PAPER.md:67, :129;
SURVEY.md 8(f) f-4) against oracle/densify.py.  Classes, counts, order and source ids bit-exact; copied parameters
bit-exact; children positions / scales to fp32 rounding (the oracle forms them in fp64)."""
import numpy as np
import pytest

from gpu_harness import GpuView
from oracle import densify as dn
from paper_2501_08174_b200 import scenegen as sg

pytestmark = pytest.mark.gpu


def gpu_densify(P, grad, den, tau, smax, xi, capacity):
    import torch
    from paper_2501_08174_b200 import binding as B
    n = P[0].shape[0]
    t = [torch.tensor(np.ascontiguousarray(a, np.float32), device="cuda") for a in P]
    surf = B.make_surfels(*t) if n > 0 else B.ocgs_surfels(None, None, None, None, None, 0)
    outs = [torch.full((capacity,) + tuple(a.shape[1:]), -7.0, dtype=torch.float32, device="cuda") for a in P]
    om = B.ocgs_surfels_mut(*[B._ptr(o) for o in outs], capacity)
    src = torch.full((capacity,), -5, dtype=torch.int32, device="cuda")
    counts = torch.zeros(4, dtype=torch.int32, device="cuda")
    ws = torch.empty(max(B.ocgs_densify_workspace_bytes(n), 16), dtype=torch.uint8, device="cuda")
    B.ocgs_densify(surf, torch.tensor(grad, device="cuda"), torch.tensor(den.astype(np.int32), device="cuda"), tau, smax,
                   torch.tensor(xi, device="cuda"), om, src, counts, ws)
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in outs], src.cpu().numpy(), counts.cpu().numpy()


def compare(P, grad, den, tau, smax, xi, capacity=None):
    n = P[0].shape[0]
    capacity = capacity if capacity is not None else 2 * n + 4
    outs, src, counts = gpu_densify(P, grad, den, tau, smax, xi, capacity)
    r = dn.densify(*P, grad, den, tau, smax, xi)
    assert list(counts) == [r["n_out"], r["n_keep"], r["n_clone"], r["n_split"]]
    k = min(r["n_out"], capacity)
    assert np.array_equal(src[:k], r["src"][:k]) and np.all(src[k:] == -5)
    kc = min(r["n_keep"] + r["n_clone"], capacity)
    for o, name in zip(outs, ("pos", "scale", "quat", "opacity", "sh")):
        ref = r[name]
        assert np.array_equal(o[:kc], ref[:kc].astype(np.float32)), name          # copies: bit-exact
        if name in ("pos", "scale"):
            assert np.allclose(o[kc:k], ref[kc:k], rtol=3e-7, atol=1e-7), name     # children: fp32 rounding of an fp64 result
        else:
            assert np.array_equal(o[kc:k], ref[kc:k].astype(np.float32)), name
        assert np.all(o[k:] == -7.0), name                                         # nothing written past n_out / capacity
    return r


def random_case(n, seed):
    rng = np.random.default_rng(seed)
    sc = sg.random_scene(n, 32, 32, 30.0, seed=seed, sh_degree=3)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    den = rng.integers(0, 5, n).astype(np.uint32)
    grad = (rng.uniform(0, 6e-4, n) * den).astype(np.float32)
    xi = rng.normal(size=(n, 2, 2)).astype(np.float32)
    return P, grad, den, xi


def test_random_inputs_several_sizes_and_thresholds():
    for n, seed in ((1, 1), (255, 2), (256, 3), (100_003, 4)):
        P, grad, den, xi = random_case(n, seed)
        smax = float(np.median(P[1].max(1)))
        r = compare(P, grad, den, 2e-4, smax, xi)
        if n > 1000:
            assert min(r["n_keep"], r["n_clone"], r["n_split"]) > 1000
    P, grad, den, xi = random_case(5000, 5)
    assert compare(P, grad, den, 1.0, 0.01, xi)["n_out"] == 5000          # nothing selected: identity
    assert compare(P, np.ones(5000, np.float32), np.ones(5000, np.uint32), 2e-4, 0.0, xi)["n_split"] == 5000   # everything split
    assert compare(P, np.ones(5000, np.float32), np.ones(5000, np.uint32), 2e-4, 1e9, xi)["n_clone"] == 5000   # everything cloned


def test_capacity_smaller_than_the_result_drops_rows_and_reports_the_count():
    P, grad, den, xi = random_case(4000, 6)
    r = compare(P, np.ones(4000, np.float32), np.ones(4000, np.uint32), 2e-4, 0.0, xi, capacity=5000)  # needs 8000 rows
    assert r["n_out"] == 8000


def test_empty_input():
    sc = sg.random_scene(4, 32, 32, 30.0, seed=1, sh_degree=3)
    P = tuple(a[:0] for a in (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh))
    outs, src, counts = gpu_densify(P, np.zeros(0, np.float32), np.zeros(0, np.uint32), 2e-4, 0.01, np.zeros((0, 2, 2), np.float32), 4)
    assert list(counts) == [0, 0, 0, 0]


def test_accumulate_over_views_matches_the_definition():
    """grad_accum / denom over three views of a scene: |d_center2d| of each view's backward pass, only for surfels inside
    that view's frustum (the workspace's id_to_rank), against the oracle's accumulate on the same per-view gradients."""
    import torch
    from paper_2501_08174_b200 import binding as B
    sc = sg.make_scene("config1")
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    n = sc.n
    ga_t = torch.zeros(n, device="cuda"); de_t = torch.zeros(n, dtype=torch.int32, device="cuda")
    ga_o, de_o = np.zeros(n), np.zeros(n, np.int64)
    g = GpuView(P, sc.cameras[0], dict(sh_degree=0))
    rng = np.random.default_rng(0)
    for v in range(3):
        g.cam = B.camera_from(sc.cameras[v])
        gp = g.preprocess(); g.bin_sort(want_ids=False)
        g.render_fwd(mask=sc.mask(v))
        gg = g.render_bwd(gC=rng.normal(size=(3, g.H, g.W)))
        d2 = torch.tensor(gg["d_center2d"], device="cuda")
        B.ocgs_densify_accumulate(g.ws, n, g.W, g.H, g.cap, d2, ga_t, de_t)
        dn.accumulate(ga_o, de_o, gg["d_center2d"], gp["tiles"] > 0, g.W, g.H)
    torch.cuda.synchronize()
    assert np.array_equal(de_t.cpu().numpy(), de_o)
    assert np.allclose(ga_t.cpu().numpy(), ga_o, rtol=1e-6, atol=1e-12)
    assert (de_o > 0).sum() > 500 and (de_o == 0).sum() > 10
