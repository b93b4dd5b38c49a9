"""Pins of the CPU oracle against things other than itself (run with -m "not gpu").

Each test names the passage / reading it pins.  Closed forms, invariants, special cases that reduce to textbook
results, brute force with an exhaustive per-pixel sort, and central finite differences.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as orc
from paper_2501_08174_b200 import scenegen as sg

Y0 = 0.5 * math.sqrt(1.0 / math.pi)


def ident_cam(W, H, f, cx=None, cy=None):
    return orc.make_camera(np.eye(4, dtype=np.float32), f, f, W / 2 if cx is None else cx, H / 2 if cy is None else cy, W, H)


def one_surfel(pos, scale, quat=(1, 0, 0, 0), opacity=0.8, rgb=(0.2, 0.5, 0.9)):
    sh = np.zeros((1, 16, 3), np.float32)
    sh[0, 0] = (np.asarray(rgb) - 0.5) / Y0
    return (np.asarray([pos], np.float32), np.asarray([scale], np.float32), np.asarray([quat], np.float32),
            np.asarray([opacity], np.float32), sh)


def stack(*surfels):
    return tuple(np.concatenate([s[i] for s in surfels]) for i in range(5))


# ---------------------------------------------------------------------------------------------
# S14: the SH basis is orthonormal on the sphere (pins every constant and polynomial)
# ---------------------------------------------------------------------------------------------
def test_sh_basis_orthonormal_by_quadrature():
    nodes, weights = np.polynomial.legendre.leggauss(24)  # exact for polynomials of degree <= 47 in cos(theta)
    nphi = 32  # exact for trigonometric degree <= 31
    G = np.zeros((16, 16))
    for ct, w in zip(nodes, weights):
        st = math.sqrt(1 - ct * ct)
        for k in range(nphi):
            ph = 2 * math.pi * (k + 0.5) / nphi
            Y = orc.sh_basis([st * math.cos(ph), st * math.sin(ph), ct])
            G += w * (2 * math.pi / nphi) * np.outer(Y, Y)
    assert np.abs(G - np.eye(16)).max() < 1e-12


def test_sh_sign_convention_degree1():
    # S14: Y1..3 = sqrt(3/4pi) * (-y, z, -x)
    c1 = math.sqrt(3 / (4 * math.pi))
    Y = orc.sh_basis([0.0, 0.0, 1.0])
    assert Y[2] == pytest.approx(c1) and abs(Y[1]) < 1e-15 and abs(Y[3]) < 1e-15
    Y = orc.sh_basis([1.0, 0.0, 0.0])
    assert Y[3] == pytest.approx(-c1)
    Y = orc.sh_basis([0.0, 1.0, 0.0])
    assert Y[1] == pytest.approx(-c1)


def test_colour_clamp_decision_fp32_sequence():
    """S14 / DESIGN.md reading R-clamp: channel c is clamped iff the fp32 sequence acc_c = fma(Y_k, sh_kc, acc_c) (k in order,
    from 1/2) is negative.  Pins: (i) the fp32 values track the fp64 colour (whose basis the quadrature test above pins) to the
    error of a 16-term fp32 sum, on random directions and coefficients and for every degree -- a wrong constant, sign or
    polynomial in the fp32 basis moves them by 1e-2; (ii) wherever the fp64 value is clear of zero the decision is its
    sign; (iii) degree 0 is exact: acc = fma(fl(Y0), sh_0, 1/2), so the requested colours below clamp exactly the channels
    that are negative after the fp32 rounding of sh_0; (iv) a clamped channel's value is exactly 0, an open one's the fp64 value."""
    rng = np.random.default_rng(7)
    cam = orc.camera_from(sg.random_scene(4, 32, 32, 30.0, seed=1, sh_degree=0).cameras[0])  # a generic pose
    worst = 0.0
    for deg in (0, 1, 2, 3):
        for _ in range(1500):
            p = rng.normal(size=3) * 2.0
            sh = rng.normal(size=(16, 3)) * 0.6
            a32, a64, cl = orc.colour_probe(p, sh, deg, cam)
            worst = max(worst, float(np.abs(a32 - a64).max()))
            for c in range(3):
                if abs(a64[c]) > 4e-6:
                    assert bool(cl >> c & 1) == (a64[c] < 0)
                assert bool(cl >> c & 1) == (a32[c] < 0)
    assert worst < 4e-6
    # degree 0, by hand
    y0f = np.float32(Y0)
    for rgb in ((-1e-3, 1e-3, 0.5), (-1e-6, 1e-6, -0.2), (0.0, -3e-7, 3e-7), (-1e-5, 1e-5, 2.0)):
        s = one_surfel((0.3, -0.2, 2.0), (0.1, 0.1), rgb=rgb)
        a32, a64, cl = orc.colour_probe(s[0][0], s[4][0], 0, ident_cam(32, 32, 50.0))
        expect = [float(Fraction(float(y0f)) * Fraction(float(s[4][0, 0, c])) + Fraction(1, 2)) for c in range(3)]  # one rounding of the exact value
        assert [float(v) for v in a32] == [float(np.float32(e)) for e in expect]
        assert cl == sum(1 << c for c in range(3) if np.float32(expect[c]) < 0)
    cfg = orc.default_config(sh_degree=0)
    s = stack(*[one_surfel((0, 0, 2.0), (0.1, 0.1), rgb=c) for c in ((-1e-3, 1e-3, 0.5), (0.25, -0.5, 0.0))])
    pre = orc.preprocess(*s, ident_cam(32, 32, 50.0), cfg)
    assert list(pre["clamp"][:2]) == [0b001, 0b010 | (int(pre["clamp"][1]) & 0b100)]
    assert pre["rgb"][0, 0] == 0.0 and pre["rgb"][1, 1] == 0.0 and np.all(pre["rgb"] >= 0.0)
    assert np.allclose(pre["rgb"][0], [0.0, 1e-3, 0.5], atol=1e-7)


# ---------------------------------------------------------------------------------------------
# north_star: "a single fronto-parallel surfel gives an analytic Gaussian footprint"
# ---------------------------------------------------------------------------------------------
def test_fronto_parallel_surfel_is_analytic_gaussian():
    W = H = 64
    f, z0, su, sv, o = 100.0, 2.0, 0.10, 0.16, 0.8
    rgb = np.array([0.2, 0.5, 0.9])
    cam = ident_cam(W, H, f)
    cfg = orc.default_config(sh_degree=0)
    s = one_surfel((0, 0, z0), (su, sv), opacity=o, rgb=rgb)
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    assert pre["visible"][0] == 1
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    u = (xs - (W / 2 - 0.5)) * z0 / (f * su)
    v = (ys - (H / 2 - 0.5)) * z0 / (f * sv)
    rho = u * u + v * v
    # fx*s/z0 = 5 and 8 px >= sigma_f, so the screen-space filter never wins
    expect = np.where(rho <= 9.0, np.minimum(0.99, o * np.exp(-0.5 * rho)), 0.0)
    assert np.abs(fwd["alpha"] - expect).max() < 1e-6  # M is fp32: ~1e-7 relative
    assert np.abs(fwd["color"] - expect[None] * rgb[:, None, None]).max() < 1e-6
    assert np.abs(fwd["depth"] - expect * z0).max() < 1e-5
    # facing normal: t_w = +z points away from the camera, so it is flipped to -z
    assert np.abs(fwd["normal"][2] + expect).max() < 1e-6 and np.abs(fwd["normal"][:2]).max() < 1e-12
    # rect: centre +- 3 sigma_px, pixel-exact
    cxp, cyp = W / 2 - 0.5, H / 2 - 0.5
    assert list(pre["rect"][0]) == [math.ceil(cxp - 3 * f * su / z0), math.ceil(cyp - 3 * f * sv / z0),
                                    math.floor(cxp + 3 * f * su / z0), math.floor(cyp + 3 * f * sv / z0)]


def test_off_axis_tilted_surfel_matches_explicit_ray_plane():
    """O4's homography form against a by-hand ray-plane intersection for one tilted surfel, one pixel."""
    W = H = 48
    f = 60.0
    ang = 0.7
    quat = (math.cos(ang / 2), math.sin(ang / 2) * 0.6, math.sin(ang / 2) * 0.8, 0.0)
    p = np.array([0.3, -0.2, 2.5])
    su, sv, o = 0.3, 0.2, 0.7
    s = one_surfel(p, (su, sv), quat=quat, opacity=o)
    cam = ident_cam(W, H, f)
    cfg = orc.default_config(sh_degree=0)
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    w, x, y, z = quat
    tu = np.array([1 - 2 * (y * y + z * z), 2 * (x * y + w * z), 2 * (x * z - w * y)])
    tv = np.array([2 * (x * y - w * z), 1 - 2 * (x * x + z * z), 2 * (y * z + w * x)])
    n = np.cross(tu, tv)
    for (px, py) in [(30, 20), (24, 24), (35, 15)]:
        d = np.array([(px - (W / 2 - 0.5)) / f, (py - (H / 2 - 0.5)) / f, 1.0])
        t = (n @ p) / (n @ d)
        hit = t * d - p
        u, v = hit @ tu / su, hit @ tv / sv
        c2 = np.array([f * p[0] / p[2] + W / 2 - 0.5, f * p[1] / p[2] + H / 2 - 0.5])
        rho = min(u * u + v * v, 2 * ((px - c2[0]) ** 2 + (py - c2[1]) ** 2))
        a = min(0.99, o * math.exp(-rho / 2)) if rho <= 2 * math.log(o * 255) and rho <= 9 else 0.0
        assert fwd["alpha"][py, px] == pytest.approx(a, abs=2e-6)
        if a > 0 and u * u + v * v <= rho:
            assert fwd["depth"][py, px] == pytest.approx(a * t, abs=1e-5)


# ---------------------------------------------------------------------------------------------
# S8: edge-on surfel through the optical axis -> isotropic screen-space Gaussian of std sigma_f
# ---------------------------------------------------------------------------------------------
def test_edge_on_surfel_reduces_to_screen_space_filter():
    W = H = 32
    f, z0, o = 50.0, 2.0, 0.9
    # rotate the frame so that t_w = +x (normal perpendicular to the optical axis): R = rot_y(90deg): t_u = -z, t_v = y
    quat = (math.cos(math.pi / 4), 0.0, math.sin(math.pi / 4), 0.0)
    s = one_surfel((0, 0, z0), (0.05, 0.05), quat=quat, opacity=o)
    cam = ident_cam(W, H, f)  # optical axis falls between pixel centres, no pixel ray lies in the plane
    cfg = orc.default_config(sh_degree=0)
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    assert pre["visible"][0] == 1
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    d2 = (xs - (W / 2 - 0.5)) ** 2 + (ys - (H / 2 - 0.5)) ** 2
    expect = np.where(2 * d2 <= 9.0, o * np.exp(-d2), 0.0)
    assert np.abs(fwd["alpha"] - expect).max() < 1e-7
    assert np.abs(fwd["depth"] - expect * z0).max() < 1e-6  # S10: centre depth when the filter term wins
    # rect = union of the filter disc (radius sigma_f*sqrt(rho_cut) = sqrt(4.5) px) and the projected ellipse, which
    # is edge-on: a segment of half-length 3 * f * s_v / z0 = 3.75 px along y
    r = math.sqrt(4.5)
    c = W / 2 - 0.5
    assert list(pre["rect"][0]) == [math.ceil(c - r), math.ceil(c - 3.75), math.floor(c + r), math.floor(c + 3.75)]


# ---------------------------------------------------------------------------------------------
# O5: compositing closed forms
# ---------------------------------------------------------------------------------------------
def test_two_layer_closed_form_and_background():
    W = H = 16
    cam = ident_cam(W, H, 40.0)
    cfg = orc.default_config(sh_degree=0, bg=(0.1, 0.2, 0.3))
    c1, c2 = np.array([0.9, 0.1, 0.3]), np.array([0.2, 0.8, 0.6])
    s = stack(one_surfel((0, 0, 3.0), (1.0, 1.0), opacity=0.6, rgb=c2), one_surfel((0, 0, 1.5), (1.0, 1.0), opacity=0.5, rgb=c1))
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    # pixel nearest the axis: offset (0.5, 0.5) px
    px = py = W // 2
    a = []
    for z0, o in ((1.5, 0.5), (3.0, 0.6)):
        u = 0.5 * z0 / 40.0
        a.append(o * math.exp(-0.5 * (2 * u * u)))
    T = (1 - a[0]) * (1 - a[1])
    expC = a[0] * c1 + (1 - a[0]) * a[1] * c2 + T * np.array([0.1, 0.2, 0.3])
    assert np.allclose(fwd["color"][:, py, px], expC, atol=1e-6)
    assert fwd["alpha"][py, px] == pytest.approx(1 - T, abs=1e-7)
    assert fwd["n_contrib"][py, px] == 2
    # depth moments (reading R-moments) about the first blended pair's depth c = 1.5: m1 = sum w (z - c), m2 = sum w (z - c)^2
    w1, w2 = a[0], (1 - a[0]) * a[1]
    assert fwd["depth"][py, px] == pytest.approx(w1 * 1.5 + w2 * 3.0, abs=1e-6)
    assert fwd["origin"][py, px] == pytest.approx(1.5, abs=1e-6)
    assert fwd["m1"][py, px] == pytest.approx(w2 * 1.5, abs=1e-6) and fwd["m2"][py, px] == pytest.approx(w2 * 1.5 ** 2, abs=1e-6)
    # ... and the pairwise distortion sum_{i<j} w_i w_j (z_i - z_j)^2 = A m2 - m1^2
    A_ = fwd["alpha"][py, px]
    assert A_ * fwd["m2"][py, px] - fwd["m1"][py, px] ** 2 == pytest.approx(w1 * w2 * 1.5 ** 2, abs=1e-6)
    # sort order: the nearer surfel (id 1) first although its id is larger (S9)
    t = (py // 16) * 1 + px // 16
    assert list(srt["ids"][srt["ranges"][t, 0]:srt["ranges"][t, 1]]) == [1, 0]


def test_opaque_front_layers_occlude_surfel_behind_exact_zero():
    """north_star: "an opaque front surfel gives zero contribution to the surfel behind it"; PAPER.md:119 (G_j gets
    'false'), PAPER.md:121 ("occluded ... cannot receive gradients")."""
    W = H = 16
    cam = ident_cam(W, H, 40.0)
    cfg = orc.default_config(sh_degree=0)
    layers = [one_surfel((0, 0, 1.0 + 0.1 * i), (5.0, 5.0), opacity=0.95) for i in range(4)]
    behind = one_surfel((0, 0, 3.0), (0.05, 0.05), opacity=0.9)
    s = stack(*layers, behind)
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    assert pre["visible"][4] == 1 and pre["tiles_touched"][4] >= 1  # in frustum, assigned to pixels
    # T after 3 layers = 0.05^3 = 1.25e-4; the 4th would leave 6.25e-6 < 1e-4 -> not blended (S11)
    assert np.all(fwd["n_contrib"] == 3)
    assert np.all(fwd["vis_count"][:3] == W * H) and fwd["vis_count"][3] == 0 and fwd["vis_count"][4] == 0
    assert fwd["contrib_sum"][4] == 0.0
    assert fwd["alpha"].max() <= 0.9999 + 1e-12  # "threshold opacity close to 1"
    rng = np.random.default_rng(0)
    g = orc.render_bwd(*s, pre, srt, cam, cfg, mask=np.zeros((H, W), np.uint8), gC=rng.normal(size=(3, H, W)),
                       gA=rng.normal(size=(H, W)), gD=rng.normal(size=(H, W)), gN=rng.normal(size=(3, H, W)))
    for k, v in [kv for kv in g.items() if kv[0] != "_abs"] + list(g["_abs"].items()):
        assert np.all(v[4] == 0.0), k
        assert np.all(v[3] == 0.0), k
    assert np.any(g["d_opacity"][:3] != 0.0)
    # prune rule (O9 / PAPER.md:119): the occluded surfel and an out-of-frustum one are both removed
    pr = orc.prune(fwd["vis_count"], fwd["contrib_sum"].astype(np.float32), s[3])
    assert list(pr["prune_mask"]) == [0, 0, 0, 1, 1] and list(pr["remap"]) == [0, 1, 2, -1, -1] and pr["n_out"] == 3


def test_out_of_frustum_surfel_is_disqualified():
    """G_k outside the viewing frustum is "not assigned to any pixel"."""
    W = H = 32
    cam = ident_cam(W, H, 40.0)
    cfg = orc.default_config(sh_degree=0)
    s = stack(one_surfel((0, 0, 2.0), (0.1, 0.1)),          # visible
              one_surfel((0, 0, -2.0), (0.1, 0.1)),         # behind the camera
              one_surfel((10.0, 0, 2.0), (0.1, 0.1)),       # far off to the side
              one_surfel((0, 0, 0.1), (0.01, 0.01)),        # in front of the near plane (S3)
              one_surfel((0, 0, 2.0), (0.1, 0.1), opacity=0.003))  # below alpha_min everywhere (S4)
    pre, srt, fwd = orc.forward_view(*s, cam, cfg)
    assert list(pre["visible"]) == [1, 0, 0, 0, 0]
    assert list(pre["tiles_touched"]) == [4, 0, 0, 0, 0] or pre["tiles_touched"][0] >= 1
    assert srt["K"] == int(pre["tiles_touched"].sum())
    assert np.all(fwd["vis_count"][1:] == 0)


# ---------------------------------------------------------------------------------------------
# Eq. 1: L_b = 1/(h w) sum A (1 - M)
# ---------------------------------------------------------------------------------------------
def test_background_loss_eq1_special_cases_and_gradient_sign():
    sc = sg.random_scene(40, 40, 32, 45.0, seed=11, sh_degree=1)
    cam = orc.camera_from(sc.cameras[0])
    cfg = orc.default_config(sh_degree=1)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    H, W = 32, 40
    ones, zeros = np.ones((H, W), np.uint8), np.zeros((H, W), np.uint8)
    pre, srt, f1 = orc.forward_view(*P, cam, cfg, mask=ones)
    assert f1["loss_bg"] == 0.0
    f0 = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=zeros)
    assert f0["loss_bg"] == pytest.approx(f0["alpha"].mean(), rel=1e-12)
    m = sc.mask(0)
    fm = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=m)
    assert fm["loss_bg"] == pytest.approx((fm["alpha"] * (1 - m)).sum() / (H * W), rel=1e-12)
    fmc = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=1 - m)
    assert fm["loss_bg"] + fmc["loss_bg"] == pytest.approx(f0["loss_bg"], rel=1e-12)  # linear in (1 - M)
    # only L_b active: dL/d opacity >= 0 everywhere ("penalizes Gaussian opacity where O is not present",
    # PAPER.md:101) and exactly 0 for surfels that only touch mask=1 pixels
    left = np.zeros((H, W), np.uint8)
    left[:, : W // 2] = 1
    g = orc.render_bwd(*P, pre, srt, cam, cfg, mask=left)
    assert np.all(g["d_opacity"] >= 0.0) and g["d_opacity"].max() > 0
    only_left = (pre["visible"] == 1) & (pre["rect"][:, 2] < W // 2)
    assert only_left.any() and np.all(g["d_opacity"][only_left] == 0.0)
    # the fused gradient equals feeding gA = gamma (1-M)/(HW) explicitly
    cfg0 = orc.default_config(sh_degree=1, gamma_bg=0.0)
    g2 = orc.render_bwd(*P, pre, srt, cam, cfg0, mask=left, gA=0.5 * (1.0 - left) / (H * W))
    for k in (k for k in g if k != "_abs"):
        assert np.allclose(g[k], g2[k], rtol=1e-12, atol=1e-18), k


# ---------------------------------------------------------------------------------------------
# O2/O3: keys, order, ranges -- brute force on a small input
# ---------------------------------------------------------------------------------------------
def test_bin_sort_matches_bruteforce_tuple_sort():
    sc = sg.random_scene(300, 96, 80, 70.0, seed=5, sh_degree=0, scale_lo=0.02, scale_hi=0.4)
    cam = orc.camera_from(sc.cameras[0])
    cfg = orc.default_config(sh_degree=0)
    pos = sc.pos.copy()
    pos[10:20, 2] = pos[10, 2]  # equal depths: ties must break by surfel id
    pre = orc.preprocess(pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    tx, ty = orc.tiles_of(cam, cfg)
    assert (tx, ty) == (6, 5)
    tuples = []
    for j in range(sc.n):
        if not pre["visible"][j]:
            continue
        x0, y0, x1, y1 = pre["rect"][j]
        for tyy in range(y0 // 16, y1 // 16 + 1):
            for txx in range(x0 // 16, x1 // 16 + 1):
                tuples.append((tyy * tx + txx, int(pre["depth_bits"][j]), j))
    tuples.sort()
    assert srt["K"] == len(tuples) == int(pre["tiles_touched"].sum())
    assert [t[2] for t in tuples] == list(srt["ids"])
    assert [(t[0] << 32) | t[1] for t in tuples] == [int(k) for k in srt["keys"]]
    r = srt["ranges"]
    assert r[0, 0] == 0 and r[-1, 1] == srt["K"] and np.all(r[1:, 0] == r[:-1, 1]) and np.all(r[:, 0] <= r[:, 1])
    for t in range(tx * ty):
        assert all(tt[0] == t for tt in tuples[r[t, 0]:r[t, 1]])


# ---------------------------------------------------------------------------------------------
# S7: bounding box is conservative and tight (sampled ellipse boundary, raw parameters, fp64)
# ---------------------------------------------------------------------------------------------
def test_bbox_contains_projected_ellipse_and_is_tight():
    sc = sg.random_scene(400, 200, 160, 150.0, seed=7, sh_degree=0, scale_lo=0.02, scale_hi=0.3)
    cam = orc.camera_from(sc.cameras[0])
    cfg = orc.default_config(sh_degree=0)
    pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
    th = np.linspace(0, 2 * math.pi, 4001)
    checked = 0
    for j in range(sc.n):
        w, x, y, z = sc.quat[j].astype(np.float64)
        tu = np.array([1 - 2 * (y * y + z * z), 2 * (x * y + w * z), 2 * (x * z - w * y)])
        tv = np.array([2 * (x * y - w * z), 1 - 2 * (x * x + z * z), 2 * (y * z + w * x)])
        o = float(sc.opacity[j])
        if o < 1 / 255 or sc.pos[j, 2] <= 0.2:
            assert not pre["visible"][j]
            continue
        rc = min(9.0, 2 * math.log(o * 255))
        r = math.sqrt(rc)
        pts = sc.pos[j].astype(np.float64)[None] + r * np.cos(th)[:, None] * sc.scale[j, 0] * tu[None] + r * np.sin(th)[:, None] * sc.scale[j, 1] * tv[None]
        if pts[:, 2].min() <= 1e-3:
            continue
        xs = 150.0 * pts[:, 0] / pts[:, 2] + 99.5
        ys = 150.0 * pts[:, 1] / pts[:, 2] + 79.5
        c = np.array([150.0 * sc.pos[j, 0] / sc.pos[j, 2] + 99.5, 150.0 * sc.pos[j, 1] / sc.pos[j, 2] + 79.5])
        rf = math.sqrt(0.5 * rc)
        lo = np.array([min(xs.min(), c[0] - rf), min(ys.min(), c[1] - rf)])
        hi = np.array([max(xs.max(), c[0] + rf), max(ys.max(), c[1] + rf)])
        exp = [max(0, math.ceil(lo[0])), max(0, math.ceil(lo[1])), min(199, math.floor(hi[0])), min(159, math.floor(hi[1]))]
        if exp[0] > exp[2] or exp[1] > exp[3]:
            continue
        if not pre["visible"][j]:
            continue
        got = list(pre["rect"][j])
        # conservative: never smaller than the sampled extent; tight: at most one pixel larger (sampling / fp32 slack)
        assert got[0] <= exp[0] and got[1] <= exp[1] and got[2] >= exp[2] and got[3] >= exp[3], (j, got, exp)
        assert got[0] >= exp[0] - 1 and got[1] >= exp[1] - 1 and got[2] <= exp[2] + 1 and got[3] <= exp[3] + 1, (j, got, exp)
        checked += 1
    assert checked > 150


def test_bbox_fp32_is_conservative_at_config2_scale():
    """S7 / reading R-bbox at the size where fp32 matters (800x600, f = 900, 140 k visible surfels): the integer rect
    produced by the fp32 sequence must contain the exact (fp64, from the raw parameters) extent of the rho_cut ellipse
    and of the filter disc, and exceed it by at most one pixel.  The extent is the closed form of the projected
    conic's axis-aligned tangents (the formula the sampled-boundary test above pins), evaluated in fp64 where its
    cancellation is harmless.  Regression: surfel 97584 of config 2 / view 3, whose rect under the uncentred fp32
    formula started at row 538 although rho(450, 537) = 8.5708 < rho_cut = 8.5892."""
    sc = sg.make_scene("config2")
    camn = sc.cameras[3]
    cam = orc.camera_from(camn)
    cfg = orc.default_config(sh_degree=3)
    pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
    vis = pre["visible"] == 1
    q = sc.quat.astype(np.float64)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    tu = np.stack([1 - 2 * (y * y + z * z), 2 * (x * y + w * z), 2 * (x * z - w * y)], 1)
    tv = np.stack([2 * (x * y - w * z), 1 - 2 * (x * x + z * z), 2 * (y * z + w * x)], 1)
    V = camn.view.astype(np.float64)
    R, t = V[:3, :3], V[:3, 3]
    pc = sc.pos.astype(np.float64) @ R.T + t
    cu = (tu @ R.T) * sc.scale[:, 0:1].astype(np.float64)
    cv = (tv @ R.T) * sc.scale[:, 1:2].astype(np.float64)
    o = sc.opacity.astype(np.float64)
    rc = np.minimum(9.0, 2 * np.log(np.maximum(o, 1e-12) * 255.0))
    rf = np.sqrt(0.5 * rc)
    f, off = 900.0, (camn.cx - 0.5, camn.cy - 0.5)
    lo, hi = np.zeros((sc.n, 2)), np.zeros((sc.n, 2))
    tt = np.stack([rc, rc, -np.ones_like(rc)], 1)
    m2 = np.stack([cu[:, 2], cv[:, 2], pc[:, 2]], 1)
    a = (tt * m2 * m2).sum(1)
    for r in (0, 1):
        mr = f * np.stack([cu[:, r], cv[:, r], pc[:, r]], 1)  # pixel coordinates relative to the principal point
        b, c = (tt * mr * m2).sum(1), (tt * mr * mr).sum(1)
        ctr = b / a
        half = np.sqrt(np.maximum(0.0, ctr * ctr - c / a))
        c2 = f * pc[:, r] / pc[:, 2]
        lo[:, r] = np.minimum(ctr - half, c2 - rf) + off[r]
        hi[:, r] = np.maximum(ctr + half, c2 + rf) + off[r]
    WH = (camn.width, camn.height)
    sel = vis & (a < 0)
    assert sel.sum() > 100_000
    rect = pre["rect"][sel].astype(np.int64)
    for r in (0, 1):
        e0 = np.clip(np.ceil(lo[sel, r]), 0, WH[r] - 1)
        e1 = np.clip(np.floor(hi[sel, r]), 0, WH[r] - 1)
        assert np.all(rect[:, r] <= e0) and np.all(rect[:, 2 + r] >= e1), "rect misses a pixel of the exact extent"
        assert np.all(rect[:, r] >= e0 - 1) and np.all(rect[:, 2 + r] <= e1 + 1), "rect more than one pixel loose"
    # surfels the fp32 path culled must have an exact extent that misses the image or is empty
    culled = (~vis) & (a < 0) & (pc[:, 2] > 0.2) & (o >= 1 / 255)
    e0x, e1x = np.ceil(lo[culled, 0]), np.floor(hi[culled, 0])
    e0y, e1y = np.ceil(lo[culled, 1]), np.floor(hi[culled, 1])
    assert np.all((e1x < 0) | (e0x > WH[0] - 1) | (e0x > e1x) | (e1y < 0) | (e0y > WH[1] - 1) | (e0y > e1y))
    assert pre["rect"][97584][1] <= 537 <= pre["rect"][97584][3]


def test_bruteforce_equals_tiled_config2_full_size_window():
    """BF == TILED on a window of the full 200 k-surfel config 2 (view 3) that contains pixel (450, 537), where the
    uncentred fp32 bbox used to drop a contributing pair (alpha jump 1/255 => 5e-4 in colour)."""
    sc = sg.make_scene("config2")
    cam = orc.camera_from(sc.cameras[3])
    cfg = orc.default_config(sh_degree=3)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    win = (448, 528, 464, 544)
    pre = orc.preprocess(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    fw = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=None, window=win)
    bf = orc.bf_render(*P, cam, cfg, mask=None, window=win, want_stats=False)
    x0, y0, x1, y1 = win
    ok = fw["fragile"][y0:y1, x0:x1] == 0
    assert ok[537 - y0, 450 - x0]
    for k in ("color", "alpha", "normal"):
        err = np.abs(fw[k][..., y0:y1, x0:x1] - bf[k][..., y0:y1, x0:x1])
        assert (err * ok).max() < 5e-5, (k, (err * ok).max())


# ---------------------------------------------------------------------------------------------
# BF (fp64, explicit ray-plane, exhaustive per-pixel sort, no tiles) == TILED
# ---------------------------------------------------------------------------------------------
def _compare_bf_tiled(sc, view, cfg, tol=5e-5):
    # tol: the TILED path evaluates from the fp32 record M (Appendix A), BF from the raw parameters in fp64.  For
    # surfels seen almost edge-on the 6e-8 rounding of M is amplified (cos of incidence 0.03 -> ~5e-6 in alpha,
    # 0.0025 -> 1.6e-4).  Pixels whose first-order fp32 error estimate exceeds 2e-5 carry fragile bit 1 and are
    # excluded like the decision-margin ones; the rest must agree to a few times that.
    cam = orc.camera_from(sc.cameras[view])
    m = sc.mask(view)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    pre, srt, fw = orc.forward_view(*P, cam, cfg, mask=m)
    bf = orc.bf_render(*P, cam, cfg, mask=m)
    ok = fw["fragile"] == 0
    assert ok.mean() > 0.995
    for k in ("color", "alpha", "depth", "normal", "origin", "m1", "m2"):
        scale = 1.0 if k not in ("depth", "origin") else np.maximum(1.0, np.abs(bf[k]))
        err = np.abs(fw[k] - bf[k]) / scale
        # M is an fp32 record (~1e-7 relative); the hit depth of oblique surfels amplifies that most
        assert (err * ok).max() < (tol if k not in ("depth", "origin", "m1", "m2") else 10 * tol), (k, (err * ok).max())
    untouched = fw["fragile_touch"] == 0
    assert np.array_equal(fw["vis_count"][untouched], bf["vis_count"][untouched])
    assert np.allclose(fw["contrib_sum"][untouched], bf["contrib_sum"][untouched], rtol=1e-4, atol=1e-6)
    if ok.all():
        assert fw["loss_bg"] == pytest.approx(bf["loss_bg"], abs=1e-7)
    return fw, bf


def test_bruteforce_equals_tiled_random_scenes():
    for seed in (1, 2, 3):
        sc = sg.random_scene(60, 56, 40, 50.0, seed=seed, sh_degree=3)
        _compare_bf_tiled(sc, 0, orc.default_config(sh_degree=3, bg=(0.3, 0.1, 0.2)))


def test_bruteforce_equals_tiled_config1_view0():
    sc = sg.make_scene("config1")
    fw, bf = _compare_bf_tiled(sc, 0, orc.default_config(sh_degree=0))
    assert fw["alpha"].max() > 0.9 and (fw["n_contrib"] > 0).mean() > 0.3


# ---------------------------------------------------------------------------------------------
# O7: analytic backward == central finite differences of the BF forward (fp64)
# ---------------------------------------------------------------------------------------------
def _fd_check(seed, n, W, H, f, sh_degree, **kw):
    sc = sg.random_scene(n, W, H, f, seed=seed, sh_degree=sh_degree, **kw)
    cam = orc.camera_from(sc.cameras[0])
    cfg = orc.default_config(sh_degree=sh_degree, bg=(0.2, 0.4, 0.1))
    m = sc.mask(0)
    rng = np.random.default_rng(seed + 100)
    wC, wA, wD, wN = rng.normal(size=(3, H, W)), rng.normal(size=(H, W)), rng.normal(size=(H, W)), rng.normal(size=(3, H, W))
    wX = rng.normal(size=(H, W))  # per-pixel weight of the pairwise depth distortion A m2 - m1^2 (reading R-moments)
    params = dict(pos=sc.pos.astype(np.float64), scale=sc.scale.astype(np.float64), quat=sc.quat.astype(np.float64),
                  opacity=sc.opacity.astype(np.float64), sh=sc.sh.astype(np.float64))

    def loss(p):
        r = orc.bf_render(p["pos"], p["scale"], p["quat"], p["opacity"], p["sh"], cam, cfg, mask=m, want_stats=False)
        L = (wC * r["color"]).sum() + (wA * r["alpha"]).sum() + (wD * r["depth"]).sum() + (wN * r["normal"]).sum()
        L += (wX * (r["alpha"] * r["m2"] - r["m1"] ** 2)).sum()  # invariant to the moments' origin, so FD sees no kink from it
        return L + cfg.gamma_bg * r["loss_bg"], r["n_blended"]

    pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    fw0 = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=m, want_fragile=False)
    # chain rule of the distortion term through the maps: d(A m2 - m1^2) = m2 dA - 2 m1 dm1 + A dm2
    g = orc.render_bwd(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, pre, srt, cam, cfg, mask=m, gC=wC, gA=wA + wX * fw0["m2"], gD=wD, gN=wN,
                       gM1=-2.0 * wX * fw0["m1"], gM2=wX * fw0["alpha"])
    names = dict(pos="d_pos", scale="d_scale", quat="d_quat", opacity="d_opacity", sh="d_sh")
    nb = (sh_degree + 1) ** 2
    checked = skipped = 0
    worst = 0.0
    for key, gname in names.items():
        arr = params[key]
        flat = arr.reshape(arr.shape[0], -1)
        for j in range(arr.shape[0]):
            for c in range(flat.shape[1]):
                if key == "sh" and c // 3 >= nb:
                    assert g[gname].reshape(n, -1)[j, c] == 0.0
                    continue
                h = 1e-6 * max(1.0, abs(flat[j, c]))
                old = flat[j, c]
                flat[j, c] = old + h
                Lp, np_ = loss(params)
                flat[j, c] = old - h
                Lm, nm_ = loss(params)
                flat[j, c] = old
                if not np.array_equal(np_, nm_):  # a discontinuity (cut-off / stop) was crossed: FD is meaningless here
                    skipped += 1
                    continue
                fd = (Lp - Lm) / (2 * h)
                an = g[gname].reshape(n, -1)[j, c]
                # relative to the size of this surfel's gradient block (small entries are sums of cancelling terms and
                # inherit the fp32-record vs fp64-parameter difference of the two forward paths)
                err = abs(fd - an) / max(1e-3, abs(fd), np.abs(g[gname].reshape(n, -1)[j]).max())
                worst = max(worst, err)
                assert err < 2e-4, (key, j, c, fd, an)
                checked += 1
    assert checked > 20 * skipped and checked > 100
    return worst


def test_backward_matches_finite_differences_sh3():
    _fd_check(seed=21, n=6, W=20, H=16, f=22.0, sh_degree=3)


def test_backward_matches_finite_differences_small_surfels_filter_active():
    # sub-pixel surfels: the screen-space filter branch (S8) and its gradient to the centre are exercised
    _fd_check(seed=22, n=8, W=16, H=16, f=18.0, sh_degree=1, scale_lo=0.01, scale_hi=0.08)


def test_d_center2d_reading_r_c2d():
    """DESIGN.md reading R-c2d (the densification statistic): d_center2d = dL/d(projected centre) at fixed view
    depth = M22 (dL/dM02, dL/dM12).  Pins: (i) central differences on the BF forward of a shift of the surfel centre by
    delta pixels in the image plane at fixed depth (p_c += (delta z/fx, 0, 0) resp. (0, delta z/fy, 0), mapped back to the
    world) on a scene of sub-pixel surfels, where the filter branch (S8) and its -4 d g_rho term are active; SH degree 0,
    so the colour does not move with the position; (ii) identity camera: p_c = p, M02 = fx p_x + ox p_z, so
    d_center2d = (z/fx, z/fy) * d_pos[:, :2] exactly -- d_pos itself is pinned by the finite-difference tests above."""
    n, W, H, f = 8, 16, 16, 18.0
    sc = sg.random_scene(n, W, H, f, seed=22, sh_degree=0, scale_lo=0.01, scale_hi=0.08)
    camn = sc.cameras[0]
    cam = orc.camera_from(camn)
    cfg = orc.default_config(sh_degree=0, bg=(0.2, 0.4, 0.1))
    m = sc.mask(0)
    rng = np.random.default_rng(5)
    wC, wA, wD, wN = rng.normal(size=(3, H, W)), rng.normal(size=(H, W)), rng.normal(size=(H, W)), rng.normal(size=(3, H, W))
    pos64 = sc.pos.astype(np.float64)
    others = [a.astype(np.float64) for a in (sc.scale, sc.quat, sc.opacity, sc.sh)]

    def loss(pos):
        r = orc.bf_render(pos, *others, cam, cfg, mask=m, want_stats=False)
        return ((wC * r["color"]).sum() + (wA * r["alpha"]).sum() + (wD * r["depth"]).sum() + (wN * r["normal"]).sum()
                + cfg.gamma_bg * r["loss_bg"]), r["n_blended"]

    pre = orc.preprocess(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    fw = orc.render_fwd(pre, srt, sc.opacity, cam, cfg, mask=m, want_fragile=False)
    g = orc.render_bwd(sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh, pre, srt, cam, cfg, mask=m, gC=wC, gA=wA, gD=wD, gN=wN)
    V = np.asarray(camn.view, np.float64).reshape(4, 4)
    Rwc = V[:3, :3]
    checked = 0
    filter_seen = False
    for j in range(n):
        if not pre["visible"][j] or fw["vis_count"][j] == 0:
            assert np.all(g["d_center2d"][j] == 0.0)
            continue
        z = float((V[:3, :3] @ pos64[j] + V[:3, 3])[2])
        for ax, fl in ((0, camn.fx), (1, camn.fy)):
            h = 1e-5
            e = np.zeros(3); e[ax] = z / fl          # one pixel along the image axis at depth z, in camera coordinates
            dw = Rwc.T @ e                            # ... in world coordinates
            pp, pm = pos64.copy(), pos64.copy()
            pp[j] += h * dw; pm[j] -= h * dw
            Lp, np_ = loss(pp); Lm, nm_ = loss(pm)
            if not np.array_equal(np_, nm_):
                continue
            fd = (Lp - Lm) / (2 * h)
            an = g["d_center2d"][j, ax]
            assert abs(fd - an) <= 2e-4 * max(1e-3, abs(fd), np.abs(g["d_center2d"][j]).max()), (j, ax, fd, an)
            checked += 1
        # the filter term was active for this surfel somewhere: sigma_px = f s / z below sigma_f for the small ones
        filter_seen |= bool(f * sc.scale[j].min() / z < 0.7)
    assert checked >= 8 and filter_seen
    # (ii) identity camera
    s = stack(one_surfel((0.13, -0.07, 2.0), (0.1, 0.06), quat=(0.9, 0.1, 0.3, 0.2)), one_surfel((-0.2, 0.1, 2.5), (0.004, 0.004)))
    s = (s[0], s[1], s[2] / np.linalg.norm(s[2], axis=1, keepdims=True).astype(np.float32), s[3], s[4])
    cam = ident_cam(24, 20, 30.0)
    cfg = orc.default_config(sh_degree=0)
    pre = orc.preprocess(*s, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    rng = np.random.default_rng(6)
    g = orc.render_bwd(*s, pre, srt, cam, cfg, gC=rng.normal(size=(3, 20, 24)), gA=rng.normal(size=(20, 24)), gD=rng.normal(size=(20, 24)))
    assert np.abs(g["d_center2d"]).min() > 0
    for j in range(2):
        z = float(s[0][j, 2])
        assert np.allclose(g["d_center2d"][j], z / 30.0 * g["d_pos"][j, :2], rtol=1e-12, atol=0)


def test_backward_sums_of_absolute_terms_bound_the_gradients():
    """The conditioning sums the gradient tolerance uses (orc_render_bwd abs_*) are what they claim:
    every entry satisfies |g| <= sum|terms| (triangle inequality through the whole chain), the sums are positively
    homogeneous in the upstream gradients (x -2 doubles them), and for a non-negative upstream on colour only the colour
    chain has no cancellation at all: sum|terms| == |d_sh| exactly."""
    sc = sg.random_scene(40, 48, 40, 40.0, seed=31, sh_degree=2)
    cam = orc.camera_from(sc.cameras[0])
    cfg = orc.default_config(sh_degree=2)
    P = (sc.pos, sc.scale, sc.quat, sc.opacity, sc.sh)
    pre = orc.preprocess(*P, cam, cfg)
    srt = orc.bin_sort(pre, cam, cfg)
    rng = np.random.default_rng(2)
    gC, gA, gD, gN = rng.normal(size=(3, 40, 48)), rng.normal(size=(40, 48)), rng.normal(size=(40, 48)), rng.normal(size=(3, 40, 48))
    g = orc.render_bwd(*P, pre, srt, cam, cfg, gC=gC, gA=gA, gD=gD, gN=gN)
    g2 = orc.render_bwd(*P, pre, srt, cam, cfg, gC=-2 * gC, gA=-2 * gA, gD=-2 * gD, gN=-2 * gN)
    assert (g["d_pos"] != 0).sum() > 50
    for k in ("d_pos", "d_scale", "d_quat", "d_opacity", "d_sh", "d_center2d"):
        a = g["_abs"][k].reshape(g[k].shape)
        assert np.all(np.abs(g[k]) <= a * (1 + 1e-12) + 1e-300), k
        assert np.allclose(g2["_abs"][k].reshape(a.shape), 2 * a, rtol=1e-12, atol=0), k
        assert np.allclose(g2[k], -2 * g[k], rtol=1e-9, atol=1e-14), k
    gp = orc.render_bwd(*P, pre, srt, cam, cfg, gC=np.abs(gC))
    sh0 = gp["d_sh"][:, 0, :]  # Y0 > 0: d_sh[0] = Y0 * sum of non-negative terms
    assert np.allclose(gp["_abs"]["d_sh"][:, 0, :], np.abs(sh0), rtol=1e-12, atol=0) and (sh0 > 0).sum() > 20


def test_prune_and_compaction_definition():
    rng = np.random.default_rng(3)
    n = 1000
    vis = rng.integers(0, 3, n).astype(np.uint32)
    cs = np.where(vis > 0, rng.uniform(0.0, 1.0, n), 0.0).astype(np.float32)
    op = rng.uniform(0, 1, n).astype(np.float32)
    pr = orc.prune(vis, cs, op)
    assert np.array_equal(pr["prune_mask"], (vis == 0).astype(np.uint8))  # tau = 0, o_min = 0: the paper's boolean rule
    keep = [j for j in range(n) if vis[j] > 0]
    assert pr["n_out"] == len(keep) and [int(pr["remap"][j]) for j in keep] == list(range(len(keep)))
    pr2 = orc.prune(vis, cs, op, tau=0.25, min_opacity=0.1)
    assert np.array_equal(pr2["prune_mask"], ((vis == 0) | (cs <= 0.25) | (op < 0.1)).astype(np.uint8))
    data = dict(a=rng.normal(size=(n, 3)).astype(np.float32))
    assert np.array_equal(orc.compact(data, pr["prune_mask"])["a"], np.stack([data["a"][j] for j in keep]))
