"""Pins of oracle/regularizers.py (depth distortion L_d and normal consistency L_n of Eq. 3; readings
R-moments / R-Ld / R-Ln) against definitions, closed forms and central finite differences."""
import math

import numpy as np
import pytest

from oracle import regularizers as rg

FX, FY, CX, CY = 40.0, 44.0, 12.0, 9.0


def smooth_maps(seed, H=18, W=24):
    rng = np.random.default_rng(seed)
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    A = 0.55 + 0.3 * np.sin(xs / 5.0) * np.cos(ys / 4.0)
    zbar = 2.0 + 0.2 * np.sin(xs / 3.0 + 0.3) + 0.15 * np.cos(ys / 2.5) + 0.01 * rng.normal(size=(H, W))
    D = A * zbar
    m1 = A * (0.05 + 0.03 * np.sin(xs / 4.0))            # sum w (z - c)
    m2 = A * (0.01 + 0.004 * rng.uniform(size=(H, W)))   # sum w (z - c)^2
    n = rng.normal(size=(3, H, W)) * 0.2 + np.array([0.1, -0.2, -0.9])[:, None, None]
    Nrm = A[None] * n
    return A, D, m1, m2, Nrm


def test_distortion_identity_against_the_double_sum():
    """R-Ld: sum_{i<j} w_i w_j (z_i - z_j)^2 == A m2 - m1^2 with A = sum w, m1 = sum w (z - c), m2 = sum w (z - c)^2, for any c."""
    rng = np.random.default_rng(0)
    for n in (1, 2, 5, 40):
        w = rng.uniform(0, 0.3, n)
        z = rng.uniform(0.5, 6.0, n)
        for c in (0.0, z[0], 17.0):
            A, m1, m2 = w.sum(), (w * (z - c)).sum(), (w * (z - c) ** 2).sum()
            assert rg.distortion_map(A, m1, m2) == pytest.approx(rg.distortion_bruteforce(w, z), rel=1e-10, abs=1e-12)
    # one layer: no distortion; two layers: w1 w2 (z1 - z2)^2
    assert rg.distortion_map(0.7, 0.0, 0.0) == 0.0  # origin = the layer's own depth
    assert rg.distortion_map(0.5 + 0.2, 0.2 * 3.0, 0.2 * 9.0) == pytest.approx(0.5 * 0.2 * 9.0, rel=1e-14)  # z = 1, 4; c = 1


def test_fronto_parallel_depth_gives_camera_facing_axis_normal():
    H, W = 10, 12
    A = np.full((H, W), 0.9)
    Nhat, _ = rg.depth_normal(A, A * 2.5, FX, FY, CX, CY)
    assert np.allclose(Nhat[:, 1:-1, 1:-1], np.array([0.0, 0.0, -1.0])[:, None, None], atol=1e-13)
    assert np.all(Nhat[:, 0, :] == 0) and np.all(Nhat[:, :, -1] == 0)  # one-pixel border


def test_planar_depth_map_reproduces_the_plane_normal_and_zero_loss_inside():
    """Back-projected points of a planar depth map lie on the plane, so their differences do: Nhat == plane normal exactly
    (no discretisation error), and with Nrm = A n the per-pixel term A - Nrm . Nhat vanishes in the interior."""
    H, W = 14, 16
    n = np.array([0.3, -0.2, -0.9]); n /= np.linalg.norm(n)
    d = n @ np.array([0.1, 0.05, 3.0])  # plane through (0.1, 0.05, 3)
    ys, xs = np.mgrid[0:H, 0:W].astype(np.float64)
    r = np.stack([(xs - (CX - 0.5)) / FX, (ys - (CY - 0.5)) / FY, np.ones((H, W))])
    zbar = d / (n[:, None, None] * r).sum(0)
    A = np.full((H, W), 0.8)
    Nrm = A[None] * n[:, None, None]
    out = rg.regularizers(A, A * zbar, np.zeros((H, W)), np.zeros((H, W)), Nrm, FX, FY, CX, CY)
    assert np.abs(out["Nhat"][:, 1:-1, 1:-1] - n[:, None, None]).max() < 1e-12
    border = H * W - (H - 2) * (W - 2)
    assert out["L_n"] == pytest.approx(0.8 * border / (H * W), abs=1e-12)  # border pixels have Nhat = 0: term = A
    assert out["L_d"] == 0.0  # a single layer per pixel: both centred moments vanish


def test_pixels_without_surface_have_no_normal():
    A, D, m1, m2, Nrm = smooth_maps(1)
    A2 = A.copy(); A2[5, 7] = 0.0
    Nhat, t = rg.depth_normal(A2, D, FX, FY, CX, CY)
    for (y, x) in ((5, 7), (5, 6), (5, 8), (4, 7), (6, 7)):
        assert np.all(Nhat[:, y, x] == 0.0)
    assert np.abs(Nhat[:, 8, 12]).sum() > 0


@pytest.mark.parametrize("w_d,w_n", [(1.0, 0.0), (0.0, 1.0), (3.0, 0.5)])
def test_gradients_match_central_finite_differences(w_d, w_n):
    A, D, m1, m2, Nrm = smooth_maps(2)
    out = rg.regularizers(A, D, m1, m2, Nrm, FX, FY, CX, CY, w_d=w_d, w_n=w_n)

    def L(A_, D_, m1_, m2_, N_):
        o = rg.regularizers(A_, D_, m1_, m2_, N_, FX, FY, CX, CY)
        return w_d * o["L_d"] + w_n * o["L_n"]

    rng = np.random.default_rng(3)
    h = 1e-6
    scale = {k: np.abs(out[k]).max() + 1e-30 for k in ("gA", "gD", "gM1", "gM2", "gN")}
    for _ in range(30):
        y, x = int(rng.integers(0, A.shape[0])), int(rng.integers(0, A.shape[1]))
        for name, idx in (("gA", (y, x)), ("gD", (y, x)), ("gM1", (y, x)), ("gM2", (y, x)), ("gN", (int(rng.integers(0, 3)), y, x))):
            maps = dict(gA=A, gD=D, gM1=m1, gM2=m2, gN=Nrm)
            p, m = {k: v.copy() for k, v in maps.items()}, {k: v.copy() for k, v in maps.items()}
            p[name][idx] += h; m[name][idx] -= h
            fd = (L(p["gA"], p["gD"], p["gM1"], p["gM2"], p["gN"]) - L(m["gA"], m["gD"], m["gM1"], m["gM2"], m["gN"])) / (2 * h)
            assert abs(out[name][idx] - fd) <= 1e-6 * scale[name] + 1e-5 * abs(fd), (name, idx, out[name][idx], fd)
