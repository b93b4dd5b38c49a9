"""Pins of oracle/densify.py (clone / split of the adaptive density control; reading R-densify) against
a by-hand example, count and ordering invariants, and a library rotation routine for the tangent frame."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

from oracle import densify as dn


def random_surfels(n, seed):
    rng = np.random.default_rng(seed)
    q = rng.normal(size=(n, 4)); q /= np.linalg.norm(q, axis=1, keepdims=True)
    return (rng.normal(size=(n, 3)).astype(np.float32), np.exp(rng.uniform(np.log(0.003), np.log(0.05), (n, 2))).astype(np.float32),
            q.astype(np.float32), rng.uniform(0.05, 0.95, n).astype(np.float32), rng.normal(size=(n, 16, 3)).astype(np.float32))


def test_by_hand_example_keep_clone_split():
    # identity rotation: t_u = x, t_v = y
    pos = np.array([[0, 0, 1], [1, 0, 1], [2, 0, 1], [3, 0, 1]], np.float32)
    scale = np.array([[0.01, 0.02], [0.01, 0.02], [0.2, 0.1], [0.2, 0.1]], np.float32)
    quat = np.tile(np.array([1, 0, 0, 0], np.float32), (4, 1))
    opacity = np.array([0.1, 0.2, 0.3, 0.4], np.float32)
    sh = np.arange(4 * 48, dtype=np.float32).reshape(4, 16, 3)
    grad = np.array([1e-4 * 4, 9e-4, 6e-4 * 3, 1e-4], np.float32)   # sums over the views of the interval
    den = np.array([4, 1, 3, 0], np.uint32)                          # averages 1e-4, 9e-4, 6e-4, (never in view -> 0)
    xi = np.zeros((4, 2, 2), np.float32)
    xi[2] = [[1.0, -2.0], [0.5, 0.25]]
    r = dn.densify(pos, scale, quat, opacity, sh, grad, den, 2e-4, 0.05, xi)
    # surfel 0: below the gradient threshold -> kept; 1: selected and small -> kept + cloned; 2: selected and large -> split;
    # 3: large but never selected -> kept
    assert list(r["cls"]) == [0, 1, 2, 0]
    assert (r["n_out"], r["n_keep"], r["n_clone"], r["n_split"]) == (6, 3, 1, 1)
    assert list(r["src"]) == [0, 1, 3, 1, 2, 2]
    assert np.allclose(r["pos"][:4], pos[[0, 1, 3, 1]])
    assert np.allclose(r["pos"][4], [2 + 0.2 * 1.0, 0 + 0.1 * -2.0, 1]) and np.allclose(r["pos"][5], [2 + 0.2 * 0.5, 0.1 * 0.25, 1])
    assert np.allclose(r["scale"][4:], np.array([0.2, 0.1]) / 1.6) and np.allclose(r["scale"][:4], scale[[0, 1, 3, 1]])
    assert np.array_equal(r["opacity"], opacity[r["src"]]) and np.array_equal(r["sh"], sh[r["src"]]) and np.array_equal(r["quat"], quat[r["src"]])


def test_counts_order_and_copies_on_random_input():
    n = 5000
    P = random_surfels(n, 1)
    rng = np.random.default_rng(2)
    den = rng.integers(0, 5, n).astype(np.uint32)
    grad = (rng.uniform(0, 6e-4, n) * den).astype(np.float32)
    xi = rng.normal(size=(n, 2, 2)).astype(np.float32)
    r = dn.densify(*P, grad, den, 2e-4, 0.02, xi)
    cls = r["cls"]
    assert r["n_out"] == n - r["n_split"] + r["n_clone"] + 2 * r["n_split"] == len(r["src"])
    assert r["n_keep"] == int((cls != 2).sum()) and r["n_clone"] == int((cls == 1).sum()) and r["n_split"] == int((cls == 2).sum())
    assert min(r["n_clone"], r["n_split"], r["n_keep"]) > 100
    k, c = r["n_keep"], r["n_clone"]
    assert np.array_equal(r["src"][:k], np.nonzero(cls != 2)[0])            # survivors, ascending id
    assert np.array_equal(r["src"][k:k + c], np.nonzero(cls == 1)[0])       # clones, ascending id
    assert np.array_equal(r["src"][k + c:], np.repeat(np.nonzero(cls == 2)[0], 2))  # two children per split surfel
    for name, arr in zip(("pos", "scale", "quat", "opacity", "sh"), P):
        assert np.array_equal(r[name][:k + c].astype(np.float32), arr[r["src"][:k + c]]), name
    # never-selected when never in view, whatever the accumulated value
    assert np.all(cls[den == 0] == 0)
    # selection rule itself, in fp32
    avg = np.where(den > 0, grad / np.maximum(den, 1).astype(np.float32), np.float32(0))
    assert np.array_equal(cls != 0, avg >= np.float32(2e-4))
    assert np.array_equal(cls == 2, (avg >= np.float32(2e-4)) & (P[1].max(1) > np.float32(0.02)))


def test_children_lie_in_the_tangent_plane_of_a_library_rotation():
    """Children are drawn in the surfel's own plane: (child - p) has no component along the normal, and its components along
    t_u, t_v are s_u xi_0, s_v xi_1 -- with the frame taken from scipy's quaternion-to-matrix routine (pins R(q))."""
    n = 400
    P = random_surfels(n, 3)
    xi = np.random.default_rng(4).normal(size=(n, 2, 2)).astype(np.float32)
    r = dn.densify(*P, np.ones(n, np.float32), np.ones(n, np.uint32), 2e-4, 0.0, xi)  # everything is split
    assert r["n_split"] == n and r["n_keep"] == 0
    q = P[2].astype(np.float64)
    Rm = Rotation.from_quat(np.stack([q[:, 1], q[:, 2], q[:, 3], q[:, 0]], 1)).as_matrix()  # scipy wants (x, y, z, w)
    for k in range(2):
        d = r["pos"][k::2] - P[0].astype(np.float64)
        local = np.einsum("nij,ni->nj", Rm, d)  # R^T d
        assert np.abs(local[:, 2]).max() < 1e-6
        assert np.allclose(local[:, 0], P[1][:, 0].astype(np.float64) * xi[:, k, 0], atol=1e-6)
        assert np.allclose(local[:, 1], P[1][:, 1].astype(np.float64) * xi[:, k, 1], atol=1e-6)
    # xi = 0: both children sit on the parent
    r0 = dn.densify(*P, np.ones(n, np.float32), np.ones(n, np.uint32), 2e-4, 0.0, np.zeros((n, 2, 2), np.float32))
    assert np.array_equal(r0["pos"].astype(np.float32), np.repeat(P[0], 2, 0))


def test_accumulate_adds_the_norm_only_where_in_frustum():
    ga, de = np.zeros(4), np.zeros(4, np.int64)
    g = np.array([[3, 4], [1, 0], [0, 0], [6, 8]], np.float32)
    dn.accumulate(ga, de, g, [1, 1, 1, 0], 2, 2)   # W/2 = H/2 = 1: the plain norm
    dn.accumulate(ga, de, g, [1, 0, 1, 0], 2, 2)
    assert list(ga) == [10.0, 1.0, 0.0, 0.0] and list(de) == [2, 1, 2, 0]
    # NDC units: pixel = ((ndc + 1) W - 1) / 2, so a unit gradient per pixel is W/2 per NDC unit along x, H/2 along y
    ga, de = np.zeros(2), np.zeros(2, np.int64)
    dn.accumulate(ga, de, np.array([[1, 0], [0, 1]], np.float32), [1, 1], 1600, 1200)
    assert list(ga) == [800.0, 600.0]
    dn.accumulate(ga, de, np.array([[3, 0], [3, 4]], np.float32), [0, 1], 8, 6)
    assert list(ga) == [800.0, 600.0 + 12.0 * 2 ** 0.5] or np.allclose(ga, [800.0, 600.0 + np.hypot(12.0, 12.0)])
