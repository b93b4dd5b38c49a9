"""Seeded synthetic scene generator (shared INPUT generator only).

This module produces the inputs both the CPU oracle (``oracle/``) and the CUDA
library consume: surfel parameter arrays, pinhole cameras and object masks for
the five workloads of ``BASELINE.json:configs``.
It holds none of the method's arithmetic (no projection, no blending, no SH
evaluation, no sorting) and imports neither the oracle nor the CUDA binding.

The scenes stand in for the paper's DTU / Mip-NeRF360 multi-view object
captures (§5.2): same view counts (49 / 64), image sizes
(800x600 .. 1600x1200), surfel counts (0.1 M .. 4 M) and an object that is
surrounded by background geometry, with a binary object mask per view
(PAPER.md:79, 97).

Conventions (Appendix B of SURVEY.md): world is right handed with up = +z;
camera looks down +z with x right, y down; ``view`` is the world->camera 4x4
row-major matrix; principal point (W/2, H/2); quaternions are (w, x, y, z),
unit length, chosen with w >= 0; all parameters are *activated* values.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Dict, List, Optional

import numpy as np

SH_Y0 = 0.5 * math.sqrt(1.0 / math.pi)  # only used to place a base colour into the DC coefficient


@dataclasses.dataclass
class Camera:
    view: np.ndarray  # [4,4] float32 world->camera
    fx: float
    fy: float
    cx: float
    cy: float
    width: int
    height: int

    @property
    def eye(self) -> np.ndarray:
        R = self.view[:3, :3].astype(np.float64)
        t = self.view[:3, 3].astype(np.float64)
        return -R.T @ t


@dataclasses.dataclass
class Scene:
    name: str
    seed: int
    pos: np.ndarray  # [N,3] f32
    scale: np.ndarray  # [N,2] f32
    quat: np.ndarray  # [N,4] f32 (w,x,y,z)
    opacity: np.ndarray  # [N] f32
    sh: np.ndarray  # [N,16,3] f32
    sh_degree: int
    cameras: List[Camera]
    group: np.ndarray  # [N] u8: 0 = object surface, 1 = background, 2 = interior (config 4)
    mask_fn: Callable[[Camera], np.ndarray]  # -> [H,W] u8, 1 = object

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])

    def mask(self, view_index: int) -> np.ndarray:
        return self.mask_fn(self.cameras[view_index])

    def perturbed(self, sigma: float = 0.01, seed_offset: int = 1000) -> "Scene":
        """Copy with +N(0, sigma) on positions, base colours (DC) and opacities
        (BASELINE.json config 1: targets are rendered from this copy)."""
        rng = np.random.Generator(np.random.PCG64(self.seed + seed_offset))
        pos = self.pos + rng.normal(0.0, sigma, self.pos.shape).astype(np.float32)
        sh = self.sh.copy()
        sh[:, 0, :] += (rng.normal(0.0, sigma, (self.n, 3)) / SH_Y0).astype(np.float32)
        op = np.clip(self.opacity + rng.normal(0.0, sigma, self.n).astype(np.float32), 1e-4, 1.0 - 1e-4)
        return dataclasses.replace(self, pos=pos.astype(np.float32), sh=sh, opacity=op.astype(np.float32))


# ----------------------------------------------------------------------------
# helpers: rotations, cameras
# ----------------------------------------------------------------------------

def _normalize(v: np.ndarray) -> np.ndarray:
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def quat_from_frame(tu: np.ndarray, tv: np.ndarray, tw: np.ndarray) -> np.ndarray:
    """Unit quaternion (w,x,y,z), w >= 0, of the rotation with columns tu, tv, tw (vectorised)."""
    m00, m10, m20 = tu[:, 0], tu[:, 1], tu[:, 2]
    m01, m11, m21 = tv[:, 0], tv[:, 1], tv[:, 2]
    m02, m12, m22 = tw[:, 0], tw[:, 1], tw[:, 2]
    n = tu.shape[0]
    q = np.empty((n, 4), np.float64)
    tr = m00 + m11 + m22
    # four branches of the standard matrix->quaternion conversion
    c0 = tr > 0
    c1 = (~c0) & (m00 >= m11) & (m00 >= m22)
    c2 = (~c0) & (~c1) & (m11 >= m22)
    c3 = (~c0) & (~c1) & (~c2)
    s = np.sqrt(np.maximum(tr[c0] + 1.0, 1e-30)) * 2
    q[c0] = np.stack([0.25 * s, (m21[c0] - m12[c0]) / s, (m02[c0] - m20[c0]) / s, (m10[c0] - m01[c0]) / s], 1)
    s = np.sqrt(np.maximum(1.0 + m00[c1] - m11[c1] - m22[c1], 1e-30)) * 2
    q[c1] = np.stack([(m21[c1] - m12[c1]) / s, 0.25 * s, (m01[c1] + m10[c1]) / s, (m02[c1] + m20[c1]) / s], 1)
    s = np.sqrt(np.maximum(1.0 + m11[c2] - m00[c2] - m22[c2], 1e-30)) * 2
    q[c2] = np.stack([(m02[c2] - m20[c2]) / s, (m01[c2] + m10[c2]) / s, 0.25 * s, (m12[c2] + m21[c2]) / s], 1)
    s = np.sqrt(np.maximum(1.0 + m22[c3] - m00[c3] - m11[c3], 1e-30)) * 2
    q[c3] = np.stack([(m10[c3] - m01[c3]) / s, (m02[c3] + m20[c3]) / s, (m12[c3] + m21[c3]) / s, 0.25 * s], 1)
    q = _normalize(q)
    q[q[:, 0] < 0] *= -1.0
    return q


def frames_from_normals(nrm: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """Surfel frame from a normal: t_w = n, t_u = unit vector orthogonal to n rotated by an
    in-plane angle U[0, 2pi), t_v = t_w x t_u (Appendix B)."""
    n = _normalize(nrm.astype(np.float64))
    helper = np.where(np.abs(n[:, 2:3]) < 0.9, np.array([[0.0, 0.0, 1.0]]), np.array([[1.0, 0.0, 0.0]]))
    a = _normalize(np.cross(helper, n))
    b = np.cross(n, a)
    ang = rng.uniform(0.0, 2.0 * math.pi, n.shape[0])[:, None]
    tu = np.cos(ang) * a + np.sin(ang) * b
    tv = np.cross(n, tu)
    return quat_from_frame(tu, tv, n)


def random_quats(n: int, rng: np.random.Generator) -> np.ndarray:
    q = _normalize(rng.normal(size=(n, 4)))
    q[q[:, 0] < 0] *= -1.0
    return q


def look_at(eye, target=(0.0, 0.0, 0.0), up=(0.0, 0.0, 1.0)) -> np.ndarray:
    eye = np.asarray(eye, np.float64)
    f = _normalize(np.asarray(target, np.float64) - eye)
    upv = np.asarray(up, np.float64)
    if abs(float(f @ upv)) > 0.999:
        upv = np.array([0.0, 1.0, 0.0])
    r = _normalize(np.cross(f, upv))
    d = np.cross(f, r)
    R = np.stack([r, d, f], 0)  # rows: x right, y down, z forward
    V = np.eye(4)
    V[:3, :3] = R
    V[:3, 3] = -R @ eye
    return V.astype(np.float32)


def make_camera(eye, width, height, f) -> Camera:
    return Camera(view=look_at(eye), fx=float(f), fy=float(f), cx=width / 2.0, cy=height / 2.0,
                  width=int(width), height=int(height))


def cap_cameras(n, radius, elev_lo_deg, elev_hi_deg, width, height, f) -> List[Camera]:
    """n cameras on a spherical cap: golden-angle azimuths, elevations equally spaced in sin(elev)."""
    cams = []
    s_lo, s_hi = math.sin(math.radians(elev_lo_deg)), math.sin(math.radians(elev_hi_deg))
    ga = math.pi * (3.0 - math.sqrt(5.0))
    for i in range(n):
        s = s_lo + (s_hi - s_lo) * (i + 0.5) / n
        c = math.sqrt(max(0.0, 1.0 - s * s))
        az = ga * i
        cams.append(make_camera((radius * c * math.cos(az), radius * c * math.sin(az), radius * s), width, height, f))
    return cams


def sphere_cameras(n, radius, width, height, f) -> List[Camera]:
    """Fibonacci sphere."""
    return cap_cameras(n, radius, -90.0, 90.0, width, height, f)


# ----------------------------------------------------------------------------
# helpers: parameter distributions
# ----------------------------------------------------------------------------

def log_uniform(rng, lo, hi, size):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), size))


def sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def make_sh(rng, n, degree, higher_sigma=0.05):
    sh = np.zeros((n, 16, 3), np.float64)
    base = rng.uniform(0.0, 1.0, (n, 3))
    sh[:, 0, :] = (base - 0.5) / SH_Y0
    nb = (degree + 1) ** 2
    if nb > 1:
        sh[:, 1:nb, :] = rng.normal(0.0, higher_sigma, (n, nb - 1, 3))
    return sh


def room_shell(rng, n, half=5.0):
    """n points on the 6 faces of [-half, half]^3 with inward normals."""
    face = rng.integers(0, 6, n)
    uv = rng.uniform(-half, half, (n, 2))
    pos = np.empty((n, 3))
    nrm = np.zeros((n, 3))
    axis = face // 2
    sign = np.where(face % 2 == 0, -1.0, 1.0)
    for a in range(3):
        m = axis == a
        o = [i for i in range(3) if i != a]
        pos[m, a] = sign[m] * half
        pos[m, o[0]] = uv[m, 0]
        pos[m, o[1]] = uv[m, 1]
        nrm[m, a] = -sign[m]
    return pos, nrm


def _spow(t, e):
    return np.sign(t) * np.abs(t) ** e


def superquadric_points(rng, n, axes, eps1, eps2):
    """Barr superquadric surface, uniform in (eta, omega) (Appendix B)."""
    eta = rng.uniform(-math.pi / 2, math.pi / 2, n)
    om = rng.uniform(-math.pi, math.pi, n)
    ce, se, co, so = np.cos(eta), np.sin(eta), np.cos(om), np.sin(om)
    a1, a2, a3 = axes
    pos = np.stack([a1 * _spow(ce, eps1) * _spow(co, eps2), a2 * _spow(ce, eps1) * _spow(so, eps2), a3 * _spow(se, eps1)], 1)
    nrm = np.stack([_spow(ce, 2 - eps1) * _spow(co, 2 - eps2) / a1, _spow(ce, 2 - eps1) * _spow(so, 2 - eps2) / a2,
                    _spow(se, 2 - eps1) / a3], 1)
    bad = np.linalg.norm(nrm, axis=1) < 1e-12
    nrm[bad] = pos[bad]
    return pos, _normalize(nrm)


def superquadric_implicit(p, axes, eps1, eps2):
    a1, a2, a3 = axes
    x, y, z = np.abs(p[..., 0] / a1), np.abs(p[..., 1] / a2), np.abs(p[..., 2] / a3)
    return (x ** (2 / eps2) + y ** (2 / eps2)) ** (eps2 / eps1) + z ** (2 / eps1) - 1.0


# ----------------------------------------------------------------------------
# masks: analytic silhouettes by ray marching an implicit function inside its bounding sphere
# ----------------------------------------------------------------------------

def _pixel_rays(cam: Camera, step: int):
    """World-space ray origin and directions through pixel centres of a grid subsampled by `step`."""
    xs = np.arange(0, cam.width, step, dtype=np.float64) + (step - 1) / 2.0
    ys = np.arange(0, cam.height, step, dtype=np.float64) + (step - 1) / 2.0
    X, Y = np.meshgrid(xs, ys)
    # integer pixel index = pixel centre; x_idx = fx X/Z + cx - 1/2
    d_cam = np.stack([(X - (cam.cx - 0.5)) / cam.fx, (Y - (cam.cy - 0.5)) / cam.fy, np.ones_like(X)], -1)
    R = cam.view[:3, :3].astype(np.float64)
    d_world = d_cam @ R  # R^T applied to each row vector
    d_world /= np.linalg.norm(d_world, axis=-1, keepdims=True)
    return cam.eye, d_world


def _upsample(mask_small: np.ndarray, cam: Camera, step: int) -> np.ndarray:
    if step == 1:
        return mask_small.astype(np.uint8)
    big = np.repeat(np.repeat(mask_small, step, 0), step, 1)
    return big[: cam.height, : cam.width].astype(np.uint8)


def implicit_silhouette(cam: Camera, implicit: Callable[[np.ndarray], np.ndarray], centre, bound_radius,
                        samples: int = 48, refine: int = 3, step: Optional[int] = None) -> np.ndarray:
    """mask = 1 where the pixel ray meets {implicit <= 0}. Rays are clipped to the bounding sphere, the implicit
    is sampled densely and the minimum refined by local re-sampling."""
    if step is None:
        step = 1 if cam.width * cam.height <= 800 * 600 else 2
    eye, d = _pixel_rays(cam, step)
    c = np.asarray(centre, np.float64)
    oc = eye - c
    b = d @ oc
    disc = b * b - (oc @ oc - bound_radius ** 2)
    hit = disc > 0
    out = np.zeros(d.shape[:2], bool)
    if not hit.any():
        return _upsample(out, cam, step)
    dh = d[hit]
    sq = np.sqrt(disc[hit])
    t0 = np.maximum(-b[hit] - sq, 1e-6)
    t1 = -b[hit] + sq
    frac = (np.arange(samples) + 0.5) / samples
    lo, hi = t0.copy(), t1.copy()
    best = np.full(dh.shape[0], np.inf)
    for _ in range(refine):
        ts = lo[:, None] + (hi - lo)[:, None] * frac[None, :]
        vals = np.empty_like(ts)
        chunk = max(1, 2_000_000 // samples)
        for s in range(0, dh.shape[0], chunk):
            P = eye[None, None, :] + ts[s:s + chunk, :, None] * dh[s:s + chunk, None, :]
            vals[s:s + chunk] = implicit(P)
        k = np.argmin(vals, 1)
        best = np.minimum(best, vals[np.arange(vals.shape[0]), k])
        w = (hi - lo) / samples
        centre_t = ts[np.arange(ts.shape[0]), k]
        lo, hi = np.maximum(centre_t - w, t0), np.minimum(centre_t + w, t1)
    out[hit] = best <= 0
    return _upsample(out, cam, step)


def sphere_silhouette(cam: Camera, radius: float) -> np.ndarray:
    """Exact ray-sphere discriminant test (config 1 / 4)."""
    eye, d = _pixel_rays(cam, 1)
    b = d @ eye
    disc = b * b - (eye @ eye - radius ** 2)
    return ((disc >= 0) & (-b > 0)).astype(np.uint8)


# ----------------------------------------------------------------------------
# the five configs
# ----------------------------------------------------------------------------

def _finish(name, seed, pos, nrm_or_quat, scale, opacity, sh, sh_degree, cams, group, mask_fn) -> Scene:
    return Scene(name=name, seed=seed, pos=np.ascontiguousarray(pos, np.float32),
                 scale=np.ascontiguousarray(scale, np.float32), quat=np.ascontiguousarray(nrm_or_quat, np.float32),
                 opacity=np.ascontiguousarray(opacity, np.float32), sh=np.ascontiguousarray(sh, np.float32),
                 sh_degree=sh_degree, cameras=cams, group=np.ascontiguousarray(group, np.uint8), mask_fn=mask_fn)


def config1(n_obj=2000, n_bg=1000, res=128, f=150.0, seed=0) -> Scene:
    """Tiny oracle scene (BASELINE.json configs[0])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    p_obj = _normalize(rng.normal(size=(n_obj, 3)))
    q_obj = frames_from_normals(p_obj, rng)
    p_bg = rng.uniform(-3.0, 3.0, (n_bg, 3))
    q_bg = random_quats(n_bg, rng)
    n = n_obj + n_bg
    scale = log_uniform(rng, 0.01, 0.05, (n, 2))
    opacity = sigmoid(rng.normal(1.0, 0.5, n))
    sh = make_sh(rng, n, 0)
    cams = [make_camera((3.0 * math.cos(a), 3.0 * math.sin(a), 0.0), res, res, f)
            for a in (0.0, math.pi / 2, math.pi, 3 * math.pi / 2)]
    group = np.concatenate([np.zeros(n_obj), np.ones(n_bg)])
    return _finish("config1_tiny", seed, np.concatenate([p_obj, p_bg]), np.concatenate([q_obj, q_bg]), scale, opacity,
                   sh, 0, cams, group, lambda cam: sphere_silhouette(cam, 1.0))


def config2(n_obj=100_000, n_bg=100_000, width=800, height=600, f=900.0, n_views=16, seed=1) -> Scene:
    """Small object scene: torus + ground plane / back wall (configs[1])."""
    rng = np.random.Generator(np.random.PCG64(seed))
    R, r = 1.0, 0.35
    th = rng.uniform(0, 2 * math.pi, n_obj)
    ph = rng.uniform(0, 2 * math.pi, n_obj)
    p_obj = np.stack([(R + r * np.cos(ph)) * np.cos(th), (R + r * np.cos(ph)) * np.sin(th), r * np.sin(ph)], 1)
    n_objn = np.stack([np.cos(ph) * np.cos(th), np.cos(ph) * np.sin(th), np.sin(ph)], 1)
    n_ground = n_bg // 2
    n_wall = n_bg - n_ground
    p_g = np.stack([rng.uniform(-4, 4, n_ground), rng.uniform(-4, 4, n_ground), np.full(n_ground, -0.5)], 1)
    p_w = np.stack([np.full(n_wall, -4.0), rng.uniform(-4, 4, n_wall), rng.uniform(-0.5, 3.5, n_wall)], 1)
    nrm = np.concatenate([n_objn, np.tile([[0.0, 0.0, 1.0]], (n_ground, 1)), np.tile([[1.0, 0.0, 0.0]], (n_wall, 1))])
    pos = np.concatenate([p_obj, p_g, p_w])
    quat = frames_from_normals(nrm, rng)
    n = pos.shape[0]
    scale = log_uniform(rng, 0.003, 0.03, (n, 2))
    opacity = sigmoid(rng.normal(0.0, 1.0, n))
    sh = make_sh(rng, n, 3)
    cams = cap_cameras(n_views, 3.5, 10.0, 70.0, width, height, f)
    group = np.concatenate([np.zeros(n_obj), np.ones(n_bg)])

    def torus_implicit(P):
        rho = np.sqrt(P[..., 0] ** 2 + P[..., 1] ** 2)
        return (rho - R) ** 2 + P[..., 2] ** 2 - r * r

    return _finish("config2_small", seed, pos, quat, scale, opacity, sh, 3, cams, group,
                   lambda cam: implicit_silhouette(cam, torus_implicit, (0, 0, 0), R + r + 1e-3))


_SQ_AXES, _SQ_E1, _SQ_E2 = (1.0, 0.8, 0.6), 0.6, 1.4


def config3(n_obj=300_000, n_bg=700_000, width=1600, height=1200, f=2800.0, n_views=49, seed=2) -> Scene:
    """Paper-shaped multi-view object capture (configs[2]) -- the headline workload."""
    rng = np.random.Generator(np.random.PCG64(seed))
    p_obj, n_objn = superquadric_points(rng, n_obj, _SQ_AXES, _SQ_E1, _SQ_E2)
    p_bg, n_bgn = room_shell(rng, n_bg, 5.0)
    pos = np.concatenate([p_obj, p_bg])
    quat = frames_from_normals(np.concatenate([n_objn, n_bgn]), rng)
    n = pos.shape[0]
    scale = log_uniform(rng, 0.003, 0.03, (n, 2))
    opacity = sigmoid(rng.normal(0.0, 1.0, n))
    sh = make_sh(rng, n, 3)
    cams = cap_cameras(n_views, 3.0, 10.0, 60.0, width, height, f)
    group = np.concatenate([np.zeros(n_obj), np.ones(n_bg)])
    return _finish("config3_paper", seed, pos, quat, scale, opacity, sh, 3, cams, group,
                   lambda cam: implicit_silhouette(cam, lambda P: superquadric_implicit(P, _SQ_AXES, _SQ_E1, _SQ_E2),
                                                   (0, 0, 0), 1.0 + 1e-3))


def config4(n_shell=250_000, n_in=400_000, n_bg=150_000, res=1024, f=1300.0, n_views=64, seed=3, scale_mul=1.0) -> Scene:
    """Occlusion-heavy pruning workload (configs[3]): near-opaque shell, occluded interior, room shell.
    scale_mul > 1 enlarges the SHELL surfels only, to keep the shell's coverage when a test shrinks the surfel counts
    (coverage ~ n_shell * scale^2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    p_shell = _normalize(rng.normal(size=(n_shell, 3)))
    q_shell = frames_from_normals(p_shell, rng)
    p_in = _normalize(rng.normal(size=(n_in, 3))) * (0.95 * rng.uniform(0, 1, (n_in, 1)) ** (1 / 3))
    q_in = random_quats(n_in, rng)
    p_bg, n_bgn = room_shell(rng, n_bg, 5.0)
    q_bg = frames_from_normals(n_bgn, rng)
    pos = np.concatenate([p_shell, p_in, p_bg])
    quat = np.concatenate([q_shell, q_in, q_bg])
    n = pos.shape[0]
    scale = log_uniform(rng, 0.003, 0.03, (n, 2))
    scale[:n_shell] *= scale_mul
    opacity = np.concatenate([sigmoid(rng.normal(3.0, 0.5, n_shell)), sigmoid(rng.normal(0.0, 1.0, n_in + n_bg))])
    sh = make_sh(rng, n, 3)
    cams = sphere_cameras(n_views, 3.0, res, res, f)
    group = np.concatenate([np.zeros(n_shell), np.full(n_in, 2), np.ones(n_bg)])
    return _finish("config4_occlusion", seed, pos, quat, scale, opacity, sh, 3, cams, group,
                   lambda cam: sphere_silhouette(cam, 1.0))


def config5(n_obj=1_000_000, n_bg=3_000_000, width=1920, height=1080, f=1700.0, n_views=32, seed=4) -> Scene:
    """Large stress scene (configs[4]): union of 3 random superquadrics + room shell, small scales."""
    rng = np.random.Generator(np.random.PCG64(seed))
    parts = []
    sqs = []
    for k in range(3):
        axes = tuple(rng.uniform(0.4, 0.9, 3))
        e1, e2 = rng.uniform(0.5, 1.5, 2)
        centre = rng.uniform(-0.5, 0.5, 3)
        Rm = _quat_to_mat(random_quats(1, rng)[0])
        cnt = n_obj // 3 if k < 2 else n_obj - 2 * (n_obj // 3)
        p, nn = superquadric_points(rng, cnt, axes, e1, e2)
        parts.append((p @ Rm.T + centre, nn @ Rm.T))
        sqs.append((axes, e1, e2, centre, Rm))
    p_obj = np.concatenate([p for p, _ in parts])
    n_objn = np.concatenate([nn for _, nn in parts])
    p_bg, n_bgn = room_shell(rng, n_bg, 5.0)
    pos = np.concatenate([p_obj, p_bg])
    quat = frames_from_normals(np.concatenate([n_objn, n_bgn]), rng)
    n = pos.shape[0]
    scale = log_uniform(rng, 0.001, 0.02, (n, 2))
    opacity = sigmoid(rng.normal(0.0, 1.0, n))
    sh = make_sh(rng, n, 3)
    cams = cap_cameras(n_views, 4.0, 10.0, 60.0, width, height, f)
    group = np.concatenate([np.zeros(n_obj), np.ones(n_bg)])

    def union_implicit(P):
        best = None
        for axes, e1, e2, centre, Rm in sqs:
            v = superquadric_implicit((P - centre) @ Rm, axes, e1, e2)
            best = v if best is None else np.minimum(best, v)
        return best

    return _finish("config5_stress", seed, pos, quat, scale, opacity, sh, 3, cams, group,
                   lambda cam: implicit_silhouette(cam, union_implicit, (0, 0, 0), 2.2))


def _quat_to_mat(q):
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


CONFIGS: Dict[str, Callable[..., Scene]] = {
    "config1": config1, "config2": config2, "config3": config3, "config4": config4, "config5": config5,
}


def make_scene(name: str, **overrides) -> Scene:
    """`overrides` shrink a config (e.g. n_obj, n_bg, width, height, n_views) for fast tests; distributions are unchanged."""
    return CONFIGS[name](**overrides)


def random_scene(n: int, width: int, height: int, f: float, seed: int, sh_degree: int = 3,
                 scale_lo=0.02, scale_hi=0.2, depth_lo=1.0, depth_hi=4.0, op_mu=0.0, op_sigma=1.0) -> Scene:
    """Unstructured tiny scene in front of one camera at the origin looking down +z (world = camera frame up to
    the look_at axes): used by brute-force / finite-difference tests."""
    rng = np.random.Generator(np.random.PCG64(seed))
    cam = Camera(view=np.eye(4, dtype=np.float32), fx=float(f), fy=float(f), cx=width / 2.0, cy=height / 2.0,
                 width=width, height=height)
    z = rng.uniform(depth_lo, depth_hi, n)
    x = rng.uniform(-0.5, 0.5, n) * width / f * z
    y = rng.uniform(-0.5, 0.5, n) * height / f * z
    pos = np.stack([x, y, z], 1)
    quat = random_quats(n, rng)
    scale = log_uniform(rng, scale_lo, scale_hi, (n, 2))
    opacity = sigmoid(rng.normal(op_mu, op_sigma, n))
    sh = make_sh(rng, n, sh_degree, higher_sigma=0.2)
    mask = (rng.uniform(size=(height, width)) < 0.5).astype(np.uint8)
    return _finish(f"random{seed}", seed, pos, quat, scale, opacity, sh, sh_degree, [cam], np.zeros(n), lambda c: mask)
