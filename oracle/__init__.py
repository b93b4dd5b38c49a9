"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see oracle/ocgs_oracle.cpp header).

Thin ctypes/numpy wrapper over ``liborc.so`` (plain C++ built by ``oracle/build.py``).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It imports nothing from the CUDA package and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liborc.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "ocgs_oracle.cpp")
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(src):
        cmd = ["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-o", _LIB_PATH, src]
        subprocess.check_call(cmd)
    return _LIB_PATH


class OrcCamera(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("width", C.c_int), ("height", C.c_int)]


class OrcConfig(C.Structure):
    _fields_ = [("tile", C.c_int), ("near_z", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
                ("t_min", C.c_float), ("rho_max", C.c_float), ("filter_sigma2", C.c_float), ("bg", C.c_float * 3),
                ("gamma_bg", C.c_float), ("tau_contrib", C.c_float), ("min_opacity", C.c_float), ("sh_degree", C.c_int)]


class OrcMargins(C.Structure):
    _fields_ = [("rho_cut_abs", C.c_double), ("near_rel", C.c_double), ("tmin_rel", C.c_double),
                ("switch_rel", C.c_double), ("cap_abs", C.c_double), ("eps32", C.c_double), ("cond_abs", C.c_double)]


def default_config(sh_degree: int = 3, bg=(0.0, 0.0, 0.0), gamma_bg: float = 0.5, **kw) -> OrcConfig:
    """Defaults of SURVEY.md §8(c): S3, S5, S6, S8, S11, S13; gamma = 0.5."""
    c = OrcConfig()
    c.tile = 16
    c.near_z = 0.2
    c.alpha_min = float(np.float32(1.0 / 255.0))
    c.alpha_max = 0.99
    c.t_min = 1e-4
    c.rho_max = 9.0
    c.filter_sigma2 = 0.5
    c.bg[0], c.bg[1], c.bg[2] = bg
    c.gamma_bg = gamma_bg
    c.tau_contrib = 0.0
    c.min_opacity = 0.0
    c.sh_degree = sh_degree
    for k, v in kw.items():
        setattr(c, k, v)
    return c


def default_margins(scale: float = 1.0) -> OrcMargins:
    """Fragile-pixel decision margins: sized to a few fp32 ulps of each quantity."""
    return OrcMargins(rho_cut_abs=4e-5 * scale, near_rel=2e-5 * scale, tmin_rel=2e-4 * scale, switch_rel=2e-5 * scale,
                      cap_abs=2e-5 * scale, eps32=2.0 ** -23, cond_abs=2e-5 / scale)


def make_camera(view, fx, fy, cx, cy, width, height) -> OrcCamera:
    cam = OrcCamera()
    v = np.ascontiguousarray(view, np.float32).reshape(16)
    for i in range(16):
        cam.view[i] = float(v[i])
    cam.fx, cam.fy, cam.cx, cam.cy = float(fx), float(fy), float(cx), float(cy)
    cam.width, cam.height = int(width), int(height)
    return cam


def camera_from(scene_cam) -> OrcCamera:
    return make_camera(scene_cam.view, scene_cam.fx, scene_cam.fy, scene_cam.cx, scene_cam.cy, scene_cam.width, scene_cam.height)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB_PATH)
        _lib.orc_bin_sort.restype = C.c_int64
        _lib.orc_render_fwd.restype = C.c_double
        _lib.orc_bf_render.restype = C.c_double
        _lib.orc_prune.restype = C.c_int
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int) -> int:
    """OpenMP threads of the following oracle calls; returns the number in force."""
    lib().orc_set_num_threads.restype = C.c_int
    return int(lib().orc_set_num_threads(C.c_int(int(n))))


def _f32(a):
    return np.ascontiguousarray(a, np.float32)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, np.float64)


# --------------------------------------------------------------------------------------------------
# TILED path
# --------------------------------------------------------------------------------------------------

def colour_probe(p, sh, degree: int, cam: OrcCamera):
    """R-clamp: (fp32 decision values, fp64 values before the clamp, clamp bits) of one surfel's colour."""
    p, sh = _f32(p).reshape(3), _f32(sh).reshape(16, 3)
    a32, a64, cl = np.zeros(3, np.float32), np.zeros(3, np.float64), np.zeros(1, np.uint8)
    lib().orc_colour_probe(_p(p), _p(sh), C.c_int(degree), C.byref(cam), _p(a32), _p(a64), _p(cl))
    return a32, a64, int(cl[0])


def preprocess(pos, scale, quat, opacity, sh, cam: OrcCamera, cfg: OrcConfig) -> Dict[str, np.ndarray]:
    pos, scale, quat, opacity, sh = _f32(pos), _f32(scale), _f32(quat), _f32(opacity), _f32(sh)
    n = pos.shape[0]
    out = dict(visible=np.zeros(n, np.uint8), depth_bits=np.zeros(n, np.uint32), rect=np.zeros((n, 4), np.int32),
               tiles_touched=np.zeros(n, np.uint32), M=np.zeros((n, 9), np.float32), c2d=np.zeros((n, 2), np.float32),
               rho_cut=np.zeros(n, np.float32), normal=np.zeros((n, 3), np.float64), rgb=np.zeros((n, 3), np.float64),
               clamp=np.zeros(n, np.uint8))
    lib().orc_preprocess(C.c_int(n), _p(pos), _p(scale), _p(quat), _p(opacity), _p(sh), C.byref(cam), C.byref(cfg),
                         _p(out["visible"]), _p(out["depth_bits"]), _p(out["rect"]), _p(out["tiles_touched"]), _p(out["M"]),
                         _p(out["c2d"]), _p(out["rho_cut"]), _p(out["normal"]), _p(out["rgb"]), _p(out["clamp"]))
    return out


def tiles_of(cam: OrcCamera, cfg: OrcConfig) -> Tuple[int, int]:
    return (cam.width + cfg.tile - 1) // cfg.tile, (cam.height + cfg.tile - 1) // cfg.tile


def bin_sort(pre: Dict[str, np.ndarray], cam: OrcCamera, cfg: OrcConfig) -> Dict[str, np.ndarray]:
    n = pre["visible"].shape[0]
    tx, ty = tiles_of(cam, cfg)
    args = (C.c_int(n), _p(pre["visible"]), _p(pre["depth_bits"]), _p(pre["rect"]), C.c_int(cfg.tile), C.c_int(tx), C.c_int(ty))
    K = int(lib().orc_bin_sort(*args, None, None, None))
    keys = np.zeros(max(K, 1), np.uint64)
    ids = np.zeros(max(K, 1), np.uint32)
    ranges = np.zeros((tx * ty, 2), np.uint32)
    K2 = int(lib().orc_bin_sort(*args, _p(keys), _p(ids), _p(ranges)))
    assert K2 == K
    return dict(K=K, keys=keys[:K], ids=ids[:K], ranges=ranges)


def render_fwd(pre, srt, opacity, cam: OrcCamera, cfg: OrcConfig, mask=None, window=None, margins: Optional[OrcMargins] = None,
               vis_count=None, contrib_sum=None, want_fragile=True) -> Dict[str, np.ndarray]:
    W, H = cam.width, cam.height
    n = pre["visible"].shape[0]
    opacity = _f32(opacity)
    x0, y0, x1, y1 = window if window is not None else (0, 0, W, H)
    out = dict(color=np.zeros((3, H, W)), alpha=np.zeros((H, W)), depth=np.zeros((H, W)), normal=np.zeros((3, H, W)),
               n_contrib=np.zeros((H, W), np.uint32), origin=np.zeros((H, W)), m1=np.zeros((H, W)), m2=np.zeros((H, W)))
    if vis_count is None:
        vis_count = np.zeros(n, np.uint32)
    if contrib_sum is None:
        contrib_sum = np.zeros(n, np.float64)
    fragile = np.zeros((H, W), np.uint8) if want_fragile else None
    ftouch = np.zeros(n, np.uint32) if want_fragile else None
    cond_rho = np.zeros(n, np.float64) if want_fragile else None
    if margins is None and want_fragile:
        margins = default_margins()
    ids = srt["ids"] if srt["K"] > 0 else np.zeros(1, np.uint32)
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    Lb = lib().orc_render_fwd(C.c_int(n), C.byref(cam), C.byref(cfg), C.byref(margins) if margins is not None else None,
                              _p(pre["M"]), _p(pre["c2d"]), _p(pre["rho_cut"]), _p(opacity), _p(pre["normal"]), _p(pre["rgb"]),
                              _p(ids), _p(srt["ranges"]), _p(m), C.c_int(x0), C.c_int(y0), C.c_int(x1), C.c_int(y1),
                              _p(out["color"]), _p(out["alpha"]), _p(out["depth"]), _p(out["normal"]), _p(out["n_contrib"]),
                              _p(vis_count), _p(contrib_sum), _p(fragile), _p(ftouch), _p(cond_rho), _p(out["origin"]), _p(out["m1"]), _p(out["m2"]))
    out.update(loss_bg=float(Lb), vis_count=vis_count, contrib_sum=contrib_sum, fragile=fragile, fragile_touch=ftouch, cond_rho=cond_rho)
    return out


def render_bwd(pos, scale, quat, opacity, sh, pre, srt, cam: OrcCamera, cfg: OrcConfig, mask=None, gC=None, gA=None, gD=None,
               gN=None, window=None, gM1=None, gM2=None) -> Dict[str, np.ndarray]:
    pos, scale, quat, opacity, sh = _f32(pos), _f32(scale), _f32(quat), _f32(opacity), _f32(sh)
    n = pos.shape[0]
    W, H = cam.width, cam.height
    x0, y0, x1, y1 = window if window is not None else (0, 0, W, H)
    out = dict(d_pos=np.zeros((n, 3)), d_scale=np.zeros((n, 2)), d_quat=np.zeros((n, 4)), d_opacity=np.zeros(n),
               d_sh=np.zeros((n, 16, 3)), d_center2d=np.zeros((n, 2)))
    oabs = np.zeros(n)
    # sums of |terms| behind every entry (conditioning of the sums; see orc_render_bwd)
    ab = dict(d_pos=np.zeros((n, 3)), d_scale=np.zeros((n, 2)), d_quat=np.zeros((n, 4)), d_sh=np.zeros((n, 16, 3)), d_center2d=np.zeros((n, 2)))
    ids = srt["ids"] if srt["K"] > 0 else np.zeros(1, np.uint32)
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    gC, gA, gD, gN, gM1, gM2 = _f64(gC), _f64(gA), _f64(gD), _f64(gN), _f64(gM1), _f64(gM2)
    lib().orc_render_bwd(C.c_int(n), _p(pos), _p(scale), _p(quat), _p(opacity), _p(sh), C.byref(cam), C.byref(cfg),
                         _p(pre["visible"]), _p(pre["M"]), _p(pre["c2d"]), _p(pre["rho_cut"]), _p(pre["normal"]), _p(pre["rgb"]),
                         _p(pre["clamp"]), _p(ids), _p(srt["ranges"]), _p(m), _p(gC), _p(gA), _p(gD), _p(gN),
                         C.c_int(x0), C.c_int(y0), C.c_int(x1), C.c_int(y1), _p(out["d_pos"]), _p(out["d_scale"]),
                         _p(out["d_quat"]), _p(out["d_opacity"]), _p(out["d_sh"]), _p(out["d_center2d"]), _p(oabs), _p(gM1), _p(gM2),
                         _p(ab["d_pos"]), _p(ab["d_scale"]), _p(ab["d_quat"]), _p(ab["d_sh"]), _p(ab["d_center2d"]))
    out["_d_opacity_abs"] = oabs
    ab["d_opacity"] = oabs
    out["_abs"] = ab
    return out


def prune(vis_count, contrib_sum, opacity, tau: float = 0.0, min_opacity: float = 0.0):
    vis_count = np.ascontiguousarray(vis_count, np.uint32)
    contrib_sum, opacity = _f32(contrib_sum), _f32(opacity)
    n = vis_count.shape[0]
    mask = np.zeros(n, np.uint8)
    remap = np.zeros(n, np.int32)
    kept = lib().orc_prune(C.c_int(n), _p(vis_count), _p(contrib_sum), _p(opacity), C.c_float(tau), C.c_float(min_opacity),
                           _p(mask), _p(remap))
    return dict(prune_mask=mask, remap=remap, n_out=int(kept))


def compact(arrays: Dict[str, np.ndarray], prune_mask: np.ndarray) -> Dict[str, np.ndarray]:
    """O9 compaction by its definition: survivors in ascending id order."""
    keep = prune_mask == 0
    return {k: np.ascontiguousarray(v[keep]) for k, v in arrays.items()}


def forward_view(pos, scale, quat, opacity, sh, cam: OrcCamera, cfg: OrcConfig, mask=None, **kw):
    """preprocess -> bin_sort -> render_fwd for one view; returns (pre, srt, fwd)."""
    pre = preprocess(pos, scale, quat, opacity, sh, cam, cfg)
    srt = bin_sort(pre, cam, cfg)
    fwd = render_fwd(pre, srt, opacity, cam, cfg, mask=mask, **kw)
    return pre, srt, fwd


# --------------------------------------------------------------------------------------------------
# BF path
# --------------------------------------------------------------------------------------------------

def bf_render(pos, scale, quat, opacity, sh, cam: OrcCamera, cfg: OrcConfig, mask=None, window=None, want_stats=True):
    pos, scale, quat, opacity, sh = _f64(pos), _f64(scale), _f64(quat), _f64(opacity), _f64(sh)
    n = pos.shape[0]
    W, H = cam.width, cam.height
    x0, y0, x1, y1 = window if window is not None else (0, 0, W, H)
    out = dict(color=np.zeros((3, H, W)), alpha=np.zeros((H, W)), depth=np.zeros((H, W)), normal=np.zeros((3, H, W)),
               n_blended=np.zeros((H, W), np.uint32), origin=np.zeros((H, W)), m1=np.zeros((H, W)), m2=np.zeros((H, W)))
    vis = np.zeros(n, np.uint32) if want_stats else None
    cs = np.zeros(n, np.float64) if want_stats else None
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    Lb = lib().orc_bf_render(C.c_int(n), _p(pos), _p(scale), _p(quat), _p(opacity), _p(sh), C.byref(cam), C.byref(cfg), _p(m),
                             C.c_int(x0), C.c_int(y0), C.c_int(x1), C.c_int(y1), _p(out["color"]), _p(out["alpha"]),
                             _p(out["depth"]), _p(out["normal"]), _p(out["n_blended"]), _p(vis), _p(cs), _p(out["origin"]), _p(out["m1"]), _p(out["m2"]))
    out.update(loss_bg=float(Lb), vis_count=vis, contrib_sum=cs)
    return out


def sh_basis(direction) -> np.ndarray:
    d = _f64(direction).reshape(3)
    Y = np.zeros(16)
    lib().orc_sh_basis(_p(d), _p(Y))
    return Y


# --------------------------------------------------------------------------------------------------
# 3D-Gaussian variant of the visibility statistics (Appendix B; reading R-3D)
# --------------------------------------------------------------------------------------------------

def preprocess3d(pos, scale3, quat, opacity, sh, cam: OrcCamera, cfg: OrcConfig) -> Dict[str, np.ndarray]:
    pos, scale3, quat, opacity, sh = _f32(pos), _f32(scale3), _f32(quat), _f32(opacity), _f32(sh)
    n = pos.shape[0]
    assert scale3.shape == (n, 3)
    out = dict(visible=np.zeros(n, np.uint8), depth_bits=np.zeros(n, np.uint32), rect=np.zeros((n, 4), np.int32),
               tiles_touched=np.zeros(n, np.uint32), conic=np.zeros((n, 3), np.float32), c2d=np.zeros((n, 2), np.float32),
               rho_cut=np.zeros(n, np.float32), rgb=np.zeros((n, 3), np.float64), clamp=np.zeros(n, np.uint8))
    lib().orc3d_preprocess(C.c_int(n), _p(pos), _p(scale3), _p(quat), _p(opacity), _p(sh), C.byref(cam), C.byref(cfg),
                           _p(out["visible"]), _p(out["depth_bits"]), _p(out["rect"]), _p(out["tiles_touched"]), _p(out["conic"]),
                           _p(out["c2d"]), _p(out["rho_cut"]), _p(out["rgb"]), _p(out["clamp"]))
    return out


def render3d_fwd(pre, srt, opacity, cam: OrcCamera, cfg: OrcConfig, mask=None, window=None, vis_count=None, contrib_sum=None,
                 want_fragile=True) -> Dict[str, np.ndarray]:
    """bin_sort(pre, ...) serves both primitives: it only reads visible / depth_bits / rect."""
    W, H = cam.width, cam.height
    n = pre["visible"].shape[0]
    opacity = _f32(opacity)
    x0, y0, x1, y1 = window if window is not None else (0, 0, W, H)
    out = dict(color=np.zeros((3, H, W)), alpha=np.zeros((H, W)), depth=np.zeros((H, W)), n_contrib=np.zeros((H, W), np.uint32))
    if vis_count is None:
        vis_count = np.zeros(n, np.uint32)
    if contrib_sum is None:
        contrib_sum = np.zeros(n, np.float64)
    fragile = np.zeros((H, W), np.uint8) if want_fragile else None
    ftouch = np.zeros(n, np.uint32) if want_fragile else None
    margins = default_margins() if want_fragile else None
    ids = srt["ids"] if srt["K"] > 0 else np.zeros(1, np.uint32)
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().orc3d_render_fwd.restype = C.c_double
    Lb = lib().orc3d_render_fwd(C.c_int(n), C.byref(cam), C.byref(cfg), C.byref(margins) if margins is not None else None,
                                _p(pre["conic"]), _p(pre["c2d"]), _p(pre["rho_cut"]), _p(opacity), _p(pre["depth_bits"]), _p(pre["rgb"]),
                                _p(ids), _p(srt["ranges"]), _p(m), C.c_int(x0), C.c_int(y0), C.c_int(x1), C.c_int(y1),
                                _p(out["color"]), _p(out["alpha"]), _p(out["depth"]), _p(out["n_contrib"]), _p(vis_count),
                                _p(contrib_sum), _p(fragile), _p(ftouch))
    out.update(loss_bg=float(Lb), vis_count=vis_count, contrib_sum=contrib_sum, fragile=fragile, fragile_touch=ftouch)
    return out


def bf3d_render(pos, scale3, quat, opacity, sh, cam: OrcCamera, cfg: OrcConfig, mask=None, window=None, want_stats=True):
    pos, scale3, quat, opacity, sh = _f64(pos), _f64(scale3), _f64(quat), _f64(opacity), _f64(sh)
    n = pos.shape[0]
    W, H = cam.width, cam.height
    x0, y0, x1, y1 = window if window is not None else (0, 0, W, H)
    out = dict(color=np.zeros((3, H, W)), alpha=np.zeros((H, W)), depth=np.zeros((H, W)), n_blended=np.zeros((H, W), np.uint32))
    vis = np.zeros(n, np.uint32) if want_stats else None
    cs = np.zeros(n, np.float64) if want_stats else None
    m = None if mask is None else np.ascontiguousarray(mask, np.uint8)
    lib().orc3d_bf_render.restype = C.c_double
    Lb = lib().orc3d_bf_render(C.c_int(n), _p(pos), _p(scale3), _p(quat), _p(opacity), _p(sh), C.byref(cam), C.byref(cfg), _p(m),
                               C.c_int(x0), C.c_int(y0), C.c_int(x1), C.c_int(y1), _p(out["color"]), _p(out["alpha"]),
                               _p(out["depth"]), _p(out["n_blended"]), _p(vis), _p(cs))
    out.update(loss_bg=float(Lb), vis_count=vis, contrib_sum=cs)
    return out
