"""Thin ctypes binding over ``csrc/libocgs.so`` (C ABI in ``include/ocgs.h``): argument marshalling only.

Every function has the name of the C entry point it calls; tensors are torch CUDA tensors whose ``data_ptr()`` is
passed through.  torch is used for device memory and streams, nothing else.  There is no CPU fallback: importing
this module without the built library, or calling it without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "csrc", "libocgs.so")

OCGS_OK, OCGS_ERR_INVALID_ARG, OCGS_ERR_CAPACITY, OCGS_ERR_CUDA, OCGS_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
EXPORTS = ["ocgs_default_config", "ocgs_workspace_layout", "ocgs_workspace_bytes", "ocgs_last_cuda_error", "ocgs_check",
           "ocgs_preprocess", "ocgs_bin_sort", "ocgs_render_fwd", "ocgs_render_bwd", "ocgs_render_fwd_l1", "ocgs_render_fwd_reg", "ocgs_render_bwd_reg", "ocgs3d_preprocess", "ocgs3d_render_fwd", "ocgs_prune_workspace_bytes",
           "ocgs_prune_stats", "ocgs_compact_rows", "ocgs_densify_workspace_bytes", "ocgs_densify_accumulate", "ocgs_densify", "ocgs_step_host", "ocgs_step_view_host", "ocgs_step_view_host_enqueue", "ocgs_step_view_prefetch_enqueue", "ocgs_visibility_pass", "ocgs3d_visibility_pass", "ocgs_masked_l1", "ocgs_photometric_workspace_bytes", "ocgs_photometric_loss", "ocgs_regularizers_workspace_bytes", "ocgs_regularizers",
           "ocgs_profile_begin", "ocgs_profile_end", "ocgs_peak_probe", "ocgs_masked_l1_static", "ocgs_staging_probe"]


class OcgsError(RuntimeError):
    def __init__(self, fn: str, code: int):
        names = {-1: "INVALID_ARG", -2: "CAPACITY", -3: "CUDA", -4: "UNSUPPORTED"}
        extra = f" (cudaError {lib().ocgs_last_cuda_error()})" if code == OCGS_ERR_CUDA else ""
        super().__init__(f"{fn} failed: OCGS_ERR_{names.get(code, code)}{extra}")
        self.code = code


class ocgs_camera(C.Structure):
    _fields_ = [("view", C.c_float * 16), ("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("width", C.c_int), ("height", C.c_int)]


class ocgs_config(C.Structure):
    _fields_ = [("tile", C.c_int), ("near_z", C.c_float), ("alpha_min", C.c_float), ("alpha_max", C.c_float),
                ("t_min", C.c_float), ("rho_max", C.c_float), ("filter_sigma2", C.c_float), ("bg", C.c_float * 3),
                ("gamma_bg", C.c_float), ("tau_contrib", C.c_float), ("min_opacity", C.c_float), ("sh_degree", C.c_int)]


class ocgs_surfels(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p), ("sh", C.c_void_p),
                ("n", C.c_int)]


class ocgs_gaussians3d(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p), ("sh", C.c_void_p),
                ("n", C.c_int)]


class ocgs_surfels_mut(C.Structure):
    _fields_ = [("pos", C.c_void_p), ("scale", C.c_void_p), ("quat", C.c_void_p), ("opacity", C.c_void_p), ("sh", C.c_void_p),
                ("capacity", C.c_int)]


_LAYOUT_FIELDS = ["total_bytes", "header", "depth_bits", "rect", "tiles", "clamp", "rec_id", "id_to_rank", "rank_to_id", "rec",
                  "offsets", "tile_keys", "tile_vals", "ranges", "grad_rec", "loss_partial", "final_T", "scratch"]


class ocgs_ws_layout(C.Structure):
    _fields_ = [(f, C.c_size_t) for f in _LAYOUT_FIELDS]


class ocgs_header(C.Structure):
    _fields_ = [("K", C.c_ulonglong), ("n_vis", C.c_uint), ("error", C.c_uint)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2501_08174_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        _lib = C.CDLL(_LIB_PATH)
        _lib.ocgs_workspace_bytes.restype = C.c_size_t
        _lib.ocgs_prune_workspace_bytes.restype = C.c_size_t
        _lib.ocgs_photometric_workspace_bytes.restype = C.c_size_t
        _lib.ocgs_densify_workspace_bytes.restype = C.c_size_t
        _lib.ocgs_regularizers_workspace_bytes.restype = C.c_size_t
        for name in EXPORTS:
            getattr(_lib, name)  # raises AttributeError if a declared symbol is not exported
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if not t.is_contiguous():
        raise ValueError("expected a contiguous tensor")
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ok(fn: str, code: int):
    if code != OCGS_OK:
        raise OcgsError(fn, code)


def ocgs_default_config(**kw) -> ocgs_config:
    c = ocgs_config()
    lib().ocgs_default_config(C.byref(c))
    for k, v in kw.items():
        if k == "bg":
            c.bg[0], c.bg[1], c.bg[2] = v
        else:
            setattr(c, k, v)
    return c


def make_camera(view, fx, fy, cx, cy, width, height) -> ocgs_camera:
    cam = ocgs_camera()
    flat = [float(x) for x in (view.reshape(-1).tolist() if hasattr(view, "reshape") else view)]
    for i in range(16):
        cam.view[i] = flat[i]
    cam.fx, cam.fy, cam.cx, cam.cy = float(fx), float(fy), float(cx), float(cy)
    cam.width, cam.height = int(width), int(height)
    return cam


def camera_from(scene_cam) -> ocgs_camera:
    return make_camera(scene_cam.view, scene_cam.fx, scene_cam.fy, scene_cam.cx, scene_cam.cy, scene_cam.width, scene_cam.height)


def make_surfels(pos, scale, quat, opacity, sh) -> ocgs_surfels:
    n = int(pos.shape[0])
    for t, per in ((pos, 3), (scale, 2), (quat, 4), (opacity, 1), (sh, 48)):
        if t.dtype != torch.float32 or t.numel() != n * per:
            raise ValueError("surfel arrays must be float32 with shapes [N,3],[N,2],[N,4],[N],[N,16,3]")
    return ocgs_surfels(_ptr(pos), _ptr(scale), _ptr(quat), _ptr(opacity), _ptr(sh), n)


def ocgs_workspace_layout(n: int, width: int, height: int, key_capacity: int) -> ocgs_ws_layout:
    L = ocgs_ws_layout()
    _ok("ocgs_workspace_layout", lib().ocgs_workspace_layout(C.c_int(n), C.c_int(width), C.c_int(height), C.c_size_t(key_capacity), C.byref(L)))
    return L


def ocgs_workspace_bytes(n: int, width: int, height: int, key_capacity: int) -> int:
    return int(lib().ocgs_workspace_bytes(C.c_int(n), C.c_int(width), C.c_int(height), C.c_size_t(key_capacity)))


def ocgs_check(ws: torch.Tensor, stream=None, raise_on_error: bool = True) -> ocgs_header:
    h = ocgs_header()
    code = lib().ocgs_check(_ptr(ws), _stream(stream), C.byref(h))
    if code != OCGS_OK and raise_on_error:
        raise OcgsError("ocgs_check", code)
    return h


def ocgs_preprocess(surfels: ocgs_surfels, cam: ocgs_camera, cfg: ocgs_config, ws: torch.Tensor, key_capacity: int, stream=None):
    _ok("ocgs_preprocess", lib().ocgs_preprocess(C.byref(surfels), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _stream(stream)))


def ocgs_bin_sort(n: int, cam: ocgs_camera, cfg: ocgs_config, ws: torch.Tensor, key_capacity: int, sorted_ids=None, stream=None):
    _ok("ocgs_bin_sort", lib().ocgs_bin_sort(C.c_int(n), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _ptr(sorted_ids), _stream(stream)))


def ocgs_render_fwd(n, cam, cfg, ws, key_capacity, mask, color, alpha, depth, normal, n_contrib, loss_bg=None, vis_count=None,
                    contrib_sum=None, stream=None):
    _ok("ocgs_render_fwd", lib().ocgs_render_fwd(C.c_int(n), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _ptr(mask),
                                                 _ptr(color), _ptr(alpha), _ptr(depth), _ptr(normal), _ptr(n_contrib), _ptr(loss_bg),
                                                 _ptr(vis_count), _ptr(contrib_sum), _stream(stream)))


def ocgs_render_fwd_l1(n, cam, cfg, ws, key_capacity, mask, target, color, alpha, depth, normal, n_contrib, loss_bg, loss_l1, dL_dcolor,
                       vis_count=None, contrib_sum=None, stream=None):
    _ok("ocgs_render_fwd_l1", lib().ocgs_render_fwd_l1(C.c_int(n), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _ptr(mask),
                                                       _ptr(target), _ptr(color), _ptr(alpha), _ptr(depth), _ptr(normal), _ptr(n_contrib),
                                                       _ptr(loss_bg), _ptr(loss_l1), _ptr(dL_dcolor), _ptr(vis_count), _ptr(contrib_sum),
                                                       _stream(stream)))


def make_gaussians3d(pos, scale3, quat, opacity, sh) -> ocgs_gaussians3d:
    n = int(pos.shape[0])
    for t, shape in ((pos, (n, 3)), (scale3, (n, 3)), (quat, (n, 4)), (opacity, (n,)), (sh, (n, 16, 3))):
        if tuple(t.shape) != shape or t.dtype != torch.float32:
            raise ValueError(f"expected float32 tensor of shape {shape}, got {tuple(t.shape)} {t.dtype}")
    return ocgs_gaussians3d(_ptr(pos), _ptr(scale3), _ptr(quat), _ptr(opacity), _ptr(sh), n)


def ocgs3d_preprocess(gaussians: ocgs_gaussians3d, cam, cfg, ws, key_capacity, stream=None):
    _ok("ocgs3d_preprocess", lib().ocgs3d_preprocess(C.byref(gaussians), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity),
                                                     _stream(stream)))


def ocgs3d_render_fwd(n, cam, cfg, ws, key_capacity, mask, color, alpha, depth, n_contrib, loss_bg=None, vis_count=None, contrib_sum=None,
                      stream=None):
    _ok("ocgs3d_render_fwd", lib().ocgs3d_render_fwd(C.c_int(n), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _ptr(mask),
                                                     _ptr(color), _ptr(alpha), _ptr(depth), _ptr(n_contrib), _ptr(loss_bg),
                                                     _ptr(vis_count), _ptr(contrib_sum), _stream(stream)))


def ocgs_visibility_pass(surfels, cam, cfg, ws, key_capacity, vis_count, contrib_sum, stream=None):
    _ok("ocgs_visibility_pass", lib().ocgs_visibility_pass(C.byref(surfels), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity),
                                                           _ptr(vis_count), _ptr(contrib_sum), _stream(stream)))


def ocgs3d_visibility_pass(gaussians, cam, cfg, ws, key_capacity, vis_count, contrib_sum, stream=None):
    _ok("ocgs3d_visibility_pass", lib().ocgs3d_visibility_pass(C.byref(gaussians), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity),
                                                               _ptr(vis_count), _ptr(contrib_sum), _stream(stream)))


def ocgs_render_fwd_reg(n, cam, cfg, ws, key_capacity, mask, color, alpha, depth, normal, n_contrib, loss_bg, vis_count, contrib_sum,
                        moments, stream=None):
    _ok("ocgs_render_fwd_reg", lib().ocgs_render_fwd_reg(C.c_int(n), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity),
                                                         _ptr(mask), _ptr(color), _ptr(alpha), _ptr(depth), _ptr(normal), _ptr(n_contrib),
                                                         _ptr(loss_bg), _ptr(vis_count), _ptr(contrib_sum), _ptr(moments), _stream(stream)))


def ocgs_render_bwd_reg(surfels, cam, cfg, ws, key_capacity, mask, n_contrib, dL_dcolor, dL_dalpha, dL_ddepth, dL_dnormal, moments, dL_dmoments,
                        d_pos, d_scale, d_quat, d_opacity, d_sh, d_center2d=None, stream=None):
    _ok("ocgs_render_bwd_reg", lib().ocgs_render_bwd_reg(C.byref(surfels), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity),
                                                         _ptr(mask), _ptr(n_contrib), _ptr(dL_dcolor), _ptr(dL_dalpha), _ptr(dL_ddepth),
                                                         _ptr(dL_dnormal), _ptr(moments), _ptr(dL_dmoments), _ptr(d_pos), _ptr(d_scale), _ptr(d_quat),
                                                         _ptr(d_opacity), _ptr(d_sh), _ptr(d_center2d), _stream(stream)))


def ocgs_render_bwd(surfels, cam, cfg, ws, key_capacity, mask, n_contrib, dL_dcolor, dL_dalpha, dL_ddepth, dL_dnormal, d_pos, d_scale,
                    d_quat, d_opacity, d_sh, d_center2d=None, stream=None):
    _ok("ocgs_render_bwd", lib().ocgs_render_bwd(C.byref(surfels), C.byref(cam), C.byref(cfg), _ptr(ws), C.c_size_t(key_capacity), _ptr(mask),
                                                 _ptr(n_contrib), _ptr(dL_dcolor), _ptr(dL_dalpha), _ptr(dL_ddepth), _ptr(dL_dnormal),
                                                 _ptr(d_pos), _ptr(d_scale), _ptr(d_quat), _ptr(d_opacity), _ptr(d_sh), _ptr(d_center2d),
                                                 _stream(stream)))


def ocgs_prune_workspace_bytes(n: int) -> int:
    return int(lib().ocgs_prune_workspace_bytes(C.c_int(n)))


def ocgs_prune_stats(surfels, vis_count, contrib_sum, cfg, prune_mask, remap, out: Optional[ocgs_surfels_mut], n_out, reset_stats, ws,
                     stream=None):
    _ok("ocgs_prune_stats", lib().ocgs_prune_stats(C.byref(surfels), _ptr(vis_count), _ptr(contrib_sum), C.byref(cfg), _ptr(prune_mask),
                                                   _ptr(remap), C.byref(out) if out is not None else None, _ptr(n_out),
                                                   C.c_int(int(reset_stats)), _ptr(ws), _stream(stream)))


def ocgs_densify_workspace_bytes(n: int) -> int:
    return int(lib().ocgs_densify_workspace_bytes(C.c_int(n)))


def ocgs_densify_accumulate(ws, n, width, height, key_capacity, d_center2d, grad_accum, denom, stream=None):
    _ok("ocgs_densify_accumulate", lib().ocgs_densify_accumulate(_ptr(ws), C.c_int(n), C.c_int(width), C.c_int(height), C.c_size_t(key_capacity),
                                                                 _ptr(d_center2d), _ptr(grad_accum), _ptr(denom), _stream(stream)))


def ocgs_densify(surfels, grad_accum, denom, grad_threshold, scale_threshold, xi, out: ocgs_surfels_mut, src, counts, scratch, stream=None):
    _ok("ocgs_densify", lib().ocgs_densify(C.byref(surfels), _ptr(grad_accum), _ptr(denom), C.c_float(grad_threshold), C.c_float(scale_threshold),
                                           _ptr(xi), C.byref(out), _ptr(src), _ptr(counts), _ptr(scratch), _stream(stream)))


def ocgs_compact_rows(inp, remap, n: int, row_floats: int, out, stream=None):
    _ok("ocgs_compact_rows", lib().ocgs_compact_rows(_ptr(inp), _ptr(remap), C.c_int(n), C.c_int(row_floats), _ptr(out), _stream(stream)))


def ocgs_step_view_host(surfels, cam, cfg, h_mask, h_target, h_losses, d_mask, d_images, d_ncontrib, d_grads, d_vis_count, d_contrib_sum,
                        d_losses, ws, key_capacity, stream=None, copy_stream=None):
    """h_*: pinned host tensors; d_grads: dict with d_pos, d_scale, d_quat, d_opacity, d_sh (device)."""
    def hp(t):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("expected a contiguous host tensor")
        return C.c_void_p(t.data_ptr())
    _ok("ocgs_step_view_host", lib().ocgs_step_view_host(C.byref(surfels), C.byref(cam), C.byref(cfg), hp(h_mask), hp(h_target), hp(h_losses),
                                                         _ptr(d_mask), _ptr(d_images), _ptr(d_ncontrib), _ptr(d_grads["d_pos"]),
                                                         _ptr(d_grads["d_scale"]), _ptr(d_grads["d_quat"]), _ptr(d_grads["d_opacity"]),
                                                         _ptr(d_grads["d_sh"]), _ptr(d_vis_count), _ptr(d_contrib_sum), _ptr(d_losses),
                                                         _ptr(ws), C.c_size_t(key_capacity), _stream(stream),
                                                         C.c_void_p(copy_stream.cuda_stream) if copy_stream is not None else None))


def ocgs_step_view_host_enqueue(surfels, cam, cfg, h_mask, h_target, h_losses, h_header, d_mask, d_images, d_ncontrib, d_grads, d_vis_count,
                                d_contrib_sum, d_losses, ws, key_capacity, stream=None, copy_stream=None):
    """ocgs_step_view_host without the closing synchronisation (stream-capturable).  h_header: pinned host int32[4] tensor or None;
    after synchronising, h_header[3] is the error word (bit 0: key capacity exceeded, bit 1: a tile list over 2^24 entries)."""
    def hp(t):
        if t is None:
            return None
        if t.is_cuda or not t.is_contiguous() or not t.is_pinned():
            raise ValueError("expected a contiguous page-locked host tensor")
        return C.c_void_p(t.data_ptr())
    _ok("ocgs_step_view_host_enqueue",
        lib().ocgs_step_view_host_enqueue(C.byref(surfels), C.byref(cam), C.byref(cfg), hp(h_mask), hp(h_target), hp(h_losses), hp(h_header),
                                          _ptr(d_mask), _ptr(d_images), _ptr(d_ncontrib), _ptr(d_grads["d_pos"]), _ptr(d_grads["d_scale"]),
                                          _ptr(d_grads["d_quat"]), _ptr(d_grads["d_opacity"]), _ptr(d_grads["d_sh"]), _ptr(d_vis_count),
                                          _ptr(d_contrib_sum), _ptr(d_losses), _ptr(ws), C.c_size_t(key_capacity), _stream(stream),
                                          C.c_void_p(copy_stream.cuda_stream) if copy_stream is not None else None))


def ocgs_step_view_prefetch_enqueue(surfels, cam, cfg, h_next_mask, h_next_target, h_losses, h_header, d_mask_cur, d_target_cur, d_mask_next,
                                    d_target_next, d_images, d_ncontrib, d_grads, d_vis_count, d_contrib_sum, d_losses, ws, key_capacity,
                                    stream=None, copy_stream=None):
    """The step on a view whose mask / target are already on the device, while the next view's are uploaded from pinned host
    memory on copy_stream (h_next_* = None: no prefetch).  Enqueue only; capturable."""
    def hp(t):
        if t is None:
            return None
        if t.is_cuda or not t.is_contiguous() or not t.is_pinned():
            raise ValueError("expected a contiguous page-locked host tensor")
        return C.c_void_p(t.data_ptr())
    _ok("ocgs_step_view_prefetch_enqueue",
        lib().ocgs_step_view_prefetch_enqueue(C.byref(surfels), C.byref(cam), C.byref(cfg), hp(h_next_mask), hp(h_next_target), hp(h_losses),
                                              hp(h_header), _ptr(d_mask_cur), _ptr(d_target_cur), _ptr(d_mask_next), _ptr(d_target_next),
                                              _ptr(d_images), _ptr(d_ncontrib), _ptr(d_grads["d_pos"]), _ptr(d_grads["d_scale"]),
                                              _ptr(d_grads["d_quat"]), _ptr(d_grads["d_opacity"]), _ptr(d_grads["d_sh"]), _ptr(d_vis_count),
                                              _ptr(d_contrib_sum), _ptr(d_losses), _ptr(ws), C.c_size_t(key_capacity), _stream(stream),
                                              C.c_void_p(copy_stream.cuda_stream) if copy_stream is not None else None))


def ocgs_step_host(h_pos, h_scale, h_quat, h_opacity, h_sh, n, cam, cfg, h_mask, h_target, h_grads, h_alpha, h_loss_bg, d_params,
                   d_mask, d_images, d_ncontrib, d_grads, d_vis_count, d_contrib_sum, d_loss_bg, ws, key_capacity, stream=None):
    def hp(t):
        return None if t is None else C.c_void_p(t.data_ptr())
    _ok("ocgs_step_host", lib().ocgs_step_host(hp(h_pos), hp(h_scale), hp(h_quat), hp(h_opacity), hp(h_sh), C.c_int(n), C.byref(cam),
                                               C.byref(cfg), hp(h_mask), hp(h_target), hp(h_grads), hp(h_alpha), hp(h_loss_bg),
                                               _ptr(d_params), _ptr(d_mask), _ptr(d_images), _ptr(d_ncontrib), _ptr(d_grads),
                                               _ptr(d_vis_count), _ptr(d_contrib_sum), _ptr(d_loss_bg), _ptr(ws),
                                               C.c_size_t(key_capacity), _stream(stream)))


def ocgs_masked_l1(color, target, mask, width, height, dL_dcolor, loss, ws, n, key_capacity, stream=None):
    _ok("ocgs_masked_l1", lib().ocgs_masked_l1(_ptr(color), _ptr(target), _ptr(mask), C.c_int(width), C.c_int(height), _ptr(dL_dcolor),
                                               _ptr(loss), _ptr(ws), C.c_int(n), C.c_size_t(key_capacity), _stream(stream)))


OCGS_MASKED_L1_STATIC_MAX_PIXELS = 2097152


def ocgs_masked_l1_static(color, target, mask, width, height, dL_dcolor, loss, stream=None):
    """ocgs_masked_l1 without a workspace: scratch in a static device array of the library, no allocation in the call."""
    code = lib().ocgs_masked_l1_static(_ptr(color), _ptr(target), _ptr(mask), C.c_int(width), C.c_int(height), _ptr(dL_dcolor), _ptr(loss),
                                       _stream(stream))
    if code == OCGS_ERR_CAPACITY:
        raise OcgsError(f"ocgs_masked_l1_static ({width}x{height} = {width * height} pixels exceed the static scratch: at most "
                        f"{OCGS_MASKED_L1_STATIC_MAX_PIXELS}; use ocgs_masked_l1 with a workspace)", code)
    _ok("ocgs_masked_l1_static", code)


def ocgs_regularizers_workspace_bytes(width: int, height: int) -> int:
    return int(lib().ocgs_regularizers_workspace_bytes(C.c_int(width), C.c_int(height)))


def ocgs_regularizers(alpha, depth, moments, normal, cam, w_d, w_n, dL_dalpha, dL_ddepth, dL_dmoments, dL_dnormal, loss, scratch, stream=None):
    _ok("ocgs_regularizers", lib().ocgs_regularizers(_ptr(alpha), _ptr(depth), _ptr(moments), _ptr(normal), C.byref(cam), C.c_float(w_d),
                                                     C.c_float(w_n), _ptr(dL_dalpha), _ptr(dL_ddepth), _ptr(dL_dmoments), _ptr(dL_dnormal),
                                                     _ptr(loss), _ptr(scratch), _stream(stream)))


def ocgs_photometric_workspace_bytes(width: int, height: int) -> int:
    return int(lib().ocgs_photometric_workspace_bytes(C.c_int(width), C.c_int(height)))


def ocgs_photometric_loss(color, target, mask, width, height, lambda_dssim, dL_dcolor, loss, scratch, stream=None):
    _ok("ocgs_photometric_loss", lib().ocgs_photometric_loss(_ptr(color), _ptr(target), _ptr(mask), C.c_int(width), C.c_int(height),
                                                             C.c_float(lambda_dssim), _ptr(dL_dcolor), _ptr(loss), _ptr(scratch),
                                                             _stream(stream)))


def ocgs_profile_begin(capacity: int, stream=None):
    _ok("ocgs_profile_begin", lib().ocgs_profile_begin(C.c_int(capacity), _stream(stream)))


def ocgs_profile_end(capacity: int, stream=None):
    """-> list of (kernel name, milliseconds) in launch order."""
    ms = (C.c_float * capacity)()
    names = C.create_string_buffer(capacity * 32)
    cnt = C.c_int(0)
    _ok("ocgs_profile_end", lib().ocgs_profile_end(_stream(stream), C.c_int(capacity), ms, names, C.byref(cnt)))
    raw = names.raw
    return [(raw[i * 32:(i + 1) * 32].split(b"\0", 1)[0].decode(), float(ms[i])) for i in range(cnt.value)]


def ocgs_peak_probe(kind: int, iters: int, out, stream=None) -> float:
    """Enqueue one launch of the FP32-FMA (kind 0) or MUFU.EX2 (kind 1) microbenchmark; -> operations of the launch."""
    ops = C.c_double(0.0)
    _ok("ocgs_peak_probe", lib().ocgs_peak_probe(C.c_int(kind), C.c_int(iters), _ptr(out), C.c_size_t(out.numel()), C.byref(ops), _stream(stream)))
    return float(ops.value)


def ocgs_staging_probe(kind: int, rec, ranks, n_rec: int, n_ranks: int, iters: int, out, stream=None) -> float:
    """Enqueue one launch of the staging microbenchmark (0: __ldg, 1: cp.async, 2: TMA gather4); -> record bytes it gathers."""
    nbytes = C.c_double(0.0)
    _ok("ocgs_staging_probe", lib().ocgs_staging_probe(C.c_int(kind), _ptr(rec), _ptr(ranks), C.c_uint(n_rec), C.c_uint(n_ranks), C.c_int(iters),
                                                        _ptr(out), C.c_size_t(out.numel()), C.byref(nbytes), _stream(stream)))
    return float(nbytes.value)


# ---- allocation helpers (device memory only; no arithmetic) --------------------------------------------------------

def alloc_workspace(n: int, width: int, height: int, key_capacity: int, device="cuda") -> torch.Tensor:
    nbytes = ocgs_workspace_bytes(n, width, height, key_capacity)
    if nbytes == 0:
        raise OcgsError("ocgs_workspace_bytes", OCGS_ERR_UNSUPPORTED)
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def ws_section(ws: torch.Tensor, layout: ocgs_ws_layout, name: str, dtype: torch.dtype, count: int) -> torch.Tensor:
    """View of a workspace section (see ocgs_ws_layout in include/ocgs.h)."""
    off = getattr(layout, name)
    nbytes = count * torch.empty(0, dtype=dtype).element_size()
    return ws[off:off + nbytes].view(dtype)


def alloc_outputs(width: int, height: int, device="cuda") -> Dict[str, torch.Tensor]:
    f = dict(dtype=torch.float32, device=device)
    return dict(color=torch.empty((3, height, width), **f), alpha=torch.empty((height, width), **f),
                depth=torch.empty((height, width), **f), normal=torch.empty((3, height, width), **f),
                n_contrib=torch.empty((height, width), dtype=torch.int32, device=device), loss_bg=torch.zeros(1, **f))


def alloc_grads(n: int, device="cuda") -> Dict[str, torch.Tensor]:
    f = dict(dtype=torch.float32, device=device)
    return dict(d_pos=torch.empty((n, 3), **f), d_scale=torch.empty((n, 2), **f), d_quat=torch.empty((n, 4), **f),
                d_opacity=torch.empty(n, **f), d_sh=torch.empty((n, 16, 3), **f), d_center2d=torch.empty((n, 2), **f))
