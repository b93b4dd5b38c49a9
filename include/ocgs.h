/* ocgs.h -- C ABI of libocgs: B200 (sm_100a) tile rasterizer for 2D Gaussian surfels, fused with the background
 * loss and the occlusion-aware pruning statistics of "Object-Centric 2D Gaussian Splatting" (arXiv 2501.08174).
 *
 * Citations are PAPER.md:<line> (the paper) or S<n>/O<n> (readings in DESIGN.md / SURVEY.md 8(c), used where the
 * paper defers the renderer mathematics to the cited 2DGS/3DGS work).
 *
 * Conventions
 *  - Every function returns 0 (OCGS_OK) or a negative error code.  Nothing throws, nothing prints.
 *  - "device" pointers are CUDA device memory owned by the caller; "host" pointers are ordinary host memory.
 *    The library allocates no device memory, keeps no global state and is re-entrant per stream.
 *  - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream).  No entry point
 *    synchronises except ocgs_check(), ocgs_profile_end(), ocgs_step_view_host() and ocgs_step_host().  A step can therefore be captured in a CUDA graph.
 *  - The data-dependent key count K never travels to the host inside a step: kernels read it from the workspace
 *    header.  If K exceeds `key_capacity` the header error flag is set, later calls of the step become no-ops, and
 *    ocgs_check() reports OCGS_ERR_CAPACITY with the needed size.  Limits: N and key_capacity below 2^30 (the radix
 *    passes carry counts in 30-bit status words); a single tile's list below 2^24 entries (list positions are packed
 *    with the hit bits handed to the backward pass), otherwise ocgs_check() reports OCGS_ERR_UNSUPPORTED.
 *  - Images are planar [C,H,W] fp32, row-major, origin top-left; integer pixel index (ix,iy) is the pixel centre,
 *    x_idx = fx X/Z + cx - 1/2 (S2).  Surfel parameters are ACTIVATED values: scale > 0, opacity in (0,1),
 *    quaternion (w,x,y,z) used through the polynomial R(q) without normalisation (S19).
 *  - Surfel arrays: pos[N,3], scale[N,2], quat[N,4], opacity[N], sh[N,16,3] fp32 (232 B per surfel).
 *    quat must be 16-byte aligned, scale 8-byte aligned (torch allocations are).
 */
#ifndef OCGS_H
#define OCGS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OCGS_OK 0
#define OCGS_ERR_INVALID_ARG (-1)
#define OCGS_ERR_CAPACITY (-2)    /* K > key_capacity (see ocgs_check) */
#define OCGS_ERR_CUDA (-3)        /* a CUDA runtime call failed; ocgs_last_cuda_error() has the cudaError_t */
#define OCGS_ERR_UNSUPPORTED (-4) /* tile != 16, sh_degree > 3, image or surfel count over the limits */

#define OCGS_MAX_DIM 32768        /* width, height <= this (pixel rects are stored as u16 pairs) */

/* world->camera pinhole camera (poses P_i in SE(3)); S2 */
typedef struct {
  float view[16]; /* row-major 4x4, camera looks down +z, x right, y down */
  float fx, fy;   /* focal lengths in pixels */
  float cx, cy;   /* principal point, corner-origin continuous coordinates (W/2, H/2 = centred) */
  int width, height;
} ocgs_camera;

/* constants of the method; ocgs_default_config() fills the defaults */
typedef struct {
  int tile;            /* 16 (S5); only 16 is supported */
  float near_z;        /* 0.2 (S3): cull centres at z <= near, skip hits at z < near */
  float alpha_min;     /* 1/255 (S11): pairs below this are skipped (expressed through rho_cut, S6) */
  float alpha_max;     /* 0.99 (S11): cap; gradient through the cap is zero (S12) */
  float t_min;         /* 1e-4 (S11): stop BEFORE blending the pair that would leave T(1-alpha) < t_min
                          ("terminated once ... p reaches a threshold opacity close to 1") */
  float rho_max;       /* 9 (S6): 3-sigma truncation */
  float filter_sigma2; /* 0.5 (S8): variance of the screen-space low-pass filter, in px^2 */
  float bg[3];         /* background colour (S13) */
  float gamma_bg;      /* 0.5: weight of L_b; render_bwd adds gamma (1-M)/(H W) to dL/dA */
  float tau_contrib;   /* 0 (S17): prune when contrib_sum <= tau */
  float min_opacity;   /* 0: prune when opacity < min_opacity */
  int sh_degree;       /* 0..3 (S14) */
} ocgs_config;

typedef struct {
  const float *pos, *scale, *quat, *opacity, *sh; /* device */
  int n;
} ocgs_surfels;

typedef struct {
  float *pos, *scale, *quat, *opacity, *sh; /* device, caller-allocated for `capacity` surfels */
  int capacity;
} ocgs_surfels_mut;

/* Byte offsets of the workspace sections (all 256-byte aligned), for inspection by tests and tools.  "by id" =
 * indexed by surfel id; "by rank" = indexed by position in the (depth bits, id) order of the visible surfels. */
typedef struct {
  size_t total_bytes;
  size_t header;        /* ocgs_header */
  size_t depth_bits;    /* u32 [N]    by id: IEEE bits of the view-space centre depth (Appendix A step 2) */
  size_t rect;          /* u16 [N,4]  by id: pixel rect ix0,iy0,ix1,iy1 inclusive; undefined when tiles == 0 */
  size_t tiles;         /* u32 [N]    by id: tiles touched, 0 = culled */
  size_t clamp;         /* u8  [N]    by id: bit c set when colour channel c was clamped at 0 */
  size_t rec_id;        /* f32 [N,24] by id: raster record */
  size_t id_to_rank;    /* u32 [N]    by id: rank, 0xFFFFFFFF when culled */
  size_t rank_to_id;    /* u32 [N]    by rank (first n_vis entries) */
  size_t rec;           /* f32 [N,24] by rank */
  size_t offsets;       /* u32 [N+1]  by rank: exclusive scan of tiles touched */
  size_t tile_keys;     /* u32 [key_capacity] tile id of each sorted list entry */
  size_t tile_vals;     /* u32 [key_capacity] rank of each sorted list entry */
  size_t ranges;        /* u32 [n_tiles,2] [start,end) of each tile's list */
  size_t grad_rec;      /* f32 [N,24] by rank: backward accumulators (20 used) */
  size_t loss_partial;  /* f32 [n_tiles] */
  size_t final_T;       /* f32 [H,W] transmittance left after the forward pass (exact, not 1 - alpha) */
  size_t scratch;       /* sort ping-pong buffers, histograms, scan partials */
} ocgs_ws_layout;

typedef struct {
  unsigned long long K; /* number of (tile, surfel) keys of the current view */
  unsigned int n_vis;   /* surfels that survived culling */
  unsigned int error;   /* bit 0: K > key_capacity */
} ocgs_header;

/* ---- host-only helpers ------------------------------------------------------------------------------------------ */
void ocgs_default_config(ocgs_config* cfg);
/* Fills `out`; returns OCGS_ERR_UNSUPPORTED when the sizes are over the limits. */
int ocgs_workspace_layout(int n, int width, int height, size_t key_capacity, ocgs_ws_layout* out);
size_t ocgs_workspace_bytes(int n, int width, int height, size_t key_capacity);
int ocgs_last_cuda_error(void);
/* Synchronises `stream`, copies the header to host.  Returns OCGS_ERR_CAPACITY if the error flag is set
 * (header_out->K then holds the capacity that was needed). header_out: host, may be NULL. */
int ocgs_check(const void* ws, void* stream, ocgs_header* header_out);

/* ---- (1) per-surfel preprocessing ------------------------------------------------------------------------------
 * PAPER.md:119 (4.3): "G_j is projected to the image and rasterized, identifying which pixels it can contribute
 * to"; a surfel outside the frustum "is disqualified from rendering and not assigned to any pixel".  O1 / Appendix A:
 * view transform, homography M = K'[s_u R t_u | s_v R t_v | p_c], cut-off rho_cut = min(rho_max, 2 ln(o/alpha_min)),
 * exact AABB of the projected rho_cut ellipse united with the filter disc, integer pixel rect, tile count,
 * facing normal, SH colour with clamp mask.  Writes ws sections depth_bits, rect, tiles, clamp, rec_id, id_to_rank
 * (all surfels) and the header (n_vis).  Integer outputs are bit-exact with the oracle (fp32 op order of Appendix A).
 * ws: device, ocgs_workspace_bytes() bytes, 256-byte aligned.  surfels/cam/cfg: host structs (device arrays inside). */
int ocgs_preprocess(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, void* ws,
                    size_t key_capacity, void* stream);

/* ---- (2) depth-ordered tile binning -----------------------------------------------------------------------------
 * PAPER.md:39 ("tile-based rasterization"), :119 ("rendered in front-to-back order"); O2/O3, S9.  Result: per-tile
 * lists ordered by (tile id, centre-depth bits, surfel id) and ranges[t] = [lower_bound(t), lower_bound(t+1)).
 * Two stable LSD radix sorts: all surfels by depth bits (ties keep id order), then the emitted
 * (tile, rank) keys by tile id.  Writes rank_to_id, rec, offsets, tile_keys, tile_vals, ranges and header.K.
 * sorted_ids: device u32 [key_capacity] or NULL; when given, receives the surfel id of each list entry. */
int ocgs_bin_sort(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                  uint32_t* sorted_ids, void* stream);

/* ---- (3) forward raster + background loss + visibility statistics ---------------------------------------------------
 * per pixel, "all assigned Gaussians are rendered in front-to-back order, accumulating their colors
 * and opacities"; stop rule S11; O4 ray-splat intersection in the surfel's (u,v) frame with the low-pass filter
 * rho = min(u^2+v^2, |x-c|^2/sigma_f^2) (S8).  Outputs (device): color[3,H,W] (+ T*bg), alpha[H,W] = 1-T (the
 * "accumulated alphas" A_i), depth[H,W] = sum w z (S10), normal[3,H,W] = sum w n, n_contrib[H,W] = list
 * position after the last blended pair; ws.final_T[H,W] = T.  loss_bg (device scalar, nullable; needs mask): Eq. 1, PAPER.md:99,
 * L_b = 1/(H W) sum A (1-M), deterministic reduction.  vis_count[N] / contrib_sum[N] (device, nullable): ACCUMULATE
 * (+=) the number of pixels that blended surfel j and sum of alpha*T ("we save which Gaussians are used
 * during the color accumulation step"; O8).  mask: device u8 [H,W], non-zero = object.  mask == NULL means ONE thing in every call
 * of this library: no mask, i.e. M = 1 everywhere (every pixel is object) -- L_b = 0 and no gamma (1-M)/(HW) term in the
 * backward pass, and the photometric terms cover the whole image. */
int ocgs_render_fwd(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                    float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg,
                    uint32_t* vis_count, float* contrib_sum, void* stream);

/* (3a) forward with the harness photometric term fused into the epilogue (S20; "M R vs M I L1 in the fwd
 * epilogue and dL/dC produced in-kernel"): = ocgs_render_fwd followed by ocgs_masked_l1(color, target, mask, ...), without
 * re-reading the colour map.  target: device f32 [3,H,W]; dL_dcolor: device f32 [3,H,W], OVERWRITTEN (bit-identical to
 * ocgs_masked_l1's); loss_l1: device f32 scalar, nullable (deterministic; its summation order differs from
 * ocgs_masked_l1's, so the two values agree to fp32 rounding, not bit for bit). */
int ocgs_render_fwd_l1(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                       const float* target, float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib,
                       float* loss_bg, float* loss_l1, float* dL_dcolor, uint32_t* vis_count, float* contrib_sum, void* stream);

/* ---- (4) backward ---------------------------------------------------------------------------------------------------
 * "Through backpropagation, the position, shape, and appearance of all involved Gaussians are updated";
 * occluded Gaussians receive no gradient (exact zeros).  O7.  Inputs: the forward's n_contrib (and the
 * lists, records and final transmittance that ocgs_render_fwd of the SAME view left in ws),
 * upstream gradients dL_dcolor[3,H,W], dL_dalpha[H,W], dL_ddepth[H,W], dL_dnormal[3,H,W] (device; any may be NULL = 0).
 * With mask != NULL and cfg->gamma_bg != 0 the gradient of gamma*L_b, gamma (1-M)/(H W), is added to dL/dA (mask == NULL: M = 1,
 * nothing is added -- the same meaning as in ocgs_render_fwd, whose L_b is then 0).
 * Outputs (device, OVERWRITTEN, zero for culled surfels): d_pos[N,3], d_scale[N,2], d_quat[N,4], d_opacity[N],
 * d_sh[N,16,3], d_center2d[N,2] (nullable) = M22 * (dL/dM02, dL/dM12), the gradient w.r.t. the projected centre at
 * fixed depth (densification statistic).  Uses ws.grad_rec as accumulator. */
int ocgs_render_bwd(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                    const uint8_t* mask, const uint32_t* n_contrib, const float* dL_dcolor,
                    const float* dL_dalpha, const float* dL_ddepth, const float* dL_dnormal, float* d_pos, float* d_scale,
                    float* d_quat, float* d_opacity, float* d_sh, float* d_center2d, void* stream);

/* ---- (3b)/(4b) forward / backward with the depth moments (reading R-moments) ---------------
 * The 2DGS regularisers the paper keeps unchanged (depth distortion L_d, normal consistency L_n) are
 * image-space functions of the rendered maps once the renderer also accumulates, per pixel, the depth moments
 *   moments[0] = c  (origin: depth of the pixel's first blended pair, 0 if none),
 *   moments[1] = m1 = sum_i w_i (z_i - c),   moments[2] = m2 = sum_i w_i (z_i - c)^2     (w_i = alpha_i T_i, z_i as in `depth`):
 *   sum_{i<j} w_i w_j (z_i - z_j)^2 = alpha * m2 - m1^2 for any origin; about c the difference is well conditioned in fp32.
 * ocgs_render_fwd_reg = ocgs_render_fwd + moments (device f32 [3,H,W], nullable = plain forward).
 * ocgs_render_bwd_reg = ocgs_render_bwd + moments (the forward's map) and dL_dmoments (device f32 [2,H,W]: upstream
 * gradients of m1 and m2, the origin held fixed); both NULL = plain backward, exactly one NULL = OCGS_ERR_INVALID_ARG. */
int ocgs_render_fwd_reg(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                        float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg,
                        uint32_t* vis_count, float* contrib_sum, float* moments, void* stream);
int ocgs_render_bwd_reg(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                        const uint8_t* mask, const uint32_t* n_contrib, const float* dL_dcolor, const float* dL_dalpha,
                        const float* dL_ddepth, const float* dL_dnormal, const float* moments, const float* dL_dmoments,
                        float* d_pos, float* d_scale, float* d_quat, float* d_opacity, float* d_sh, float* d_center2d, void* stream);

/* ---- regularisers of Eq. 3 (readings R-Ld, R-Ln) -------------------------
 * L_d = 1/(HW) sum_p (alpha m2 - m1^2) (depth distortion, squared pairwise form) and
 * L_n = 1/(HW) sum_p (alpha - normal . Nhat) (normal consistency; Nhat = camera-facing unit normal of the expected-depth
 * surface depth/alpha by central differences of the back-projected points, zero on the image border and next to pixels
 * with alpha <= 1e-4), unmasked.  Inputs: the maps of ocgs_render_fwd_reg (device f32; normal and moments [3,H,W]) and
 * the camera.  Outputs (device f32, OVERWRITTEN): dL_dalpha[H,W], dL_ddepth[H,W], dL_dmoments[2,H,W], dL_dnormal[3,H,W]
 * = gradients of w_d L_d + w_n L_n (pass them to ocgs_render_bwd_reg, adding other losses' gradients first if any);
 * loss: device f32[2] or NULL <- (L_d, L_n), unweighted, deterministic.
 * scratch: device memory of at least ocgs_regularizers_workspace_bytes(width, height), 256-B aligned. */
size_t ocgs_regularizers_workspace_bytes(int width, int height);
int ocgs_regularizers(const float* alpha, const float* depth, const float* moments, const float* normal, const ocgs_camera* cam,
                      float w_d, float w_n, float* dL_dalpha, float* dL_ddepth, float* dL_dmoments, float* dL_dnormal, float* loss,
                      void* scratch, void* stream);

/* ---- 3D-Gaussian variant of the visibility statistics (Appendix B; R-3D) ----
 * "We demonstrate the versatility of our pruning strategy by implementing it in 3DGS": the same forward walk, statistics
 * and prune rule on 3D Gaussians (mean, three scales, rotation, opacity, SH colour; EWA projection
 * Sigma' = J W Sigma W^T J^T + 0.3 I; a pair contributes iff (x-c)^T Sigma'^-1 (x-c) <= rho_cut).  Forward only.
 * ocgs3d_preprocess fills the same workspace sections as ocgs_preprocess; ocgs_bin_sort is then called unchanged;
 * ocgs3d_render_fwd = ocgs_render_fwd without the normal map (depth accumulates the Gaussians' centre depths).
 * Pruning: ocgs_prune_stats with a NULL `out` (only in->n and in->opacity are read) gives mask / remap / count, and
 * ocgs_compact_rows moves each parameter array (row lengths 3, 3, 4, 1, 48). */
typedef struct {
  const float* pos;      /* [N,3] */
  const float* scale;    /* [N,3] activated (> 0) standard deviations along the Gaussian's axes */
  const float* quat;     /* [N,4] (w,x,y,z) */
  const float* opacity;  /* [N] */
  const float* sh;       /* [N,16,3] */
  int n;
} ocgs_gaussians3d;
int ocgs3d_preprocess(const ocgs_gaussians3d* gaussians, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                      void* stream);
int ocgs3d_render_fwd(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                      float* color, float* alpha, float* depth, uint32_t* n_contrib, float* loss_bg, uint32_t* vis_count,
                      float* contrib_sum, void* stream);

/* ---- the visibility pass: statistics of one view, nothing else --------------------------------------------------------
 * PAPER.md:129 / :219 / :234: the pruning statistics come from "rendering all training views"; PAPER.md:119 defines what
 * is counted (a pair counts iff G_j is actually blended into the pixel, in front-to-back order, before the pixel stops).
 * ocgs_visibility_pass = (1) without the SH colour and the normal (surfels->sh is not read and may be NULL), (2), and the
 * walk of (3) without the colour / depth / normal blends, the maps, L_b and the blended lists: for every surfel j
 *   vis_count[j]   += number of pixels that blended it,      contrib_sum[j] += sum over those pixels of alpha_ij T_ij
 * exactly as ocgs_render_fwd accumulates them (vis_count bit-identical; contrib_sum up to the order of float atomics).
 * The workspace afterwards holds this view's lists but NO blended lists: do not call ocgs_render_bwd on it.
 * ocgs3d_visibility_pass: the same for 3D Gaussians (Appendix B).
 * vis_count u32[N], contrib_sum f32[N]: device, ACCUMULATED into.  Asynchronous on `stream`; errors as (1)-(3). */
int ocgs_visibility_pass(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                         uint32_t* vis_count, float* contrib_sum, void* stream);
int ocgs3d_visibility_pass(const ocgs_gaussians3d* gaussians, const ocgs_camera* cam, const ocgs_config* cfg, void* ws,
                           size_t key_capacity, uint32_t* vis_count, float* contrib_sum, void* stream);

/* ---- (5) prune statistics -> mask -> stream compaction ----------------------------------------------------------------
 * "We propose to assign both G_j and G_k with false" -- a surfel that was never blended in any render
 * of the interval is removed whether it was outside the frustum or occluded; PAPER.md:101 (opacity threshold), S17.
 * prune[j] = (vis_count[j]==0) | (contrib_sum[j] <= tau) | (opacity[j] < min_opacity).  Survivors keep ascending id
 * order: out[remap[j]] = in[j], remap[j] = -1 when pruned.  prune_mask u8[N], remap i32[N], n_out i32 (device scalar).
 * `out` may be NULL (mask/remap/count only).  reset_stats != 0 zeroes vis_count / contrib_sum afterwards.
 * ws: device scratch of at least ocgs_prune_workspace_bytes(n). */
size_t ocgs_prune_workspace_bytes(int n);
int ocgs_prune_stats(const ocgs_surfels* in, uint32_t* vis_count, float* contrib_sum, const ocgs_config* cfg,
                     uint8_t* prune_mask, int32_t* remap, const ocgs_surfels_mut* out, int* n_out, int reset_stats,
                     void* ws, void* stream);

/* Compaction of any other per-surfel array with the remap of ocgs_prune_stats (pruning happens every 100 /
 * 600 iterations INSIDE the optimisation, so optimiser moments and accumulated densification statistics must follow the
 * parameters): out[remap[j], :] = in[j, :] for remap[j] >= 0, rows of `row_floats` floats.
 * in, out: device f32 [n, row_floats], distinct buffers; rows of `out` beyond the survivor count are left untouched. */
int ocgs_compact_rows(const float* in, const int32_t* remap, int n, int row_floats, float* out, void* stream);

/* ---- clone / split densification (reading R-densify) ---------------------
 * ocgs_densify_accumulate: after ocgs_render_bwd of a view, grad_accum[j] += |(width/2, height/2) * d_center2d_j| (d_center2d is
 *   per pixel; the statistic is per NDC unit, the unit the default grad_threshold 2e-4 is calibrated in) and denom[j] += 1 for every
 *   surfel that passed this view's frustum test (read from the workspace of that view's ocgs_preprocess / ocgs_bin_sort).
 * ocgs_densify: avg = grad_accum / denom (0 if denom = 0); avg >= grad_threshold selects a surfel; selected surfels with
 *   max(scale) <= scale_threshold are CLONED, the others SPLIT into two children at p + s_u xi[j,k,0] t_u + s_v xi[j,k,1] t_v
 *   (xi: device f32 [N,2,2], standard normal numbers supplied by the caller) with scales / 1.6, the parent removed.
 *   `out` (capacity >= N, ideally 2 N) receives, in this order: non-split surfels (ascending id), clones (ascending id),
 *   children (ascending parent id, child 0 then 1); src (device i32 [capacity], nullable) the source id of each row;
 *   counts (device i32[4]) = (n_out, n_keep, n_clone, n_split).  Rows beyond out->capacity are dropped: the caller
 *   compares counts[0] with the capacity after synchronising.  ws: ocgs_densify_workspace_bytes(N) bytes of device scratch. */
size_t ocgs_densify_workspace_bytes(int n);
int ocgs_densify_accumulate(void* ws, int n, int width, int height, size_t key_capacity, const float* d_center2d, float* grad_accum,
                            uint32_t* denom, void* stream);
int ocgs_densify(const ocgs_surfels* in, const float* grad_accum, const uint32_t* denom, float grad_threshold, float scale_threshold,
                 const float* xi, const ocgs_surfels_mut* out, int32_t* src, int* counts, void* ws, void* stream);

/* ---- harness photometric term (S20; the L1 part of Eq. 2) --------------------------------------------
 * loss = 1/(3 H W) sum |M (R - I)| (device scalar, nullable), dL_dcolor[3,H,W] = M sign(R - I)/(3 H W).  color, target:
 * device [3,H,W]; mask device u8 [H,W], nullable (= all ones).  Uses ws.loss_partial as scratch (n, key_capacity: the values
 * the workspace was sized with). */
int ocgs_masked_l1(const float* color, const float* target, const uint8_t* mask, int width, int height, float* dL_dcolor,
                   float* loss, void* ws, int n, size_t key_capacity, void* stream);

/* The same term for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no workspace argument -- the per-block partial sums live in a 32 KB static device array inside the library (held by
 * every GPU that loads it until the process exits), and the call itself calls no cudaMalloc / cudaFree / allocating routine.
 * Arguments as ocgs_masked_l1 (color, target, dL_dcolor device f32 [3,H,W]; mask device u8 [H,W], nullable = all ones; loss device
 * f32 scalar, nullable); results bit-identical to ocgs_masked_l1's.  Limit: width * height <= OCGS_MASKED_L1_STATIC_MAX_PIXELS
 * (2 097 152, e.g. 1920x1080), beyond it OCGS_ERR_CAPACITY and nothing is launched.  The first call on a device looks the array's
 * address up (cudaGetSymbolAddress): make it before a capture starts.  All calls share the array: nothing in it has to start at
 * zero (a call writes every slot it reads), but calls that OVERLAP on the GPU -- different streams, parallel graph branches -- race
 * on it: serialise them.  Asynchronous on `stream`. */
#define OCGS_MASKED_L1_STATIC_MAX_PIXELS 2097152
int ocgs_masked_l1_static(const float* color, const float* target, const uint8_t* mask, int width, int height, float* dL_dcolor,
                          float* loss, void* stream);

/* ---- masked photometric loss L_c^M (Eq. 2) ---------------------------------------
 * L_c^M = L_c(I M, R M) with L_c = (1 - lambda) mean|x - y| + lambda (1 - mean SSIM(x, y)): the loss the paper takes from
 * "Equation 7 in the 3DGS paper" (reading S20b of DESIGN.md: SSIM of Wang et al. 2004 per channel over an
 * 11x11 Gaussian window, sigma 1.5, zero padding, C1 = 0.01^2, C2 = 0.03^2, both means over all 3 H W values).
 * color, target: device f32 [3,H,W]; mask: device u8 [H,W], nullable (= all ones), non-zero = object.
 * dL_dcolor: device f32 [3,H,W], OVERWRITTEN with dL_c^M/dcolor (zero outside the mask).
 * loss: device f32[3] or NULL; receives (L_c^M, its L1 term mean|x-y|, its D-SSIM term 1 - mean SSIM), deterministic.
 * scratch: device memory of at least ocgs_photometric_workspace_bytes(width, height), caller-owned, 256-B aligned.
 * Asynchronous on `stream`; returns OCGS_ERR_INVALID_ARG on null pointers / non-positive sizes / lambda outside [0,1]. */
size_t ocgs_photometric_workspace_bytes(int width, int height);
int ocgs_photometric_loss(const float* color, const float* target, const uint8_t* mask, int width, int height,
                          float lambda_dssim, float* dL_dcolor, float* loss, void* scratch, void* stream);

/* ---- diagnostics: per-launch device timing ----------------------------------------------------------------------------
 * Between ocgs_profile_begin and ocgs_profile_end every kernel (and memset) the library enqueues from the calling thread
 * is followed by a CUDA event; ocgs_profile_end synchronises `stream` and returns, for each launch in order, the
 * elapsed milliseconds since the previous mark (ms_out[max_out], host) and its name (names_out, host, 32 bytes each).
 * Thread-local; the only state the library keeps, and only while profiling. */
int ocgs_profile_begin(int capacity, void* stream);
int ocgs_profile_end(void* stream, int max_out, float* ms_out, char* names_out, int* count);

/* ---- diagnostics: measured ALU peaks of the device ("the builder must measure an FP32-FMA peak and a
 * MUFU.EX2 peak microbenchmark on the box and use those" for the rooflines of the raster kernels, PAPER.md:119 renderer) ----
 * Enqueues ONE launch of a microbenchmark on `stream`: kind 0 = eight independent chains of a <- fma(a, b, c) per thread
 * (2 flop per step; b, c uniform operands), kind 1 = eight chains of a <- -ex2(a) (one MUFU.EX2 per step), kind 2 = kind 0 with
 * b, c in registers (the three-register FFMA real kernels issue), kinds 3 / 4 = packed fma.rn.f32x2 chains (SASS FFMA2, 4 flop per
 * step) with b, c as scalars broadcast to both halves (kind 3) or as full pairs (kind 4); 8 blocks of 256 threads per SM,
 * `iters` x 8 steps per chain.  *ops_per_launch (host) receives the flop (kinds 0, 2, 3, 4) or EX2 (kind 1) count of the launch;
 * the caller times the launch with CUDA events and divides.
 * d_out: device f32[out_floats], out_floats >= 8 x 256 x number of SMs (OCGS_ERR_CAPACITY otherwise), scratch the kernels store
 * their results to.  Asynchronous; not part of any step. */
int ocgs_peak_probe(int kind, int iters, float* d_out, size_t out_floats, double* ops_per_launch, void* stream);

/* ---- diagnostics: the staging step of the raster kernels in isolation, three ways ("TMA where the layout
 * allows ... cp.async.bulk.tensor.2d ... tile::gather4 ... probe it, fall back to LDG.128 / cp.async"; the renderer is PAPER.md:119) ----
 * Enqueues ONE launch: 6 persistent CTAs of 256 threads per SM, each gathering `iters` batches of records (rows of `rec`, 24 floats =
 * 96 bytes each, selected by consecutive windows of `ranks`) into shared memory and reading a sixth of every batch back.
 * kind 0: __ldg + st.shared + __syncthreads, batches of 256 (what the raster kernels do); kind 1: cp.async 16 B, double-buffered
 * batches of 128; kind 2: TMA cp.async.bulk.tensor.2d tile::gather4 over a [n_rec, 24] fp32 tensor map + mbarrier, double-buffered
 * batches of 128 (needs a driver that exports cuTensorMapEncodeTiled, else OCGS_ERR_UNSUPPORTED).
 * rec: device f32 [n_rec, 24], 128-byte aligned; ranks: device u32 [n_ranks], every value < n_rec, n_ranks >= 256;
 * d_out: device f32 [out_floats], out_floats >= 6 x 256 x number of SMs: per-thread sums of what was read (the test's evidence that
 * the right rows arrived); *bytes_per_launch (host): record bytes gathered by the launch.  Asynchronous; not part of any step. */
int ocgs_staging_probe(int kind, const float* rec, const uint32_t* ranks, uint32_t n_rec, uint32_t n_ranks, int iters, float* d_out,
                       size_t out_floats, double* bytes_per_launch, void* stream);

/* ---- end-to-end TRAINING step: per-view inputs from the host, parameters resident on the device (bench.py "e2e") -------
 * What a training loop does per iteration (pick a view, render, losses, backpropagate): the model -- the
 * surfel parameters and their gradients -- lives in device memory (`surfels`, d_grad_*), the view's data come from the
 * host.  Copies the target image h_target [3,H,W] f32 and the mask h_mask [H,W] u8 from (pinned) host memory into
 * d_images / d_mask, runs (1)-(3) with L_b and the statistics on, ocgs_masked_l1, then (4) into the device gradient
 * arrays, copies the two loss scalars back into h_losses[0..1] = (L_b, masked L1) and synchronises.
 * d_images: device [14*H*W] floats (color 3, alpha 1, depth 1, normal 3, target 3, dL_dcolor 3); d_ncontrib u32 [H*W];
 * d_losses: device f32[2].  Every call of one step must pass the n, image size and key_capacity the workspace was sized with.
 * copy_stream (nullable): a second stream for the two uploads, so that they overlap preprocess / sort / forward (the
 * mask is awaited before the forward pass, the target before the photometric term); NULL = upload on `stream`. */
int ocgs_step_view_host(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask,
                        const float* h_target, float* h_losses, uint8_t* d_mask, float* d_images, uint32_t* d_ncontrib,
                        float* d_grad_pos, float* d_grad_scale, float* d_grad_quat, float* d_grad_opacity, float* d_grad_sh,
                        uint32_t* d_vis_count, float* d_contrib_sum, float* d_losses, void* ws, size_t key_capacity, void* stream,
                        void* copy_stream);
/* The same step WITHOUT the closing synchronisation: everything, including the copy of the two loss scalars into h_losses and
 * (if h_header is not NULL) of the workspace header into *h_header, is only enqueued; the caller synchronises `stream` and
 * then reads h_losses and checks h_header->error (bit 0: K > key_capacity, bit 1: a tile list over 2^24 entries).  h_mask,
 * h_target, h_losses and h_header must be page-locked.  The call contains no synchronising operation, so it can be
 * captured into a CUDA graph (cudaStreamBeginCapture on `stream`; copy_stream joins the capture through events) and the
 * graph replayed once per iteration for the same view: the uploads are memcpy nodes and happen on every replay. */
int ocgs_step_view_host_enqueue(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask,
                                const float* h_target, float* h_losses, ocgs_header* h_header, uint8_t* d_mask, float* d_images,
                                uint32_t* d_ncontrib, float* d_grad_pos, float* d_grad_scale, float* d_grad_quat, float* d_grad_opacity,
                                float* d_grad_sh, uint32_t* d_vis_count, float* d_contrib_sum, float* d_losses, void* ws,
                                size_t key_capacity, void* stream, void* copy_stream);

/* The step with the NEXT view's inputs prefetched (what a data loader does): this view's mask and target are already in
 * device memory (d_mask_cur, d_target_cur: put there by the previous call's prefetch, or by the caller for the first step);
 * while the step runs, h_next_mask / h_next_target (page-locked host, NULL = nothing to prefetch) are uploaded on
 * copy_stream into d_mask_next / d_target_next, off the critical path.  Because the target is resident when the forward
 * pass starts, the masked L1 is fused into it (ocgs_render_fwd_l1).  Otherwise as ocgs_step_view_host_enqueue: nothing
 * synchronises, losses and header come back through h_losses / h_header, the call is capturable into a CUDA graph.
 * d_images: device [11*H*W] floats (color 3, alpha 1, depth 1, normal 3, dL_dcolor 3); d_target_*: device [3*H*W] floats. */
int ocgs_step_view_prefetch_enqueue(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg,
                                    const uint8_t* h_next_mask, const float* h_next_target, float* h_losses, ocgs_header* h_header,
                                    const uint8_t* d_mask_cur, const float* d_target_cur, uint8_t* d_mask_next, float* d_target_next,
                                    float* d_images, uint32_t* d_ncontrib, float* d_grad_pos, float* d_grad_scale, float* d_grad_quat,
                                    float* d_grad_opacity, float* d_grad_sh, uint32_t* d_vis_count, float* d_contrib_sum,
                                    float* d_losses, void* ws, size_t key_capacity, void* stream, void* copy_stream);

/* ---- end-to-end step with HOST parameters (bench.py "e2e_host_params") ---------------------------------------------------------------
 * Copies the surfel parameters, mask and target image from (pinned) host memory to the given device staging buffers,
 * runs (1)-(3) with L_b and statistics on, ocgs_masked_l1, then (4); copies the gradients, the alpha map and loss_bg back
 * and synchronises.  Every pointer named h_* is host memory, d_* device memory owned by the caller.
 * h_grads: host [N*58] floats in the order pos(3N) scale(2N) quat(4N) opacity(N) sh(48N).  d_params and d_grads: device
 * staging of at least 58*N + 16 floats each (sections start on multiples of 4 floats).  key_capacity must be the value
 * the workspace was sized with (every call of one step passes the same n, image size and key_capacity).
 * d_images: device [14*H*W] floats (color 3, alpha 1, depth 1, normal 3, target 3, dL_dcolor 3); d_ncontrib u32 [H*W]. */
int ocgs_step_host(const float* h_pos, const float* h_scale, const float* h_quat, const float* h_opacity,
                   const float* h_sh, int n, const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask,
                   const float* h_target, float* h_grads, float* h_alpha, float* h_loss_bg, float* d_params,
                   uint8_t* d_mask, float* d_images, uint32_t* d_ncontrib, float* d_grads, uint32_t* d_vis_count,
                   float* d_contrib_sum, float* d_loss_bg, void* ws, size_t key_capacity, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* OCGS_H */
