// gaussian3d.cu -- ocgs3d_preprocess: the 3D-Gaussian variant of O1 (Appendix B: the visibility / prune
// statistics "in 3DGS"; reading R-3D).  EWA projection of Sigma = R diag(s^2) R^T to the
// screen, Sigma' = J W Sigma W^T J^T + 0.3 I, exact AABB of the rho_cut ellipse, SH colour.  It fills the same workspace
// sections as ocgs_preprocess (depth bits, rects, tile counts, sort keys, 96-byte records by id), so ocgs_bin_sort and the
// forward kernel's list machinery are reused unchanged; the forward kernel evaluates the record with the 3D pair rule.
// The integer-deciding part repeats, with round-to-nearest intrinsics, the fp32 sequence written out in
// oracle/ocgs_oracle.cpp ("3D-Gaussian variant"), so rects / tile counts / depth keys are bit-identical to the oracle's.
// Record (common.cuh slots): f4[0] = (conic_xx, conic_xy, conic_yy, 0), f4[2].zw = centre, f4[3] = (rho_cut, z_j, rect0, rect1),
// f4[4] = (opacity, r, g, b); everything else zero.
#include "projection.cuh"

namespace ocgs {

struct Projected3 {
  float conic[3], cx, cy, rho_cut, tz;
  int ix0, iy0, ix1, iy1;
  bool visible;
};

__device__ __forceinline__ void project_gaussian3d(const float p[3], const float s[3], float4 q, float o, const CamParams& cam,
                                                   const ocgs_config& cfg, Projected3& r) {
  r.visible = false;
  const float w = q.x, x = q.y, y = q.z, z = q.w;
  const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z), xy = __fmul_rn(x, y), xz = __fmul_rn(x, z),
              yz = __fmul_rn(y, z), wx = __fmul_rn(w, x), wy = __fmul_rn(w, y), wz = __fmul_rn(w, z);
  const float col[3][3] = {
      {__fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(yy, zz))), __fmul_rn(2.0f, __fadd_rn(xy, wz)), __fmul_rn(2.0f, __fsub_rn(xz, wy))},
      {__fmul_rn(2.0f, __fsub_rn(xy, wz)), __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, zz))), __fmul_rn(2.0f, __fadd_rn(yz, wx))},
      {__fmul_rn(2.0f, __fadd_rn(xz, wy)), __fmul_rn(2.0f, __fsub_rn(yz, wx)), __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, yy)))}};
  const float* V = cam.V;
  float t[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) t[k] = view_point_row(V, k, p[0], p[1], p[2]);
  r.tz = t[2];
  r.rho_cut = 0.f; r.cx = 0.f; r.cy = 0.f;
  if (!(t[2] > cfg.near_z)) return;
  if (o < cfg.alpha_min) return;
  float b[3][3];  // b[k] = s_k * W R e_k
#pragma unroll
  for (int k = 0; k < 3; ++k)
#pragma unroll
    for (int i = 0; i < 3; ++i) b[k][i] = __fmul_rn(s[k], view_dir_row(V, i, col[k][0], col[k][1], col[k][2]));
#define OCGS_S(i, j) __fmaf_rn(b[0][i], b[0][j], __fmaf_rn(b[1][i], b[1][j], __fmul_rn(b[2][i], b[2][j])))
  const float S00 = OCGS_S(0, 0), S01 = OCGS_S(0, 1), S02 = OCGS_S(0, 2), S11 = OCGS_S(1, 1), S12 = OCGS_S(1, 2), S22 = OCGS_S(2, 2);
#undef OCGS_S
  const float itz = __fdiv_rn(1.0f, t[2]);
  const float j00 = __fmul_rn(cam.fx, itz), j02 = -__fmul_rn(__fmul_rn(j00, t[0]), itz);
  const float j11 = __fmul_rn(cam.fy, itz), j12 = -__fmul_rn(__fmul_rn(j11, t[1]), itz);
  const float T0x = __fmaf_rn(j00, S00, __fmul_rn(j02, S02)), T0y = __fmaf_rn(j00, S01, __fmul_rn(j02, S12)),
              T0z = __fmaf_rn(j00, S02, __fmul_rn(j02, S22));
  const float T1y = __fmaf_rn(j11, S11, __fmul_rn(j12, S12)), T1z = __fmaf_rn(j11, S12, __fmul_rn(j12, S22));
  const float cxx = __fadd_rn(__fmaf_rn(T0x, j00, __fmul_rn(T0z, j02)), 0.3f);
  const float cxy = __fmaf_rn(T0y, j11, __fmul_rn(T0z, j12));
  const float cyy = __fadd_rn(__fmaf_rn(T1y, j11, __fmul_rn(T1z, j12)), 0.3f);
  const float det = __fmaf_rn(cxx, cyy, -__fmul_rn(cxy, cxy));
  if (!(det > 0.0f)) return;
  r.conic[0] = __fdiv_rn(cyy, det); r.conic[1] = -__fdiv_rn(cxy, det); r.conic[2] = __fdiv_rn(cxx, det);
  r.cx = __fmaf_rn(j00, t[0], cam.ox);
  r.cy = __fmaf_rn(j11, t[1], cam.oy);
  const double rr = 2.0 * log((double)o / (double)cfg.alpha_min);
  const float rc = (float)fmin((double)cfg.rho_max, rr);
  r.rho_cut = rc;
  const float h[2] = {__fmaf_rn(__fsqrt_rn(__fmul_rn(rc, cxx)), 1.0000152587890625f, 0.0078125f),
                      __fmaf_rn(__fsqrt_rn(__fmul_rn(rc, cyy)), 1.0000152587890625f, 0.0078125f)};
  const float lim = 1073741824.0f;
  const float c2[2] = {r.cx, r.cy};
  const int WH[2] = {cam.W, cam.H};
  int lo[2], hi[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const float mn = fmaxf(-lim, fminf(lim, __fsub_rn(c2[k], h[k])));
    const float mx = fmaxf(-lim, fminf(lim, __fadd_rn(c2[k], h[k])));
    lo[k] = (int)ceilf(mn);
    hi[k] = (int)floorf(mx);
    if (hi[k] < 0 || lo[k] > WH[k] - 1 || lo[k] > hi[k]) return;
  }
  r.ix0 = max(lo[0], 0); r.iy0 = max(lo[1], 0);
  r.ix1 = min(hi[0], cam.W - 1); r.iy1 = min(hi[1], cam.H - 1);
  r.visible = true;
}

__global__ void __launch_bounds__(256) preprocess3d_kernel(const float* __restrict__ pos, const float* __restrict__ scale,
                                                           const float4* __restrict__ quat, const float* __restrict__ opacity,
                                                           const float4* __restrict__ sh, int n, CamParams cam, ocgs_config cfg,
                                                           uint32_t* __restrict__ depth_bits, ushort4* __restrict__ rect,
                                                           uint32_t* __restrict__ tiles, uint8_t* __restrict__ clamp_bits,
                                                           float4* __restrict__ rec_id, uint32_t* __restrict__ id_to_rank,
                                                           uint32_t* __restrict__ sort_key, uint32_t* __restrict__ sort_val,
                                                           ocgs_header* __restrict__ header) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  bool vis = false;
  if (j < n) {
    const float p[3] = {pos[3 * j], pos[3 * j + 1], pos[3 * j + 2]};
    const float s[3] = {scale[3 * j], scale[3 * j + 1], scale[3 * j + 2]};
    const float o = opacity[j];
    Projected3 pr;
    project_gaussian3d(p, s, quat[j], o, cam, cfg, pr);
    vis = pr.visible;
    const uint32_t zb = __float_as_uint(pr.tz);
    depth_bits[j] = zb;
    sort_key[j] = vis ? zb : 0xFFFFFFFFu;
    sort_val[j] = (uint32_t)j;
    id_to_rank[j] = 0xFFFFFFFFu;
    uint32_t nt = 0;
    uint8_t cl = 0;
    if (vis) {
      const int tx0 = pr.ix0 >> 4, tx1 = (pr.ix1 >> 4) + 1, ty0 = pr.iy0 >> 4, ty1 = (pr.iy1 >> 4) + 1;
      nt = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
      rect[j] = make_ushort4((unsigned short)pr.ix0, (unsigned short)pr.iy0, (unsigned short)pr.ix1, (unsigned short)pr.iy1);
      float colr[3];
      cl = sh_colour_rn(p, sh + (size_t)j * 12, cam, cfg.sh_degree, colr);  // reading R-clamp: the fixed fp32 colour sequence
      float4* out = rec_id + (size_t)j * 6;
      out[0] = make_float4(pr.conic[0], pr.conic[1], pr.conic[2], 0.f);
      out[1] = make_float4(0.f, 0.f, 0.f, 0.f);
      out[2] = make_float4(0.f, 0.f, pr.cx, pr.cy);
      out[3] = make_float4(pr.rho_cut, pr.tz, __uint_as_float((uint32_t)pr.ix0 | ((uint32_t)pr.iy0 << 16)),
                           __uint_as_float((uint32_t)pr.ix1 | ((uint32_t)pr.iy1 << 16)));
      out[4] = make_float4(o, colr[0], colr[1], colr[2]);
      out[5] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    tiles[j] = nt;
    clamp_bits[j] = cl;
  }
  const unsigned ball = __ballot_sync(0xFFFFFFFFu, vis);
  if ((threadIdx.x & 31) == 0 && ball) atomicAdd(&header->n_vis, (unsigned)__popc(ball));
}

int launch_preprocess3d(const ocgs_gaussians3d& g, const CamParams& cam, const ocgs_config& cfg, Workspace& w, cudaStream_t st) {
  OCGS_CUDA_OK(cudaMemsetAsync(w.header, 0, sizeof(ocgs_header), st));
  if (g_prof_on) prof_mark(st, "memset_header");
  if (g.n == 0) return OCGS_OK;
  const int blocks = (int)div_up((size_t)g.n, 256);
  preprocess3d_kernel<<<blocks, 256, 0, st>>>(g.pos, g.scale, (const float4*)g.quat, g.opacity, (const float4*)g.sh, g.n, cam, cfg,
                                              w.depth_bits, w.rect, w.tiles, w.clamp, (float4*)w.rec_id, w.id_to_rank, w.dkeyA,
                                              w.rank_to_id, w.header);
  OCGS_LAUNCHED(st, "preprocess3d_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
