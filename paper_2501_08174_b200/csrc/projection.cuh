// projection.cuh -- per-surfel projection (O1) and real SH basis (S14), device side.
// The integer-deciding part uses round-to-nearest intrinsics only, so nvcc cannot contract or re-associate it and
// rects / tile counts / depth keys are bit-identical to the fp32 sequence the paper-derived spec fixes.
#pragma once
#include "common.cuh"

namespace ocgs {

struct Projected {
  float M[9];      // row-major homography: local (u,v,1) -> homogeneous pixel-index coordinates
  float pc[3];     // view-space centre
  float cx, cy;    // c2d
  float rho_cut;
  float vu[3], vv[3];  // R_wc t_u, R_wc t_v (unscaled)
  int ix0, iy0, ix1, iy1;
  bool visible;
};

__device__ __forceinline__ float view_point_row(const float* V, int k, float x, float y, float z) {
  return __fmaf_rn(V[4 * k + 0], x, __fmaf_rn(V[4 * k + 1], y, __fmaf_rn(V[4 * k + 2], z, V[4 * k + 3])));
}
__device__ __forceinline__ float view_dir_row(const float* V, int k, float x, float y, float z) {
  return __fmaf_rn(V[4 * k + 0], x, __fmaf_rn(V[4 * k + 1], y, __fmul_rn(V[4 * k + 2], z)));
}

// Appendix A steps 1-8.
__device__ __forceinline__ void project_surfel(const float p[3], float su, float sv, float4 q, float o, const CamParams& cam,
                                               const ocgs_config& cfg, Projected& r) {
  r.visible = false;
  const float w = q.x, x = q.y, y = q.z, z = q.w;
  const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z), xy = __fmul_rn(x, y), xz = __fmul_rn(x, z),
              yz = __fmul_rn(y, z), wx = __fmul_rn(w, x), wy = __fmul_rn(w, y), wz = __fmul_rn(w, z);
  const float tu0 = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(yy, zz))), tu1 = __fmul_rn(2.0f, __fadd_rn(xy, wz)),
              tu2 = __fmul_rn(2.0f, __fsub_rn(xz, wy));
  const float tv0 = __fmul_rn(2.0f, __fsub_rn(xy, wz)), tv1 = __fsub_rn(1.0f, __fmul_rn(2.0f, __fadd_rn(xx, zz))),
              tv2 = __fmul_rn(2.0f, __fadd_rn(yz, wx));
  const float* V = cam.V;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    r.pc[k] = view_point_row(V, k, p[0], p[1], p[2]);
    r.vu[k] = view_dir_row(V, k, tu0, tu1, tu2);
    r.vv[k] = view_dir_row(V, k, tv0, tv1, tv2);
  }
  const float c0[3] = {__fmul_rn(su, r.vu[0]), __fmul_rn(su, r.vu[1]), __fmul_rn(su, r.vu[2])};
  const float c1[3] = {__fmul_rn(sv, r.vv[0]), __fmul_rn(sv, r.vv[1]), __fmul_rn(sv, r.vv[2])};
  float* M = r.M;
  M[0] = __fmaf_rn(cam.fx, c0[0], __fmul_rn(cam.ox, c0[2]));
  M[1] = __fmaf_rn(cam.fx, c1[0], __fmul_rn(cam.ox, c1[2]));
  M[2] = __fmaf_rn(cam.fx, r.pc[0], __fmul_rn(cam.ox, r.pc[2]));
  M[3] = __fmaf_rn(cam.fy, c0[1], __fmul_rn(cam.oy, c0[2]));
  M[4] = __fmaf_rn(cam.fy, c1[1], __fmul_rn(cam.oy, c1[2]));
  M[5] = __fmaf_rn(cam.fy, r.pc[1], __fmul_rn(cam.oy, r.pc[2]));
  M[6] = c0[2]; M[7] = c1[2]; M[8] = r.pc[2];
  r.rho_cut = 0.0f; r.cx = 0.0f; r.cy = 0.0f;
  if (!(r.pc[2] > cfg.near_z)) return;
  if (o < cfg.alpha_min) return;
  const double rr = 2.0 * log((double)o / (double)cfg.alpha_min);
  const float rc = (float)fmin((double)cfg.rho_max, rr);
  r.rho_cut = rc;
  const float a = __fmaf_rn(rc, __fmaf_rn(M[6], M[6], __fmul_rn(M[7], M[7])), -__fmul_rn(M[8], M[8]));
  if (!(a < 0.0f)) return;
  // conic tangents about the projected centre c2d (reading R-bbox: no cancellation in fp32), padded outwards
  r.cx = __fdiv_rn(M[2], M[8]);
  r.cy = __fdiv_rn(M[5], M[8]);
  const float c2[2] = {r.cx, r.cy};
  float m[2], h[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const float* Mr = M + 3 * k;
    const float nc = -c2[k];
    const float A0 = __fmaf_rn(nc, M[6], Mr[0]), A1 = __fmaf_rn(nc, M[7], Mr[1]), A2 = __fmaf_rn(nc, M[8], Mr[2]);
    const float b = __fmaf_rn(rc, __fmaf_rn(A0, M[6], __fmul_rn(A1, M[7])), -__fmul_rn(A2, M[8]));
    const float cc = __fmaf_rn(rc, __fmaf_rn(A0, A0, __fmul_rn(A1, A1)), -__fmul_rn(A2, A2));
    m[k] = __fdiv_rn(b, a);
    h[k] = __fsqrt_rn(fmaxf(0.0f, __fmaf_rn(m[k], m[k], -__fdiv_rn(cc, a))));
    h[k] = __fmaf_rn(h[k], 1.0000152587890625f, 0.0078125f);
  }
  const float rf = __fadd_rn(__fsqrt_rn(__fmul_rn(cfg.filter_sigma2, rc)), 0.0078125f);
  const float lim = 1073741824.0f;
  const int WH[2] = {cam.W, cam.H};
  int lo[2], hi[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    float mn = fminf(__fadd_rn(c2[k], __fsub_rn(m[k], h[k])), __fsub_rn(c2[k], rf));
    float mx = fmaxf(__fadd_rn(c2[k], __fadd_rn(m[k], h[k])), __fadd_rn(c2[k], rf));
    mn = fmaxf(-lim, fminf(lim, mn));
    mx = fmaxf(-lim, fminf(lim, mx));
    lo[k] = (int)ceilf(mn);
    hi[k] = (int)floorf(mx);
    if (hi[k] < 0 || lo[k] > WH[k] - 1 || lo[k] > hi[k]) return;
  }
  r.ix0 = max(lo[0], 0); r.iy0 = max(lo[1], 0);
  r.ix1 = min(hi[0], cam.W - 1); r.iy1 = min(hi[1], cam.H - 1);
  r.visible = true;
}

// Real SH basis constants (S14), rounded from sqrt closed forms: Y0 = 1/2 sqrt(1/pi), Y1 = sqrt(3/(4 pi)), ...
#define SH_K0 0.28209479177387814f
#define SH_K1 0.4886025119029199f
#define SH_K2A 1.0925484305920792f   /* 1/2 sqrt(15/pi) */
#define SH_K2B 0.31539156525252005f  /* 1/4 sqrt(5/pi) */
#define SH_K2C 0.5462742152960396f   /* 1/4 sqrt(15/pi) */
#define SH_K3A 0.5900435899266435f   /* 1/4 sqrt(35/(2 pi)) */
#define SH_K3B 2.890611442640554f    /* 1/2 sqrt(105/pi) */
#define SH_K3C 0.4570457994644658f   /* 1/4 sqrt(21/(2 pi)) */
#define SH_K3D 0.3731763325901154f   /* 1/4 sqrt(7/pi) */
#define SH_K3E 1.445305721320277f    /* 1/4 sqrt(105/pi) */

__device__ __forceinline__ void sh_basis(float x, float y, float z, int degree, float* Y) {
  Y[0] = SH_K0;
  if (degree < 1) return;
  Y[1] = -SH_K1 * y; Y[2] = SH_K1 * z; Y[3] = -SH_K1 * x;
  if (degree < 2) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  Y[4] = SH_K2A * x * y; Y[5] = -SH_K2A * y * z; Y[6] = SH_K2B * (2.0f * zz - xx - yy);
  Y[7] = -SH_K2A * x * z; Y[8] = SH_K2C * (xx - yy);
  if (degree < 3) return;
  Y[9] = -SH_K3A * y * (3.0f * xx - yy); Y[10] = SH_K3B * x * y * z; Y[11] = -SH_K3C * y * (4.0f * zz - xx - yy);
  Y[12] = SH_K3D * z * (2.0f * zz - 3.0f * xx - 3.0f * yy); Y[13] = -SH_K3C * x * (4.0f * zz - xx - yy);
  Y[14] = SH_K3E * z * (xx - yy); Y[15] = -SH_K3A * x * (xx - 3.0f * yy);
}

// DESIGN.md reading R-clamp: the colour sum whose sign decides the clamp bit is a FIXED fp32 sequence (round-to-nearest
// intrinsics only, so nvcc can neither contract nor re-associate it): dir = (p - campos) / sqrt(fma(dx,dx, fma(dy,dy, dz dz))),
// the basis below with the multiplication order written out, then acc_c = fma(Y_k, sh[k][c], acc_c) for k in order from 1/2.
__device__ __forceinline__ void sh_basis_rn(float x, float y, float z, int degree, float* Y) {
  Y[0] = SH_K0;
  if (degree < 1) return;
  Y[1] = __fmul_rn(-SH_K1, y); Y[2] = __fmul_rn(SH_K1, z); Y[3] = __fmul_rn(-SH_K1, x);
  if (degree < 2) return;
  const float xx = __fmul_rn(x, x), yy = __fmul_rn(y, y), zz = __fmul_rn(z, z);
  const float xx_yy = __fsub_rn(xx, yy);
  Y[4] = __fmul_rn(__fmul_rn(SH_K2A, x), y);
  Y[5] = __fmul_rn(__fmul_rn(-SH_K2A, y), z);
  Y[6] = __fmul_rn(SH_K2B, __fsub_rn(__fmaf_rn(2.0f, zz, -xx), yy));
  Y[7] = __fmul_rn(__fmul_rn(-SH_K2A, x), z);
  Y[8] = __fmul_rn(SH_K2C, xx_yy);
  if (degree < 3) return;
  const float b = __fsub_rn(__fmaf_rn(4.0f, zz, -xx), yy);
  Y[9] = __fmul_rn(__fmul_rn(-SH_K3A, y), __fmaf_rn(3.0f, xx, -yy));
  Y[10] = __fmul_rn(__fmul_rn(__fmul_rn(SH_K3B, x), y), z);
  Y[11] = __fmul_rn(__fmul_rn(-SH_K3C, y), b);
  Y[12] = __fmul_rn(__fmul_rn(SH_K3D, z), __fmaf_rn(-3.0f, yy, __fmaf_rn(-3.0f, xx, __fmul_rn(2.0f, zz))));
  Y[13] = __fmul_rn(__fmul_rn(-SH_K3C, x), b);
  Y[14] = __fmul_rn(__fmul_rn(SH_K3E, z), xx_yy);
  Y[15] = __fmul_rn(__fmul_rn(-SH_K3A, x), __fmaf_rn(-3.0f, yy, xx));
}

// SH colour of one surfel (S14) by the R-clamp sequence: col[c] = max(0, acc_c), bit c of the result set iff acc_c < 0
__device__ __forceinline__ uint8_t sh_colour_rn(const float p[3], const float4* __restrict__ shj, const CamParams& cam, int degree, float col[3]) {
  const float d0 = __fsub_rn(p[0], cam.campos[0]), d1 = __fsub_rn(p[1], cam.campos[1]), d2 = __fsub_rn(p[2], cam.campos[2]);
  const float len = __fsqrt_rn(__fmaf_rn(d0, d0, __fmaf_rn(d1, d1, __fmul_rn(d2, d2))));
  const float x = __fdiv_rn(d0, len), y = __fdiv_rn(d1, len), z = __fdiv_rn(d2, len);
  float Y[16];
  sh_basis_rn(x, y, z, degree, Y);
  const int nb = (degree + 1) * (degree + 1);
  col[0] = col[1] = col[2] = 0.5f;
  const int nvec = (3 * nb + 3) / 4;
  // the row is read in two batches of six 16-byte loads, all of a batch in flight together (a loop that stops at nvec issues them one
  // round trip after the other: 36 % of preprocess_kernel's stall samples); the sums keep their order
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    float4 f[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) f[i] = 6 * h + i < nvec ? __ldg(shj + 6 * h + i) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const float ff[4] = {f[i].x, f[i].y, f[i].z, f[i].w};
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int idx = 4 * (6 * h + i) + e;
        if (idx < 3 * nb) {
          const int k = idx / 3, c = idx - 3 * k;  // per channel the terms arrive in ascending k
          col[c] = __fmaf_rn(Y[k], ff[e], col[c]);
        }
      }
    }
  }
  uint8_t cl = 0;
#pragma unroll
  for (int c = 0; c < 3; ++c)
    if (col[c] < 0.0f) { col[c] = 0.0f; cl |= (uint8_t)(1u << c); }
  return cl;
}

// gradient of sum_k a_k Y_k(x,y,z) w.r.t. (x,y,z), the polynomials taken with x,y,z independent
__device__ __forceinline__ void sh_basis_grad(float x, float y, float z, int degree, const float* a, float* g) {
  g[0] = g[1] = g[2] = 0.0f;
  if (degree < 1) return;
  g[1] += -SH_K1 * a[1]; g[2] += SH_K1 * a[2]; g[0] += -SH_K1 * a[3];
  if (degree < 2) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  g[0] += SH_K2A * y * a[4]; g[1] += SH_K2A * x * a[4];
  g[1] += -SH_K2A * z * a[5]; g[2] += -SH_K2A * y * a[5];
  g[0] += -2.0f * SH_K2B * x * a[6]; g[1] += -2.0f * SH_K2B * y * a[6]; g[2] += 4.0f * SH_K2B * z * a[6];
  g[0] += -SH_K2A * z * a[7]; g[2] += -SH_K2A * x * a[7];
  g[0] += 2.0f * SH_K2C * x * a[8]; g[1] += -2.0f * SH_K2C * y * a[8];
  if (degree < 3) return;
  g[0] += -SH_K3A * 6.0f * x * y * a[9]; g[1] += -SH_K3A * (3.0f * xx - 3.0f * yy) * a[9];
  g[0] += SH_K3B * y * z * a[10]; g[1] += SH_K3B * x * z * a[10]; g[2] += SH_K3B * x * y * a[10];
  g[0] += SH_K3C * 2.0f * x * y * a[11]; g[1] += -SH_K3C * (4.0f * zz - xx - 3.0f * yy) * a[11]; g[2] += -SH_K3C * 8.0f * y * z * a[11];
  g[0] += -SH_K3D * 6.0f * x * z * a[12]; g[1] += -SH_K3D * 6.0f * y * z * a[12]; g[2] += SH_K3D * (6.0f * zz - 3.0f * xx - 3.0f * yy) * a[12];
  g[0] += -SH_K3C * (4.0f * zz - 3.0f * xx - yy) * a[13]; g[1] += SH_K3C * 2.0f * x * y * a[13]; g[2] += -SH_K3C * 8.0f * x * z * a[13];
  g[0] += SH_K3E * 2.0f * x * z * a[14]; g[1] += -SH_K3E * 2.0f * y * z * a[14]; g[2] += SH_K3E * (xx - yy) * a[14];
  g[0] += -SH_K3A * (3.0f * xx - 3.0f * yy) * a[15]; g[1] += SH_K3A * 6.0f * x * y * a[15];
}

}  // namespace ocgs
