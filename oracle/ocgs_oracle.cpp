// ocgs_oracle.cpp -- CPU ORACLE. TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU implementation of the hot path of "Object-Centric 2D Gaussian
// Splatting" (Rogge & Stricker, arXiv 2501.08174): tile rasterisation of 2D Gaussian surfels with the
// background loss L_b (Eq. 1) and the occlusion-aware visibility statistics (PAPER.md:119,
// :129).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call this.  It shares no code, header, table or constant with the CUDA library and includes no CUDA
// header.  The product never falls back to it.
//
// Two paths:
//   TILED  orc_preprocess -> orc_bin_sort -> orc_render_fwd / orc_render_bwd -> orc_prune
//          follows steps O1..O9 in order.  O1's integer-deciding part is the fp32 sequence of
//          SURVEY.md Appendix A (so rects / tile counts / depth keys are well defined bit patterns);
//          everything per pixel is fp64 evaluated from the fp32 record (M, c2d, rho_cut).
//   BF     orc_bf_render: brute force, all fp64 from the raw parameters, explicit ray-plane
//          intersection, every (pixel, surfel) pair, exhaustive per-pixel sort by (centre depth, id).
//          It knows nothing about bounding boxes, tiles or M.  BF == TILED is a pin of the tile machinery;
//          central differences on BF pin the analytic backward.
//
// Parity pins: every function here is pinned by tests/test_oracle_*.py (closed forms, invariants,
// BF == TILED, finite differences, SH orthonormality).  No function is "parity unpinned".
//
// Passages followed are cited per function as PAPER.md:<line> (§/Eq.) or, where the paper defers to
// the cited 2DGS/3DGS work, as the DESIGN.md reading (S-numbers of SURVEY.md §8(c)).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct OrcCamera {
  float view[16];  // world->camera, row-major; +z forward, x right, y down (S2)
  float fx, fy, cx, cy;
  int width, height;
};

struct OrcConfig {
  int tile;             // 16 (S5)
  float near_z;         // 0.2 (S3)
  float alpha_min;      // 1/255 (S11)
  float alpha_max;      // 0.99 (S11)
  float t_min;          // 1e-4 (S11)
  float rho_max;        // 9 (S6)
  float filter_sigma2;  // sigma_f^2 = 0.5 (S8)
  float bg[3];          // background colour (S13)
  float gamma_bg;       // 0.5
  float tau_contrib;    // 0 (S17)
  float min_opacity;    // 0 (O9)
  int sh_degree;        // 0..3 (S14)
};

// Decision margins for the fragile-pixel policy (S22).  A pixel is flagged when any decision taken while
// walking its list is closer to its threshold than the margin.
struct OrcMargins {
  double rho_cut_abs;   // |rho - rho_cut|
  double near_rel;      // |z - near| / near
  double tmin_rel;      // |T(1-alpha) - t_min| / t_min
  double switch_rel;    // |rho3 - rho2| / max(rho, 1e-12)   (depth source switch, S10)
  double cap_abs;       // |o G - alpha_max|                  (gradient switch, S12)
  double eps32;         // unit used by the fp32 forward-error estimate of a pair (2^-23)
  double cond_abs;      // pixel flagged ill-conditioned when sum_i T_i * err_est_i exceeds this
};

}  // extern "C"

namespace {

// ------------------------------------------------------------------------------------------------
// O1 / Appendix A: fp32, IEEE-exact operations only, no contraction (compile with -ffp-contract=off).
// ------------------------------------------------------------------------------------------------
struct Pre {
  bool visible;
  float M[9];
  float c2d[2];
  float rho_cut;
  float depth;
  int rect[4];
};

inline void view_point(const float* V, const float* p, float* out) {
  for (int k = 0; k < 3; ++k)
    out[k] = std::fmaf(V[4 * k + 0], p[0], std::fmaf(V[4 * k + 1], p[1], std::fmaf(V[4 * k + 2], p[2], V[4 * k + 3])));
}
inline void view_dir(const float* V, const float* e, float* out) {
  for (int k = 0; k < 3; ++k)
    out[k] = std::fmaf(V[4 * k + 0], e[0], std::fmaf(V[4 * k + 1], e[1], V[4 * k + 2] * e[2]));
}

Pre preprocess_one(const float* p, const float* s, const float* q, float o, const OrcCamera& cam, const OrcConfig& cfg) {
  Pre r;
  std::memset(&r, 0, sizeof(r));
  r.visible = false;
  const float* V = cam.view;
  // step 1: rotation columns
  const float w = q[0], x = q[1], y = q[2], z = q[3];
  const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y, wz = w * z;
  const float tu[3] = {1.0f - 2.0f * (yy + zz), 2.0f * (xy + wz), 2.0f * (xz - wy)};
  const float tv[3] = {2.0f * (xy - wz), 1.0f - 2.0f * (xx + zz), 2.0f * (yz + wx)};
  // step 2: view transform; depth key
  float pc[3], vu[3], vv[3];
  view_point(V, p, pc);
  r.depth = pc[2];
  if (!(pc[2] > cfg.near_z)) return r;  // S3: centre behind near plane
  if (o < cfg.alpha_min) return r;      // S4: never reaches alpha_min
  view_dir(V, tu, vu);
  view_dir(V, tv, vv);
  // step 3: columns
  const float c0[3] = {s[0] * vu[0], s[0] * vu[1], s[0] * vu[2]};
  const float c1[3] = {s[1] * vv[0], s[1] * vv[1], s[1] * vv[2]};
  const float* c[3] = {c0, c1, pc};
  // step 4: M = K' [c0 | c1 | c2]
  const float ox = cam.cx - 0.5f, oy = cam.cy - 0.5f;
  float* M = r.M;
  for (int i = 0; i < 3; ++i) {
    M[0 + i] = std::fmaf(cam.fx, c[i][0], ox * c[i][2]);
    M[3 + i] = std::fmaf(cam.fy, c[i][1], oy * c[i][2]);
    M[6 + i] = c[i][2];
  }
  // step 5: cut-off (S6) -- the only transcendental, in double, rounded once
  const double rr = 2.0 * std::log((double)o / (double)cfg.alpha_min);
  const float rc = (float)std::fmin((double)cfg.rho_max, rr);
  r.rho_cut = rc;
  // step 6: conic tangents (S7), in coordinates CENTRED on the projected centre c2d (reading R-bbox).
  // The roots of a x^2 - 2 b x + c = 0 taken about the image origin (m^2 - c/a with m ~ 500, h ~ 3) cancel
  // catastrophically in fp32 (half-extent off by 1e-2 px, so the integer rect can MISS a contributing pixel and S7's
  // "conservative" fails); about c2d the same closed form has m' ~ 0 and -c'/a ~ h^2: no cancellation.
  const float a = std::fmaf(rc, std::fmaf(M[6], M[6], M[7] * M[7]), -(M[8] * M[8]));
  if (!(a < 0.0f)) return r;  // ellipse reaches the eye plane
  r.c2d[0] = M[2] / M[8];
  r.c2d[1] = M[5] / M[8];
  float m[2], h[2];
  for (int k = 0; k < 2; ++k) {
    const float* Mr = M + 3 * k;
    const float nc = -r.c2d[k];
    const float A0 = std::fmaf(nc, M[6], Mr[0]), A1 = std::fmaf(nc, M[7], Mr[1]), A2 = std::fmaf(nc, M[8], Mr[2]);  // M_r - c_r M_2
    const float b = std::fmaf(rc, std::fmaf(A0, M[6], A1 * M[7]), -(A2 * M[8]));
    const float cc = std::fmaf(rc, std::fmaf(A0, A0, A1 * A1), -(A2 * A2));
    m[k] = b / a;
    h[k] = std::sqrt(std::fmax(0.0f, std::fmaf(m[k], m[k], -(cc / a))));
    // outward pad (1 + 2^-16) h + 2^-7 px: far above the fp32 error of this sequence, far below a pixel; pixels
    // inside the pad but outside the ellipse are rejected by the per-pixel rho test (S6), so the image is unchanged
    h[k] = std::fmaf(h[k], 1.0000152587890625f, 0.0078125f);
  }
  // step 7: filter disc (S8), same absolute pad
  const float rf = std::sqrt(cfg.filter_sigma2 * rc) + 0.0078125f;
  // step 8: integer bounds
  const float lim = 1073741824.0f;
  const int WH[2] = {cam.width, cam.height};
  int lo[2], hi[2];
  for (int k = 0; k < 2; ++k) {
    float mn = std::fmin(r.c2d[k] + (m[k] - h[k]), r.c2d[k] - rf);
    float mx = std::fmax(r.c2d[k] + (m[k] + h[k]), r.c2d[k] + rf);
    mn = std::fmax(-lim, std::fmin(lim, mn));
    mx = std::fmax(-lim, std::fmin(lim, mx));
    lo[k] = (int)std::ceil(mn);
    hi[k] = (int)std::floor(mx);
    if (hi[k] < 0 || lo[k] > WH[k] - 1 || lo[k] > hi[k]) return r;
  }
  for (int k = 0; k < 2; ++k) {
    lo[k] = std::max(lo[k], 0);
    hi[k] = std::min(hi[k], WH[k] - 1);
  }
  r.rect[0] = lo[0]; r.rect[1] = lo[1]; r.rect[2] = hi[0]; r.rect[3] = hi[1];
  r.visible = true;
  return r;
}

// ------------------------------------------------------------------------------------------------
// Real spherical harmonics, degree <= 3 (S14), fp64, constants from their closed forms.
// ------------------------------------------------------------------------------------------------
struct SHConst {
  double c0, c1, c2a, c2b, c2c, c3a, c3b, c3c, c3d, c3e;
  SHConst() {
    const double pi = 3.14159265358979323846;
    c0 = 0.5 * std::sqrt(1.0 / pi);
    c1 = std::sqrt(3.0 / (4.0 * pi));
    c2a = 0.5 * std::sqrt(15.0 / pi);    // xy, yz, xz
    c2b = 0.25 * std::sqrt(5.0 / pi);    // 2zz-xx-yy
    c2c = 0.25 * std::sqrt(15.0 / pi);   // xx-yy
    c3a = 0.25 * std::sqrt(35.0 / (2.0 * pi));  // y(3xx-yy), x(xx-3yy)
    c3b = 0.5 * std::sqrt(105.0 / pi);          // xyz
    c3c = 0.25 * std::sqrt(21.0 / (2.0 * pi));  // y(4zz-xx-yy), x(4zz-xx-yy)
    c3d = 0.25 * std::sqrt(7.0 / pi);           // z(2zz-3xx-3yy)
    c3e = 0.25 * std::sqrt(105.0 / pi);         // z(xx-yy)
  }
};
const SHConst SHC;

// Y[16] and optionally the gradient of each polynomial w.r.t. (x,y,z) treated as independent variables.
void sh_basis(const double d[3], double Y[16], double dY[16][3]) {
  const double x = d[0], y = d[1], z = d[2];
  const double xx = x * x, yy = y * y, zz = z * z;
  Y[0] = SHC.c0;
  Y[1] = -SHC.c1 * y; Y[2] = SHC.c1 * z; Y[3] = -SHC.c1 * x;
  Y[4] = SHC.c2a * x * y; Y[5] = -SHC.c2a * y * z; Y[6] = SHC.c2b * (2 * zz - xx - yy);
  Y[7] = -SHC.c2a * x * z; Y[8] = SHC.c2c * (xx - yy);
  Y[9] = -SHC.c3a * y * (3 * xx - yy); Y[10] = SHC.c3b * x * y * z; Y[11] = -SHC.c3c * y * (4 * zz - xx - yy);
  Y[12] = SHC.c3d * z * (2 * zz - 3 * xx - 3 * yy); Y[13] = -SHC.c3c * x * (4 * zz - xx - yy);
  Y[14] = SHC.c3e * z * (xx - yy); Y[15] = -SHC.c3a * x * (xx - 3 * yy);
  if (!dY) return;
  auto set = [&](int k, double gx, double gy, double gz) { dY[k][0] = gx; dY[k][1] = gy; dY[k][2] = gz; };
  set(0, 0, 0, 0);
  set(1, 0, -SHC.c1, 0); set(2, 0, 0, SHC.c1); set(3, -SHC.c1, 0, 0);
  set(4, SHC.c2a * y, SHC.c2a * x, 0);
  set(5, 0, -SHC.c2a * z, -SHC.c2a * y);
  set(6, -2 * SHC.c2b * x, -2 * SHC.c2b * y, 4 * SHC.c2b * z);
  set(7, -SHC.c2a * z, 0, -SHC.c2a * x);
  set(8, 2 * SHC.c2c * x, -2 * SHC.c2c * y, 0);
  set(9, -SHC.c3a * 6 * x * y, -SHC.c3a * (3 * xx - 3 * yy), 0);
  set(10, SHC.c3b * y * z, SHC.c3b * x * z, SHC.c3b * x * y);
  set(11, SHC.c3c * 2 * x * y, -SHC.c3c * (4 * zz - xx - 3 * yy), -SHC.c3c * 8 * y * z);
  set(12, -SHC.c3d * 6 * x * z, -SHC.c3d * 6 * y * z, SHC.c3d * (6 * zz - 3 * xx - 3 * yy));
  set(13, -SHC.c3c * (4 * zz - 3 * xx - yy), SHC.c3c * 2 * x * y, -SHC.c3c * 8 * x * z);
  set(14, SHC.c3e * 2 * x * z, -SHC.c3e * 2 * y * z, SHC.c3e * (xx - yy));
  set(15, -SHC.c3a * (3 * xx - 3 * yy), SHC.c3a * 6 * x * y, 0);
}

struct Rot { double tu[3], tv[3], tw[3]; };
Rot rot_from_quat(const double q[4]) {  // S19: polynomial R(q), no normalisation
  const double w = q[0], x = q[1], y = q[2], z = q[3];
  Rot r;
  r.tu[0] = 1 - 2 * (y * y + z * z); r.tu[1] = 2 * (x * y + w * z); r.tu[2] = 2 * (x * z - w * y);
  r.tv[0] = 2 * (x * y - w * z); r.tv[1] = 1 - 2 * (x * x + z * z); r.tv[2] = 2 * (y * z + w * x);
  r.tw[0] = 2 * (x * z + w * y); r.tw[1] = 2 * (y * z - w * x); r.tw[2] = 1 - 2 * (x * x + y * y);
  return r;
}
inline void mat3_vec(const float* V, const double* e, double* out) {  // rotation part of the view matrix
  for (int k = 0; k < 3; ++k) out[k] = (double)V[4 * k] * e[0] + (double)V[4 * k + 1] * e[1] + (double)V[4 * k + 2] * e[2];
}
inline void mat3T_vec(const float* V, const double* e, double* out) {
  for (int k = 0; k < 3; ++k) out[k] = (double)V[k] * e[0] + (double)V[4 + k] * e[1] + (double)V[8 + k] * e[2];
}
inline void cam_position(const float* V, double* c) {  // -R^T t
  const double t[3] = {(double)V[3], (double)V[7], (double)V[11]};
  mat3T_vec(V, t, c);
  for (int k = 0; k < 3; ++k) c[k] = -c[k];
}
inline double dot3(const double* a, const double* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
inline void cross3(const double* a, const double* b, double* o) {
  o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}
inline uint32_t float_bits(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }

// colour (S14): rgb = max(0, 1/2 + sum_k Y_k(dir) sh_k), dir = normalise(p - cam_pos); clamp bit c set when channel c is clamped.
// The clamp is a DECISION (zero gradient on clamped channels, S12), and where floating point decides a bit both sides take
// the decision in the same precision: DESIGN.md reading R-clamp fixes the fp32 sequence below (IEEE-exact single operations
// only: +, -, x, /, sqrt, fma; this file compiles with -ffp-contract=off).  The colour VALUE stays fp64 (surfel_colour).
//   d = p - campos (campos: fp64 -R^T t of the fp32 view entries, rounded once);  n2 = fma(dx,dx, fma(dy,dy, dz*dz));
//   len = sqrt(n2);  (x,y,z) = d / len;  xx = x*x, yy = y*y, zz = z*z;  K* = fp32 roundings of the closed forms of S14;
//   Y0 = K0;  Y1 = (-K1)*y;  Y2 = K1*z;  Y3 = (-K1)*x;
//   Y4 = (K2A*x)*y;  Y5 = ((-K2A)*y)*z;  Y6 = K2B*(fma(2,zz,-xx) - yy);  Y7 = ((-K2A)*x)*z;  Y8 = K2C*(xx - yy);
//   Y9 = ((-K3A)*y)*fma(3,xx,-yy);  Y10 = ((K3B*x)*y)*z;  b = fma(4,zz,-xx) - yy;  Y11 = ((-K3C)*y)*b;
//   Y12 = (K3D*z)*fma(-3,yy, fma(-3,xx, 2*zz));  Y13 = ((-K3C)*x)*b;  Y14 = (K3E*z)*(xx - yy);  Y15 = ((-K3A)*x)*fma(-3,yy,xx);
//   acc_c = 1/2;  for k = 0 .. (degree+1)^2 - 1 in order: acc_c = fma(Y_k, sh[k][c], acc_c);   channel c clamped  <=>  acc_c < 0.
void colour_f32(const float* p, const float* sh, int degree, const double* campos, float acc[3]) {
  const float k0 = (float)SHC.c0, k1 = (float)SHC.c1, k2a = (float)SHC.c2a, k2b = (float)SHC.c2b, k2c = (float)SHC.c2c,
              k3a = (float)SHC.c3a, k3b = (float)SHC.c3b, k3c = (float)SHC.c3c, k3d = (float)SHC.c3d, k3e = (float)SHC.c3e;
  const float d0 = p[0] - (float)campos[0], d1 = p[1] - (float)campos[1], d2 = p[2] - (float)campos[2];
  const float len = std::sqrt(std::fmaf(d0, d0, std::fmaf(d1, d1, d2 * d2)));
  const float x = d0 / len, y = d1 / len, z = d2 / len;
  const float xx = x * x, yy = y * y, zz = z * z;
  float Y[16];
  Y[0] = k0;
  Y[1] = (-k1) * y; Y[2] = k1 * z; Y[3] = (-k1) * x;
  Y[4] = (k2a * x) * y; Y[5] = ((-k2a) * y) * z; Y[6] = k2b * (std::fmaf(2.0f, zz, -xx) - yy); Y[7] = ((-k2a) * x) * z; Y[8] = k2c * (xx - yy);
  const float b = std::fmaf(4.0f, zz, -xx) - yy;
  Y[9] = ((-k3a) * y) * std::fmaf(3.0f, xx, -yy); Y[10] = ((k3b * x) * y) * z; Y[11] = ((-k3c) * y) * b;
  Y[12] = (k3d * z) * std::fmaf(-3.0f, yy, std::fmaf(-3.0f, xx, 2.0f * zz)); Y[13] = ((-k3c) * x) * b; Y[14] = (k3e * z) * (xx - yy);
  Y[15] = ((-k3a) * x) * std::fmaf(-3.0f, yy, xx);
  const int nb = (degree + 1) * (degree + 1);
  for (int c = 0; c < 3; ++c) {
    float a = 0.5f;
    for (int k = 0; k < nb; ++k) a = std::fmaf(Y[k], sh[3 * k + c], a);
    acc[c] = a;
  }
}

void surfel_colour(const float* p, const float* sh, int degree, const double* campos, double* rgb, uint8_t* clamp, double* unclamped = nullptr) {
  double v[3] = {p[0] - campos[0], p[1] - campos[1], p[2] - campos[2]};
  const double len = std::sqrt(dot3(v, v));
  double d[3] = {v[0] / len, v[1] / len, v[2] / len};
  double Y[16];
  sh_basis(d, Y, nullptr);
  const int nb = (degree + 1) * (degree + 1);
  float dec[3];
  colour_f32(p, sh, degree, campos, dec);
  *clamp = 0;
  for (int c = 0; c < 3; ++c) {
    double acc = 0.5;
    for (int k = 0; k < nb; ++k) acc += Y[k] * (double)sh[3 * k + c];
    if (unclamped) unclamped[c] = acc;
    if (dec[c] < 0.0f) { acc = 0.0; *clamp |= (uint8_t)(1u << c); }  // the decision: R-clamp (fp32 sequence)
    rgb[c] = acc < 0.0 ? 0.0 : acc;  // a channel the fp32 decision left open while the fp64 value is (by < 4e-6) negative
  }
}

// facing normal in view space (O1): n = R_wc t_w, flipped when n . p_c > 0.  Returns the sign applied.
double surfel_normal(const float* q, const float* V, const double* pc, double* n) {
  const double qd[4] = {q[0], q[1], q[2], q[3]};
  const Rot r = rot_from_quat(qd);
  mat3_vec(V, r.tw, n);
  double sgn = 1.0;
  if (dot3(n, pc) > 0.0) { sgn = -1.0; for (int k = 0; k < 3; ++k) n[k] = -n[k]; }
  return sgn;
}

// ------------------------------------------------------------------------------------------------
// O4: one (pixel, surfel) pair from the fp32 record, fp64 arithmetic.
// ------------------------------------------------------------------------------------------------
struct PairEval {
  bool valid;      // passes q_z != 0, near and cut-off tests
  bool surf;       // rho3 <= rho2 (surfel term wins)
  bool capped;     // o G > alpha_max
  bool fragile;
  double u, v, qz, k[3], l[3], rho, z, G, alpha, dx, dy;
  double drho_est; // fp32 forward-error estimate of rho for this pair
  double err_est;  // a-priori bound on |delta alpha| (+ relative depth term) of an fp32 evaluation of this pair
};

inline PairEval eval_pair(double x, double y, const float* Mf, const float* c2df, float rho_cut_f, float of,
                          const OrcConfig& cfg, const OrcMargins* mg) {
  PairEval e;
  e.valid = false; e.fragile = false; e.surf = true; e.capped = false; e.err_est = 0.0; e.drho_est = 0.0;
  double M[9];
  for (int i = 0; i < 9; ++i) M[i] = Mf[i];
  for (int i = 0; i < 3; ++i) { e.k[i] = x * M[6 + i] - M[i]; e.l[i] = y * M[6 + i] - M[3 + i]; }
  double q[3];
  cross3(e.k, e.l, q);
  e.qz = q[2];
  if (q[2] == 0.0) return e;
  e.u = q[0] / q[2]; e.v = q[1] / q[2];
  const double rho3 = e.u * e.u + e.v * e.v;
  e.dx = x - (double)c2df[0]; e.dy = y - (double)c2df[1];
  const double rho2 = (e.dx * e.dx + e.dy * e.dy) / (double)cfg.filter_sigma2;
  e.surf = rho3 <= rho2;
  e.rho = e.surf ? rho3 : rho2;
  e.z = e.surf ? (M[6] * e.u + M[7] * e.v + M[8]) : M[8];
  const double near = cfg.near_z, rc = rho_cut_f;
  double drho3 = 0.0, drho2 = 0.0, dz3 = 0.0;
  if (mg && mg->eps32 > 0.0 && e.rho <= 2.0 * rc + 1.0) {
    // Forward error of evaluating this pair in fp32 from the fp32 record, first order, for the centred form
    // k = (x - c)*M2 - (M0 - c*M2) (no large-number cancellation in forming k).  For surfels seen almost edge-on
    // q_z = k0 l1 - k1 l0 cancels and the map record -> alpha is intrinsically ill-conditioned.
    const double ep = mg->eps32, cx = c2df[0], cy = c2df[1];
    double dk[3], dl[3], dq[3];
    for (int i = 0; i < 2; ++i) {
      dk[i] = ep * (std::fabs(e.dx * M[6 + i]) + std::fabs(M[i]) + std::fabs(cx * M[6 + i]));
      dl[i] = ep * (std::fabs(e.dy * M[6 + i]) + std::fabs(M[3 + i]) + std::fabs(cy * M[6 + i]));
    }
    dk[2] = ep * std::fabs(e.dx * M[8]);
    dl[2] = ep * std::fabs(e.dy * M[8]);
    const double* k = e.k; const double* l = e.l;
    auto A = [](double v) { return std::fabs(v); };
    dq[0] = A(l[2]) * dk[1] + A(k[1]) * dl[2] + A(l[1]) * dk[2] + A(k[2]) * dl[1] + ep * (A(k[1] * l[2]) + A(k[2] * l[1]));
    dq[1] = A(l[0]) * dk[2] + A(k[2]) * dl[0] + A(l[2]) * dk[0] + A(k[0]) * dl[2] + ep * (A(k[2] * l[0]) + A(k[0] * l[2]));
    dq[2] = A(l[1]) * dk[0] + A(k[0]) * dl[1] + A(l[0]) * dk[1] + A(k[1]) * dl[0] + ep * (A(k[0] * l[1]) + A(k[1] * l[0]));
    const double du = (dq[0] + A(e.u) * dq[2]) / A(e.qz) + ep * A(e.u), dv = (dq[1] + A(e.v) * dq[2]) / A(e.qz) + ep * A(e.v);
    drho3 = 2.0 * (A(e.u) * du + A(e.v) * dv);
    dz3 = A(M[6]) * du + A(M[7]) * dv;
    drho2 = 4.0 * ep * rho2;
  }
  const double drho = e.surf ? drho3 : drho2, dz = e.surf ? dz3 : 0.0;
  if (mg) {
    // S22: a decision is fragile when it is within its margin -- a few fp32 ulps of the quantity, or, for a pair whose fp32
    // evaluation is ill-conditioned (surfel seen almost edge-on), that pair's own first-order error estimate if larger.
    // the switch only matters if the pair can be blended under either reading
    const double m_cut = std::fmax(mg->rho_cut_abs, drho), m_near = std::fmax(mg->near_rel * near, dz);
    if (std::fabs(rho3 - rho2) <= std::fmax(mg->switch_rel * std::fmax(e.rho, 1e-12), drho3 + drho2) && e.rho <= rc + m_cut) e.fragile = true;
    if (std::fabs(e.z - near) <= m_near && e.rho <= rc + m_cut) e.fragile = true;
    if (std::fabs(e.rho - rc) <= m_cut && e.z >= near - m_near) e.fragile = true;
  }
  if (e.z < near) return e;
  if (e.rho > rc) return e;
  e.G = std::exp(-0.5 * e.rho);
  const double araw = (double)of * e.G;
  e.capped = araw > (double)cfg.alpha_max;
  e.alpha = e.capped ? (double)cfg.alpha_max : araw;
  if (mg && std::fabs(araw - (double)cfg.alpha_max) <= std::fmax(mg->cap_abs, 0.5 * araw * drho)) e.fragile = true;
  e.valid = true;
  if (mg && mg->eps32 > 0.0) {
    e.drho_est = drho;
    const double dalpha = e.capped ? 0.0 : 0.5 * e.alpha * drho;
    e.err_est = dalpha + e.alpha * dz / std::fmax(1.0, std::fabs(e.z));
  }
  return e;
}

}  // namespace

extern "C" {

// ------------------------------------------------------------------------------------------------
// O1 preprocess.  PAPER.md:119 (§4.3): "G_j is projected to the image and rasterized, identifying
// which pixels it can contribute to"; out-of-frustum surfels are "disqualified from rendering".
// Outputs per surfel: visible flag, depth key bits, pixel rect (ix0,iy0,ix1,iy1 inclusive), tile count,
// M (row-major 3x3), c2d, rho_cut (fp32, Appendix A); facing normal and colour (fp64), clamp bits.
// ------------------------------------------------------------------------------------------------
void orc_preprocess(int n, const float* pos, const float* scale, const float* quat, const float* opacity, const float* sh,
                    const OrcCamera* cam, const OrcConfig* cfg, uint8_t* visible, uint32_t* depth_bits, int32_t* rect,
                    uint32_t* tiles_touched, float* M, float* c2d, float* rho_cut, double* normal, double* rgb, uint8_t* clamp) {
  double campos[3];
  cam_position(cam->view, campos);
#pragma omp parallel for schedule(static)
  for (int j = 0; j < n; ++j) {
    const Pre r = preprocess_one(pos + 3 * j, scale + 2 * j, quat + 4 * j, opacity[j], *cam, *cfg);
    visible[j] = r.visible ? 1 : 0;
    depth_bits[j] = float_bits(r.depth);
    std::memcpy(M + 9 * j, r.M, sizeof(r.M));
    c2d[2 * j] = r.c2d[0]; c2d[2 * j + 1] = r.c2d[1];
    rho_cut[j] = r.rho_cut;
    for (int k = 0; k < 4; ++k) rect[4 * j + k] = r.visible ? r.rect[k] : 0;
    tiles_touched[j] = 0;
    clamp[j] = 0;
    for (int k = 0; k < 3; ++k) { normal[3 * j + k] = 0; rgb[3 * j + k] = 0; }
    if (!r.visible) continue;
    const int T = cfg->tile;
    const int tx0 = r.rect[0] / T, tx1 = r.rect[2] / T + 1, ty0 = r.rect[1] / T, ty1 = r.rect[3] / T + 1;
    tiles_touched[j] = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
    // view-space centre in fp64 for the facing test
    const float* V = cam->view;
    double pcd[3];
    for (int k = 0; k < 3; ++k)
      pcd[k] = (double)V[4 * k] * pos[3 * j] + (double)V[4 * k + 1] * pos[3 * j + 1] + (double)V[4 * k + 2] * pos[3 * j + 2] + (double)V[4 * k + 3];
    surfel_normal(quat + 4 * j, V, pcd, normal + 3 * j);
    surfel_colour(pos + 3 * j, sh + 48 * j, cfg->sh_degree, campos, rgb + 3 * j, clamp + j);
  }
}

// pin access (tests/test_oracle_pins.py): the fp32 decision values of R-clamp beside the fp64 colour values before the clamp
void orc_colour_probe(const float* p, const float* sh, int degree, const OrcCamera* cam, float* acc32, double* acc64, uint8_t* clamp) {
  double campos[3], rgb[3];
  cam_position(cam->view, campos);
  colour_f32(p, sh, degree, campos, acc32);
  surfel_colour(p, sh, degree, campos, rgb, clamp, acc64);
}

// ------------------------------------------------------------------------------------------------
// O2 + O3: keys, stable sort by (tile, depth bits, surfel id), per-tile ranges.
// PAPER.md:39 ("tile-based rasterization"), :119 ("rendered in front-to-back order").
// Call with keys == nullptr to obtain K only.  ranges[t] = [lower_bound(t), lower_bound(t+1)).
// ------------------------------------------------------------------------------------------------
int64_t orc_bin_sort(int n, const uint8_t* visible, const uint32_t* depth_bits, const int32_t* rect, int tile, int tiles_x,
                     int tiles_y, uint64_t* keys, uint32_t* ids, uint32_t* ranges) {
  int64_t K = 0;
  for (int j = 0; j < n; ++j) {
    if (!visible[j]) continue;
    const int tx0 = rect[4 * j] / tile, tx1 = rect[4 * j + 2] / tile + 1, ty0 = rect[4 * j + 1] / tile, ty1 = rect[4 * j + 3] / tile + 1;
    K += (int64_t)(tx1 - tx0) * (ty1 - ty0);
  }
  if (!keys) return K;
  struct KV { uint64_t key; uint32_t id; };
  std::vector<KV> kv;
  kv.reserve((size_t)K);
  for (int j = 0; j < n; ++j) {
    if (!visible[j]) continue;
    const int tx0 = rect[4 * j] / tile, tx1 = rect[4 * j + 2] / tile + 1, ty0 = rect[4 * j + 1] / tile, ty1 = rect[4 * j + 3] / tile + 1;
    for (int ty = ty0; ty < ty1; ++ty)
      for (int tx = tx0; tx < tx1; ++tx)
        kv.push_back({((uint64_t)(uint32_t)(ty * tiles_x + tx) << 32) | depth_bits[j], (uint32_t)j});
  }
  // emission is in ascending id, so a stable sort on the key alone breaks ties by surfel id
  std::stable_sort(kv.begin(), kv.end(), [](const KV& a, const KV& b) { return a.key < b.key; });
  for (int64_t i = 0; i < K; ++i) { keys[i] = kv[(size_t)i].key; ids[i] = kv[(size_t)i].id; }
  const int nt = tiles_x * tiles_y;
  int64_t i = 0;
  for (int t = 0; t < nt; ++t) {
    while (i < K && (uint32_t)(keys[i] >> 32) < (uint32_t)t) ++i;
    ranges[2 * t] = (uint32_t)i;
    int64_t e = i;
    while (e < K && (uint32_t)(keys[e] >> 32) == (uint32_t)t) ++e;
    ranges[2 * t + 1] = (uint32_t)e;
    i = e;
  }
  return K;
}

// ------------------------------------------------------------------------------------------------
// O4 + O5 + O6 + O8: forward.  PAPER.md:119: "all assigned Gaussians are rendered in front-to-back
// order, accumulating their colors and opacities to p.  Rendering is terminated once either p reaches a
// threshold opacity close to 1 or all assigned Gaussians have been exhausted"; "we save
// which Gaussians are used during the color accumulation step"; Eq. 1 for L_b.
// Pixels inside the window [wx0,wx1) x [wy0,wy1) are computed, the rest is left untouched.
// vis_count / contrib_sum ACCUMULATE (O8).  Returns L_b summed over the window (divided by W*H).
// fragile (bit 0 = a decision within its margin, bit 1 = ill-conditioned, S22) / fragile_touch / cond_rho may be null.
// cond_rho[N] (max-accumulated): largest fp32 error estimate of rho over the blended pairs of each surfel.
// ------------------------------------------------------------------------------------------------
double orc_render_fwd(int n, const OrcCamera* cam, const OrcConfig* cfg, const OrcMargins* mg, const float* M, const float* c2d,
                      const float* rho_cut, const float* opacity, const double* normal, const double* rgb, const uint32_t* ids,
                      const uint32_t* ranges, const uint8_t* mask, int wx0, int wy0, int wx1, int wy1, double* color,
                      double* alpha, double* depth, double* nrm, uint32_t* n_contrib, uint32_t* vis_count, double* contrib_sum,
                      uint8_t* fragile, uint32_t* fragile_touch, double* cond_rho,
                      double* origin, double* m1, double* m2 /*nullable together: depth moments about the first blended pair's depth (reading R-moments)*/) {
  (void)n;
  const int W = cam->width, H = cam->height, T = cfg->tile;
  const int tiles_x = (W + T - 1) / T, tiles_y = (H + T - 1) / T;
  const size_t HW = (size_t)W * H;
  double Lb = 0.0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : Lb)
  for (int t = 0; t < tiles_x * tiles_y; ++t) {
    const int tx = t % tiles_x, ty = t / tiles_x;
    const uint32_t start = ranges[2 * t], end = ranges[2 * t + 1];
    for (int y = std::max(ty * T, wy0); y < std::min({(ty + 1) * T, H, wy1}); ++y)
      for (int x = std::max(tx * T, wx0); x < std::min({(tx + 1) * T, W, wx1}); ++x) {
        double Tr = 1.0, C[3] = {0, 0, 0}, D = 0, M1 = 0, M2 = 0, c0 = 0, N[3] = {0, 0, 0};
        uint32_t last = 0;
        bool frag = false;
        double cerr = 0.0;
        for (uint32_t pos = start; pos < end; ++pos) {
          const uint32_t j = ids[pos];
          const PairEval e = eval_pair((double)x, (double)y, M + 9 * j, c2d + 2 * j, rho_cut[j], opacity[j], *cfg, mg);
          frag |= e.fragile;
          if (!e.valid) continue;
          const double Tn = Tr * (1.0 - e.alpha);
          if (mg && std::fabs(Tn - (double)cfg->t_min) <= mg->tmin_rel * (double)cfg->t_min) frag = true;
          if (Tn < (double)cfg->t_min) break;  // S11: stop before blending this pair
          const double w = e.alpha * Tr;
          cerr += Tr * e.err_est;
          if (cond_rho && e.drho_est > cond_rho[j]) {  // per-surfel conditioning: worst fp32 rho error among its blended pairs
#pragma omp critical(condrho)
            if (e.drho_est > cond_rho[j]) cond_rho[j] = e.drho_est;
          }
          for (int c = 0; c < 3; ++c) { C[c] += w * rgb[3 * j + c]; N[c] += w * normal[3 * j + c]; }
          D += w * e.z;
          if (last == 0) c0 = e.z;  // origin of the depth moments: depth of the first blended pair
          M1 += w * (e.z - c0);
          M2 += w * (e.z - c0) * (e.z - c0);
          if (vis_count) {
#pragma omp atomic
            vis_count[j] += 1;
          }
          if (contrib_sum) {
#pragma omp atomic
            contrib_sum[j] += w;
          }
          Tr = Tn;
          last = pos - start + 1;
        }
        const size_t p = (size_t)y * W + x;
        for (int c = 0; c < 3; ++c) { color[c * HW + p] = C[c] + Tr * (double)cfg->bg[c]; nrm[c * HW + p] = N[c]; }
        alpha[p] = 1.0 - Tr;
        depth[p] = D;
        if (origin) { origin[p] = c0; m1[p] = M1; m2[p] = M2; }
        n_contrib[p] = last;
        const bool illc = mg && cerr > mg->cond_abs;
        if (fragile) fragile[p] = (uint8_t)((frag ? 1 : 0) | (illc ? 2 : 0));  // bit 0: decision margin, bit 1: ill-conditioned
        if ((frag || illc) && fragile_touch)
          for (uint32_t pos = start; pos < end; ++pos) {
#pragma omp atomic
            fragile_touch[ids[pos]] += 1;
          }
        const double m = mask ? (mask[p] ? 1.0 : 0.0) : 1.0;  // no mask: every pixel is object (M = 1), L_b = 0
        Lb += (1.0 - Tr) * (1.0 - m);
      }
  }
  return Lb / (double)HW;
}

// ------------------------------------------------------------------------------------------------
// O7 backward.  PAPER.md:67: "Through backpropagation, the position, shape, and appearance of all
// involved Gaussians are updated"; occluded Gaussians "cannot receive gradients".
// Upstream gradients gC[3HW], gA[HW], gD[HW], gN[3HW] (any may be null = 0); with mask != null and
// gamma_bg != 0 the background-loss gradient gamma (1-M)/(H W) is added to gA (Eq. 1 / Eq. 3).
// Outputs are OVERWRITTEN.  d_opacity_abs (nullable) = sum over pairs of |term of d_opacity| (summation conditioning).
// d_center2d = M22 * (dL/dM02, dL/dM12) (reading R-c2d).
// ------------------------------------------------------------------------------------------------
void orc_render_bwd(int n, const float* pos, const float* scale, const float* quat, const float* opacity, const float* sh,
                    const OrcCamera* cam, const OrcConfig* cfg, const uint8_t* visible, const float* M, const float* c2d,
                    const float* rho_cut, const double* normal, const double* rgb, const uint8_t* clamp, const uint32_t* ids,
                    const uint32_t* ranges, const uint8_t* mask, const double* gC, const double* gA, const double* gD,
                    const double* gN, int wx0, int wy0, int wx1, int wy1, double* d_pos, double* d_scale, double* d_quat,
                    double* d_opacity, double* d_sh, double* d_center2d, double* d_opacity_abs,
                    const double* gM1, const double* gM2 /*nullable: upstream of the depth moments m1, m2 (origin held fixed)*/,
                    double* abs_pos, double* abs_scale, double* abs_quat, double* abs_sh, double* abs_center2d
                    /*nullable together: for every gradient entry the sum of the ABSOLUTE values of the terms it is the sum of
                      (per-pair terms, then the same linear chain with absolute coefficients) -- the conditioning of the sum: an fp32
                      evaluation cannot be closer than ~eps32 x this, whatever the size of the entry itself*/) {
  const int W = cam->width, H = cam->height, T = cfg->tile;
  const int tiles_x = (W + T - 1) / T, tiles_y = (H + T - 1) / T;
  const size_t HW = (size_t)W * H;
  // per-surfel intermediate gradients: gM[9], g_c2d[2], g_o, g_rgb[3], g_n[3]
  std::vector<double> goabs((size_t)n, 0.0);
  std::vector<double> gM((size_t)n * 9, 0.0), gc2((size_t)n * 2, 0.0), go((size_t)n, 0.0), grgb((size_t)n * 3, 0.0), gn((size_t)n * 3, 0.0);
  const bool want_abs = abs_pos != nullptr;
  std::vector<double> gMa(want_abs ? (size_t)n * 9 : 0, 0.0), gc2a(want_abs ? (size_t)n * 2 : 0, 0.0), grgba(want_abs ? (size_t)n * 3 : 0, 0.0),
      gna(want_abs ? (size_t)n * 3 : 0, 0.0);

#pragma omp parallel
  {
    struct Rec { uint32_t j; PairEval e; double Tr; };
    std::vector<Rec> seq;
#pragma omp for schedule(dynamic, 1)
    for (int t = 0; t < tiles_x * tiles_y; ++t) {
      const int tx = t % tiles_x, ty = t / tiles_x;
      const uint32_t start = ranges[2 * t], end = ranges[2 * t + 1];
      for (int y = std::max(ty * T, wy0); y < std::min({(ty + 1) * T, H, wy1}); ++y)
        for (int x = std::max(tx * T, wx0); x < std::min({(tx + 1) * T, W, wx1}); ++x) {
          const size_t p = (size_t)y * W + x;
          double gc[3] = {0, 0, 0}, gnn[3] = {0, 0, 0}, ga = 0, gd = 0;
          if (gC) for (int c = 0; c < 3; ++c) gc[c] = gC[c * HW + p];
          if (gN) for (int c = 0; c < 3; ++c) gnn[c] = gN[c * HW + p];
          if (gA) ga = gA[p];
          if (gD) gd = gD[p];
          const double gm1 = gM1 ? gM1[p] : 0.0, gm2 = gM2 ? gM2[p] : 0.0;
          if (mask && cfg->gamma_bg != 0.0f) ga += (double)cfg->gamma_bg * (mask[p] ? 0.0 : 1.0) / (double)HW;
          // forward replay
          seq.clear();
          double Tr = 1.0;
          for (uint32_t pos_i = start; pos_i < end; ++pos_i) {
            const uint32_t j = ids[pos_i];
            const PairEval e = eval_pair((double)x, (double)y, M + 9 * j, c2d + 2 * j, rho_cut[j], opacity[j], *cfg, nullptr);
            if (!e.valid) continue;
            const double Tn = Tr * (1.0 - e.alpha);
            if (Tn < (double)cfg->t_min) break;
            seq.push_back({j, e, Tr});
            Tr = Tn;
          }
          const double Tfin = Tr;
          double SC[3] = {Tfin * cfg->bg[0], Tfin * cfg->bg[1], Tfin * cfg->bg[2]}, SD = 0, SM1 = 0, SM2 = 0, SN[3] = {0, 0, 0};
          const double c0 = seq.empty() ? 0.0 : seq[0].e.z;  // origin of the depth moments (a constant: the terms built on it do not depend on it)
          for (size_t i = seq.size(); i-- > 0;) {
            const uint32_t j = seq[i].j;
            const PairEval& e = seq[i].e;
            const double Ti = seq[i].Tr, w = e.alpha * Ti, inv1ma = 1.0 / (1.0 - e.alpha);
            const double dz = e.z - c0;
            double galpha = ga * Tfin * inv1ma + gd * (e.z * Ti - SD * inv1ma) + gm1 * (dz * Ti - SM1 * inv1ma) + gm2 * (dz * dz * Ti - SM2 * inv1ma);
            for (int c = 0; c < 3; ++c) {
              galpha += gc[c] * (rgb[3 * j + c] * Ti - SC[c] * inv1ma);
              galpha += gnn[c] * (normal[3 * j + c] * Ti - SN[c] * inv1ma);
            }
            for (int c = 0; c < 3; ++c) { SC[c] += w * rgb[3 * j + c]; SN[c] += w * normal[3 * j + c]; }
            SD += w * e.z;
            SM1 += w * dz;
            SM2 += w * dz * dz;
            double a_rgb[3], a_n[3];
            for (int c = 0; c < 3; ++c) { a_rgb[c] = w * gc[c]; a_n[c] = w * gnn[c]; }
            const double gz = w * gd + w * gm1 + 2.0 * dz * w * gm2;  // z enters D = sum w z, m1 = sum w (z-c), m2 = sum w (z-c)^2
            double a_o = 0, grho = 0;
            if (!e.capped) {  // S12: zero gradient through the cap
              a_o = e.G * galpha;
              grho = -0.5 * e.G * ((double)opacity[j] * galpha);
            }
            double aM[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, ac[2] = {0, 0};
            const double Mj[9] = {M[9 * j], M[9 * j + 1], M[9 * j + 2], M[9 * j + 3], M[9 * j + 4], M[9 * j + 5], M[9 * j + 6], M[9 * j + 7], M[9 * j + 8]};
            if (e.surf) {
              const double gu = 2 * e.u * grho + Mj[6] * gz, gv = 2 * e.v * grho + Mj[7] * gz;
              aM[6] += e.u * gz; aM[7] += e.v * gz; aM[8] += gz;
              const double gq[3] = {gu / e.qz, gv / e.qz, -(gu * e.u + gv * e.v) / e.qz};
              double gk[3], gl[3];
              cross3(e.l, gq, gk);  // q = k x l  =>  gk = l x gq, gl = gq x k
              cross3(gq, e.k, gl);
              for (int i2 = 0; i2 < 3; ++i2) {
                aM[i2] -= gk[i2];
                aM[3 + i2] -= gl[i2];
                aM[6 + i2] += (double)x * gk[i2] + (double)y * gl[i2];
              }
            } else {
              ac[0] = -2.0 * e.dx / (double)cfg->filter_sigma2 * grho;
              ac[1] = -2.0 * e.dy / (double)cfg->filter_sigma2 * grho;
              aM[8] += gz;  // z = z_j = M22
            }
            for (int i2 = 0; i2 < 9; ++i2) if (aM[i2] != 0.0) {
#pragma omp atomic
              gM[9 * (size_t)j + i2] += aM[i2];
              if (want_abs) {
#pragma omp atomic
                gMa[9 * (size_t)j + i2] += std::fabs(aM[i2]);
              }
            }
            for (int i2 = 0; i2 < 2; ++i2) if (ac[i2] != 0.0) {
#pragma omp atomic
              gc2[2 * (size_t)j + i2] += ac[i2];
              if (want_abs) {
#pragma omp atomic
                gc2a[2 * (size_t)j + i2] += std::fabs(ac[i2]);
              }
            }
            if (a_o != 0.0) {
#pragma omp atomic
              go[j] += a_o;
#pragma omp atomic
              goabs[j] += std::fabs(a_o);
            }
            for (int c = 0; c < 3; ++c) {
              if (a_rgb[c] != 0.0) {
#pragma omp atomic
                grgb[3 * (size_t)j + c] += a_rgb[c];
                if (want_abs) {
#pragma omp atomic
                  grgba[3 * (size_t)j + c] += std::fabs(a_rgb[c]);
                }
              }
              if (a_n[c] != 0.0) {
#pragma omp atomic
                gn[3 * (size_t)j + c] += a_n[c];
                if (want_abs) {
#pragma omp atomic
                  gna[3 * (size_t)j + c] += std::fabs(a_n[c]);
                }
              }
            }
          }
        }
    }
  }

  // per-surfel chain: record -> parameters
  double campos[3];
  cam_position(cam->view, campos);
  const float* V = cam->view;
  const double ox = (double)(cam->cx - 0.5f), oy = (double)(cam->cy - 0.5f), fx = cam->fx, fy = cam->fy;
  const int nb = (cfg->sh_degree + 1) * (cfg->sh_degree + 1);
#pragma omp parallel for schedule(static)
  for (int j = 0; j < n; ++j) {
    for (int k = 0; k < 3; ++k) d_pos[3 * j + k] = 0;
    for (int k = 0; k < 2; ++k) { d_scale[2 * j + k] = 0; d_center2d[2 * j + k] = 0; }
    for (int k = 0; k < 4; ++k) d_quat[4 * j + k] = 0;
    d_opacity[j] = 0;
    if (d_opacity_abs) d_opacity_abs[j] = goabs[j];  // sum of |terms|: conditioning of the d_opacity summation
    for (int k = 0; k < 48; ++k) d_sh[48 * (size_t)j + k] = 0;
    if (want_abs) {
      for (int k = 0; k < 3; ++k) abs_pos[3 * j + k] = 0;
      for (int k = 0; k < 2; ++k) { abs_scale[2 * j + k] = 0; abs_center2d[2 * j + k] = 0; }
      for (int k = 0; k < 4; ++k) abs_quat[4 * j + k] = 0;
      for (int k = 0; k < 48; ++k) abs_sh[48 * (size_t)j + k] = 0;
    }
    if (!visible[j]) continue;
    double g[9];
    for (int k = 0; k < 9; ++k) g[k] = gM[9 * (size_t)j + k];
    const double M22 = M[9 * j + 8];
    // c2d = (M02, M12) / M22
    g[2] += gc2[2 * j] / M22;
    g[5] += gc2[2 * j + 1] / M22;
    g[8] -= (gc2[2 * j] * (double)c2d[2 * j] + gc2[2 * j + 1] * (double)c2d[2 * j + 1]) / M22;
    d_center2d[2 * j] = M22 * g[2];
    d_center2d[2 * j + 1] = M22 * g[5];
    // M = K' [c0|c1|c2]
    double gcol[3][3];
    for (int i = 0; i < 3; ++i) {
      gcol[i][0] = fx * g[i];
      gcol[i][1] = fy * g[3 + i];
      gcol[i][2] = ox * g[i] + oy * g[3 + i] + g[6 + i];
    }
    const double qd[4] = {quat[4 * j], quat[4 * j + 1], quat[4 * j + 2], quat[4 * j + 3]};
    const Rot r = rot_from_quat(qd);
    double vu[3], vv[3];
    mat3_vec(V, r.tu, vu);
    mat3_vec(V, r.tv, vv);
    d_scale[2 * j] = dot3(gcol[0], vu);
    d_scale[2 * j + 1] = dot3(gcol[1], vv);
    double gtu[3], gtv[3], gtw[3], tmp[3];
    mat3T_vec(V, gcol[0], tmp);
    for (int k = 0; k < 3; ++k) gtu[k] = (double)scale[2 * j] * tmp[k];
    mat3T_vec(V, gcol[1], tmp);
    for (int k = 0; k < 3; ++k) gtv[k] = (double)scale[2 * j + 1] * tmp[k];
    double gp[3];
    mat3T_vec(V, gcol[2], gp);
    // normal: n = sgn * R_wc t_w
    double pcd[3];
    for (int k = 0; k < 3; ++k)
      pcd[k] = (double)V[4 * k] * pos[3 * j] + (double)V[4 * k + 1] * pos[3 * j + 1] + (double)V[4 * k + 2] * pos[3 * j + 2] + (double)V[4 * k + 3];
    double ntmp[3];
    const double sgn = surfel_normal(quat + 4 * j, V, pcd, ntmp);
    const double gnj[3] = {gn[3 * (size_t)j], gn[3 * (size_t)j + 1], gn[3 * (size_t)j + 2]};
    mat3T_vec(V, gnj, gtw);
    for (int k = 0; k < 3; ++k) gtw[k] *= sgn;
    // R(q) polynomial
    const double w = qd[0], x = qd[1], y = qd[2], z = qd[3];
    d_quat[4 * j + 0] = 2 * (z * gtu[1] - y * gtu[2] - z * gtv[0] + x * gtv[2] + y * gtw[0] - x * gtw[1]);
    d_quat[4 * j + 1] = 2 * (y * gtu[1] + z * gtu[2] + y * gtv[0] - 2 * x * gtv[1] + w * gtv[2] + z * gtw[0] - w * gtw[1] - 2 * x * gtw[2]);
    d_quat[4 * j + 2] = 2 * (-2 * y * gtu[0] + x * gtu[1] - w * gtu[2] + x * gtv[0] + z * gtv[2] + w * gtw[0] + z * gtw[1] - 2 * y * gtw[2]);
    d_quat[4 * j + 3] = 2 * (-2 * z * gtu[0] + w * gtu[1] + x * gtu[2] - w * gtv[0] - 2 * z * gtv[1] + y * gtv[2] + x * gtw[0] + y * gtw[1]);
    d_opacity[j] = go[j];
    // colour
    double vdir[3] = {pos[3 * j] - campos[0], pos[3 * j + 1] - campos[1], pos[3 * j + 2] - campos[2]};
    const double len = std::sqrt(dot3(vdir, vdir));
    double dir[3] = {vdir[0] / len, vdir[1] / len, vdir[2] / len};
    double Y[16], dY[16][3];
    sh_basis(dir, Y, dY);
    double gdir[3] = {0, 0, 0};
    for (int c = 0; c < 3; ++c) {
      if (clamp[j] & (1u << c)) continue;  // S12: zero gradient on clamped channels
      const double gcol_c = grgb[3 * (size_t)j + c];
      for (int k = 0; k < nb; ++k) {
        d_sh[48 * (size_t)j + 3 * k + c] = Y[k] * gcol_c;
        const double s = (double)sh[48 * (size_t)j + 3 * k + c] * gcol_c;
        gdir[0] += dY[k][0] * s; gdir[1] += dY[k][1] * s; gdir[2] += dY[k][2] * s;
      }
    }
    const double dd = dot3(dir, gdir);
    for (int k = 0; k < 3; ++k) gp[k] += (gdir[k] - dir[k] * dd) / len;
    for (int k = 0; k < 3; ++k) d_pos[3 * j + k] = gp[k];
    if (want_abs) {
      // the same linear chain with the absolute values of every coefficient, applied to the sums of |terms|
      auto A = [](double v) { return std::fabs(v); };
      double ga[9];
      for (int k = 0; k < 9; ++k) ga[k] = gMa[9 * (size_t)j + k];
      const double c0a = gc2a[2 * j], c1a = gc2a[2 * j + 1];
      ga[2] += c0a / A(M22);
      ga[5] += c1a / A(M22);
      ga[8] += (c0a * A((double)c2d[2 * j]) + c1a * A((double)c2d[2 * j + 1])) / A(M22);
      abs_center2d[2 * j] = A(M22) * ga[2];
      abs_center2d[2 * j + 1] = A(M22) * ga[5];
      double gca[3][3];
      for (int i = 0; i < 3; ++i) {
        gca[i][0] = A(fx) * ga[i];
        gca[i][1] = A(fy) * ga[3 + i];
        gca[i][2] = A(ox) * ga[i] + A(oy) * ga[3 + i] + ga[6 + i];
      }
      auto VTa = [&](const double* e, double* out) {  // |R_wc^T| e
        for (int k = 0; k < 3; ++k) out[k] = A((double)V[k]) * e[0] + A((double)V[4 + k]) * e[1] + A((double)V[8 + k]) * e[2];
      };
      abs_scale[2 * j] = gca[0][0] * A(vu[0]) + gca[0][1] * A(vu[1]) + gca[0][2] * A(vu[2]);
      abs_scale[2 * j + 1] = gca[1][0] * A(vv[0]) + gca[1][1] * A(vv[1]) + gca[1][2] * A(vv[2]);
      double ua[3], va[3], wa[3], pa[3], t3[3];
      VTa(gca[0], t3);
      for (int k = 0; k < 3; ++k) ua[k] = A((double)scale[2 * j]) * t3[k];
      VTa(gca[1], t3);
      for (int k = 0; k < 3; ++k) va[k] = A((double)scale[2 * j + 1]) * t3[k];
      VTa(gca[2], pa);
      const double gnja[3] = {gna[3 * (size_t)j], gna[3 * (size_t)j + 1], gna[3 * (size_t)j + 2]};
      VTa(gnja, wa);
      const double aw = A(w), ax = A(x), ay = A(y), az = A(z);
      abs_quat[4 * j + 0] = 2 * (az * ua[1] + ay * ua[2] + az * va[0] + ax * va[2] + ay * wa[0] + ax * wa[1]);
      abs_quat[4 * j + 1] = 2 * (ay * ua[1] + az * ua[2] + ay * va[0] + 2 * ax * va[1] + aw * va[2] + az * wa[0] + aw * wa[1] + 2 * ax * wa[2]);
      abs_quat[4 * j + 2] = 2 * (2 * ay * ua[0] + ax * ua[1] + aw * ua[2] + ax * va[0] + az * va[2] + aw * wa[0] + az * wa[1] + 2 * ay * wa[2]);
      abs_quat[4 * j + 3] = 2 * (2 * az * ua[0] + aw * ua[1] + ax * ua[2] + aw * va[0] + 2 * az * va[1] + ay * va[2] + ax * wa[0] + ay * wa[1]);
      double gda[3] = {0, 0, 0};
      for (int c = 0; c < 3; ++c) {
        if (clamp[j] & (1u << c)) continue;
        const double gca_c = grgba[3 * (size_t)j + c];
        for (int k = 0; k < nb; ++k) {
          abs_sh[48 * (size_t)j + 3 * k + c] = A(Y[k]) * gca_c;
          const double sa = A((double)sh[48 * (size_t)j + 3 * k + c]) * gca_c;
          gda[0] += A(dY[k][0]) * sa; gda[1] += A(dY[k][1]) * sa; gda[2] += A(dY[k][2]) * sa;
        }
      }
      const double dda = A(dir[0]) * gda[0] + A(dir[1]) * gda[1] + A(dir[2]) * gda[2];
      for (int k = 0; k < 3; ++k) abs_pos[3 * j + k] = pa[k] + (gda[k] + A(dir[k]) * dda) / len;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O9 prune rule.  PAPER.md:119: "We propose to assign both G_j and G_k with false" (never blended, whether
// in-frustum-but-occluded or out of frustum); PAPER.md:101 (opacity threshold); S17 (tau extension).
// remap[j] = new index of survivor j in ascending id order, -1 if pruned.  Returns the survivor count.
// ------------------------------------------------------------------------------------------------
int orc_prune(int n, const uint32_t* vis_count, const float* contrib_sum, const float* opacity, float tau, float min_opacity,
              uint8_t* prune_mask, int32_t* remap) {
  int kept = 0;
  for (int j = 0; j < n; ++j) {
    const bool prune = (vis_count[j] == 0) || (contrib_sum[j] <= tau) || (opacity[j] < min_opacity);
    prune_mask[j] = prune ? 1 : 0;
    remap[j] = prune ? -1 : kept++;
  }
  return kept;
}

// ------------------------------------------------------------------------------------------------
// BF: brute force in fp64 from the raw parameters (SURVEY.md §8(c) "BF").  For every pixel of the window,
// every surfel: textbook ray-plane intersection t = (n.p_c)/(n.d), n = A x B, local coordinates by Cramer's rule, the low-pass filter (S8), the same per-pair rules (S3, S6, S11), exhaustive sort of the
// pixel's candidates by (fp32 centre-depth bits, id) (S9).  No bounding boxes, no tiles, no M.
// Parameters are fp64 so that central differences can perturb them.
// out_* are per pixel of the FULL image (planar), only window pixels are written.
// ------------------------------------------------------------------------------------------------
double orc_bf_render(int n, const double* pos, const double* scale, const double* quat, const double* opacity, const double* sh,
                     const OrcCamera* cam, const OrcConfig* cfg, const uint8_t* mask, int wx0, int wy0, int wx1, int wy1,
                     double* color, double* alpha, double* depth, double* nrm, uint32_t* n_blended, uint32_t* vis_count,
                     double* contrib_sum, double* origin, double* m1, double* m2 /*nullable together*/) {
  const int W = cam->width, H = cam->height;
  const size_t HW = (size_t)W * H;
  const float* V = cam->view;
  double campos[3];
  cam_position(V, campos);
  struct S { bool ok; double pc[3], au[3], av[3], nn[3], facing[3], A[3], B[3], pn[3], pn2, su, sv, o, rho_cut, rgb[3], c2d[2]; uint32_t key; };
  std::vector<S> ss((size_t)n);
  const double ox = (double)(cam->cx - 0.5f), oy = (double)(cam->cy - 0.5f);
  const int nb = (cfg->sh_degree + 1) * (cfg->sh_degree + 1);
  for (int j = 0; j < n; ++j) {
    S& s = ss[(size_t)j];
    const double* p = pos + 3 * j;
    for (int k = 0; k < 3; ++k) s.pc[k] = (double)V[4 * k] * p[0] + (double)V[4 * k + 1] * p[1] + (double)V[4 * k + 2] * p[2] + (double)V[4 * k + 3];
    // ordering key: the fp32 centre depth of Appendix A step 2 (S9), so ties resolve like the tiled path
    const float pf[3] = {(float)p[0], (float)p[1], (float)p[2]};
    float pcf[3];
    view_point(V, pf, pcf);
    s.key = float_bits(pcf[2]);
    const Rot r = rot_from_quat(quat + 4 * j);
    mat3_vec(V, r.tu, s.au);
    mat3_vec(V, r.tv, s.av);
    mat3_vec(V, r.tw, s.nn);
    const double sg = dot3(s.nn, s.pc) > 0.0 ? -1.0 : 1.0;
    for (int k = 0; k < 3; ++k) s.facing[k] = sg * s.nn[k];
    s.su = scale[2 * j]; s.sv = scale[2 * j + 1]; s.o = opacity[j];
    for (int k = 0; k < 3; ++k) { s.A[k] = s.su * s.au[k]; s.B[k] = s.sv * s.av[k]; }
    cross3(s.A, s.B, s.pn);
    s.pn2 = dot3(s.pn, s.pn);
    s.ok = s.pc[2] > (double)cfg->near_z && s.o >= (double)cfg->alpha_min;
    if (!s.ok) continue;
    s.rho_cut = std::fmin((double)cfg->rho_max, 2.0 * std::log(s.o / (double)cfg->alpha_min));
    // S4: the rho_cut ellipse must stay in front of the eye plane: depth along the ellipse is
    // pc.z + su au.z u + sv av.z v with u^2+v^2 = rho_cut; its minimum must be > 0
    const double zr = std::sqrt(s.rho_cut * ((s.su * s.au[2]) * (s.su * s.au[2]) + (s.sv * s.av[2]) * (s.sv * s.av[2])));
    if (!(s.pc[2] - zr > 0.0)) { s.ok = false; continue; }
    s.c2d[0] = cam->fx * s.pc[0] / s.pc[2] + ox;
    s.c2d[1] = cam->fy * s.pc[1] / s.pc[2] + oy;
    double v[3] = {p[0] - campos[0], p[1] - campos[1], p[2] - campos[2]};
    const double len = std::sqrt(dot3(v, v));
    const double d[3] = {v[0] / len, v[1] / len, v[2] / len};
    double Y[16];
    sh_basis(d, Y, nullptr);
    for (int c = 0; c < 3; ++c) {
      double acc = 0.5;
      for (int k = 0; k < nb; ++k) acc += Y[k] * sh[48 * (size_t)j + 3 * k + c];
      s.rgb[c] = acc < 0.0 ? 0.0 : acc;
    }
  }
  double Lb = 0.0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : Lb)
  for (int y = wy0; y < wy1; ++y) {
    struct Cand { uint32_t key; int j; double alpha, z; };
    std::vector<Cand> cands;
    for (int x = wx0; x < wx1; ++x) {
      cands.clear();
      const double d[3] = {((double)x - ox) / (double)cam->fx, ((double)y - oy) / (double)cam->fy, 1.0};
      for (int j = 0; j < n; ++j) {
        const S& s = ss[(size_t)j];
        if (!s.ok) continue;
        // ray t*d meets the plane p_c + u*A + v*B (A = s_u a_u, B = s_v a_v): t = (p_c.n)/(d.n), n = A x B, then (u, v)
        // by Cramer's rule in the plane (also valid when a_u, a_v are not orthonormal, i.e. for a non-unit quaternion, S19)
        const double nd = dot3(s.pn, d);
        if (nd == 0.0) continue;
        const double t = dot3(s.pn, s.pc) / nd;
        const double hit[3] = {t * d[0] - s.pc[0], t * d[1] - s.pc[1], t * d[2] - s.pc[2]};
        double hxB[3], Axh[3];
        cross3(hit, s.B, hxB);
        cross3(s.A, hit, Axh);
        const double u = dot3(hxB, s.pn) / s.pn2, v = dot3(Axh, s.pn) / s.pn2;
        const double rho3 = u * u + v * v;
        const double ex = (double)x - s.c2d[0], ey = (double)y - s.c2d[1];
        const double rho2 = (ex * ex + ey * ey) / (double)cfg->filter_sigma2;
        const bool surf = rho3 <= rho2;
        const double rho = surf ? rho3 : rho2;
        const double z = surf ? t : s.pc[2];
        if (z < (double)cfg->near_z) continue;
        if (rho > s.rho_cut) continue;
        const double a = std::fmin((double)cfg->alpha_max, s.o * std::exp(-0.5 * rho));
        cands.push_back({s.key, j, a, z});
      }
      std::sort(cands.begin(), cands.end(), [](const Cand& a, const Cand& b) { return a.key != b.key ? a.key < b.key : a.j < b.j; });
      double Tr = 1.0, C[3] = {0, 0, 0}, D = 0, M1 = 0, M2 = 0, c0 = 0, N[3] = {0, 0, 0};
      uint32_t cnt = 0;
      for (const Cand& c : cands) {
        const double Tn = Tr * (1.0 - c.alpha);
        if (Tn < (double)cfg->t_min) break;
        const double w = c.alpha * Tr;
        const S& s = ss[(size_t)c.j];
        for (int k = 0; k < 3; ++k) { C[k] += w * s.rgb[k]; N[k] += w * s.facing[k]; }
        D += w * c.z;
        if (cnt == 0) c0 = c.z;
        M1 += w * (c.z - c0);
        M2 += w * (c.z - c0) * (c.z - c0);
        if (vis_count) {
#pragma omp atomic
          vis_count[c.j] += 1;
        }
        if (contrib_sum) {
#pragma omp atomic
          contrib_sum[c.j] += w;
        }
        Tr = Tn;
        ++cnt;
      }
      const size_t p = (size_t)y * W + x;
      for (int k = 0; k < 3; ++k) { color[k * HW + p] = C[k] + Tr * (double)cfg->bg[k]; nrm[k * HW + p] = N[k]; }
      alpha[p] = 1.0 - Tr;
      depth[p] = D;
      if (origin) { origin[p] = c0; m1[p] = M1; m2[p] = M2; }
      if (n_blended) n_blended[p] = cnt;
      const double m = mask ? (mask[p] ? 1.0 : 0.0) : 1.0;  // no mask: every pixel is object (M = 1), L_b = 0
      Lb += (1.0 - Tr) * (1.0 - m);
    }
  }
  return Lb / (double)HW;
}

// ================================================================================================
// 3D-Gaussian variant of the visibility statistics (Appendix B: "We demonstrate the versatility of
// our pruning strategy by implementing it in 3DGS").  Only the primitive changes: O1 (projection)
// and O4 (per-pair evaluation); keys, order, compositing, termination, statistics and the prune rule are the ones above.
// The paper gives no formulas for 3DGS (PAPER.md:63 defers to Kerbl et al. 2023); readings (R-3D):
//   Gaussian j: mean p, covariance Sigma = R(q) diag(s^2) R(q)^T, opacity o, SH colour as for surfels.
//   EWA projection: t = W p + t_wc, J = d(fx tx/tz, fy ty/tz)/dt, Sigma' = J W Sigma W^T J^T + 0.3 I (the published
//   screen-space dilation), centre c = (fx tx/tz + cx - 1/2, fy ty/tz + cy - 1/2); rho(x) = (x - c)^T Sigma'^-1 (x - c);
//   the pair contributes iff rho <= rho_cut = min(9, 2 ln(o/alpha_min)) (S6, same pixel-exact cut as for surfels, which
//   keeps the image independent of the tiling), alpha = min(alpha_max, o exp(-rho/2)); depth of a pair = centre depth t_z.
//   Box: exact AABB of the rho_cut ellipse, half extents sqrt(rho_cut Sigma'_xx), sqrt(rho_cut Sigma'_yy), padded like R-bbox.
// Integer-deciding sequence (fp32, each operation rounded once, fma written explicitly; the GPU kernel repeats it):
//   R columns as in Appendix A step 1 (plus t_w = (2(xz+wy), 2(yz-wx), 1-2(xx+yy))); t = view_point(p); cull !(t_z > near),
//   o < alpha_min; m_k = view_dir(R column k), b_k = s_k m_k (k = 0..2); S_ij = fma(b_0i, b_0j, fma(b_1i, b_1j, b_2i b_2j));
//   itz = 1/t_z; j00 = fx itz; j02 = -((j00 t_x) itz); j11 = fy itz; j12 = -((j11 t_y) itz);
//   T0 = (fma(j00,S00, j02 S02), fma(j00,S01, j02 S12), fma(j00,S02, j02 S22)), T1 likewise with (j11, j12) and rows 1, 2;
//   cxx = fma(T0x,j00, T0z j02) + 0.3; cxy = fma(T0y,j11, T0z j12); cyy = fma(T1y,j11, T1z j12) + 0.3;
//   det = fma(cxx,cyy, -(cxy cxy)); cull !(det > 0); conic = (cyy/det, -cxy/det, cxx/det);
//   c = (fma(j00,t_x, cx-1/2), fma(j11,t_y, cy-1/2)); rho_cut as Appendix A step 5;
//   h_x = fma(sqrt(rho_cut cxx), 1+2^-16, 2^-7), h_y likewise; bounds ceil(c - h) .. floor(c + h), clamps as step 8.
// ================================================================================================
namespace {

struct Pre3 {
  bool visible;
  float conic[3], cov[3], c2d[2], rho_cut, depth;
  int rect[4];
};

Pre3 preprocess3d_one(const float* p, const float* s, const float* q, float o, const OrcCamera& cam, const OrcConfig& cfg) {
  Pre3 r;
  std::memset(&r, 0, sizeof(r));
  const float* V = cam.view;
  const float w = q[0], x = q[1], y = q[2], z = q[3];
  const float xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y, wz = w * z;
  const float col[3][3] = {{1.0f - 2.0f * (yy + zz), 2.0f * (xy + wz), 2.0f * (xz - wy)},
                           {2.0f * (xy - wz), 1.0f - 2.0f * (xx + zz), 2.0f * (yz + wx)},
                           {2.0f * (xz + wy), 2.0f * (yz - wx), 1.0f - 2.0f * (xx + yy)}};
  float t[3];
  view_point(V, p, t);
  r.depth = t[2];
  if (!(t[2] > cfg.near_z)) return r;
  if (o < cfg.alpha_min) return r;
  float b[3][3];  // b[k] = s_k * W R e_k
  for (int k = 0; k < 3; ++k) {
    float m[3];
    view_dir(V, col[k], m);
    for (int i = 0; i < 3; ++i) b[k][i] = s[k] * m[i];
  }
  auto S = [&](int i, int j) { return std::fmaf(b[0][i], b[0][j], std::fmaf(b[1][i], b[1][j], b[2][i] * b[2][j])); };
  const float S00 = S(0, 0), S01 = S(0, 1), S02 = S(0, 2), S11 = S(1, 1), S12 = S(1, 2), S22 = S(2, 2);
  const float itz = 1.0f / t[2];
  const float j00 = cam.fx * itz, j02 = -((j00 * t[0]) * itz), j11 = cam.fy * itz, j12 = -((j11 * t[1]) * itz);
  const float T0x = std::fmaf(j00, S00, j02 * S02), T0y = std::fmaf(j00, S01, j02 * S12), T0z = std::fmaf(j00, S02, j02 * S22);
  const float T1y = std::fmaf(j11, S11, j12 * S12), T1z = std::fmaf(j11, S12, j12 * S22);
  const float cxx = std::fmaf(T0x, j00, T0z * j02) + 0.3f;
  const float cxy = std::fmaf(T0y, j11, T0z * j12);
  const float cyy = std::fmaf(T1y, j11, T1z * j12) + 0.3f;
  const float det = std::fmaf(cxx, cyy, -(cxy * cxy));
  if (!(det > 0.0f)) return r;
  r.cov[0] = cxx; r.cov[1] = cxy; r.cov[2] = cyy;
  r.conic[0] = cyy / det; r.conic[1] = -cxy / det; r.conic[2] = cxx / det;
  r.c2d[0] = std::fmaf(j00, t[0], cam.cx - 0.5f);
  r.c2d[1] = std::fmaf(j11, t[1], cam.cy - 0.5f);
  const double rr = 2.0 * std::log((double)o / (double)cfg.alpha_min);
  const float rc = (float)std::fmin((double)cfg.rho_max, rr);
  r.rho_cut = rc;
  const float h[2] = {std::fmaf(std::sqrt(rc * cxx), 1.0000152587890625f, 0.0078125f),
                      std::fmaf(std::sqrt(rc * cyy), 1.0000152587890625f, 0.0078125f)};
  const float lim = 1073741824.0f;
  const int WH[2] = {cam.width, cam.height};
  int lo[2], hi[2];
  for (int k = 0; k < 2; ++k) {
    float mn = std::fmax(-lim, std::fmin(lim, r.c2d[k] - h[k]));
    float mx = std::fmax(-lim, std::fmin(lim, r.c2d[k] + h[k]));
    lo[k] = (int)std::ceil(mn);
    hi[k] = (int)std::floor(mx);
    if (hi[k] < 0 || lo[k] > WH[k] - 1 || lo[k] > hi[k]) return r;
    lo[k] = std::max(lo[k], 0);
    hi[k] = std::min(hi[k], WH[k] - 1);
  }
  r.rect[0] = lo[0]; r.rect[1] = lo[1]; r.rect[2] = hi[0]; r.rect[3] = hi[1];
  r.visible = true;
  return r;
}

}  // namespace

extern "C" {

void orc3d_preprocess(int n, const float* pos, const float* scale, const float* quat, const float* opacity, const float* sh,
                      const OrcCamera* cam, const OrcConfig* cfg, uint8_t* visible, uint32_t* depth_bits, int32_t* rect,
                      uint32_t* tiles_touched, float* conic, float* c2d, float* rho_cut, double* rgb, uint8_t* clamp) {
  double campos[3];
  cam_position(cam->view, campos);
#pragma omp parallel for schedule(static)
  for (int j = 0; j < n; ++j) {
    const Pre3 r = preprocess3d_one(pos + 3 * j, scale + 3 * j, quat + 4 * j, opacity[j], *cam, *cfg);
    visible[j] = r.visible ? 1 : 0;
    depth_bits[j] = float_bits(r.depth);
    for (int k = 0; k < 3; ++k) { conic[3 * j + k] = r.conic[k]; rgb[3 * j + k] = 0; }
    c2d[2 * j] = r.c2d[0]; c2d[2 * j + 1] = r.c2d[1];
    rho_cut[j] = r.rho_cut;
    for (int k = 0; k < 4; ++k) rect[4 * j + k] = r.visible ? r.rect[k] : 0;
    tiles_touched[j] = 0;
    clamp[j] = 0;
    if (!r.visible) continue;
    const int T = cfg->tile;
    tiles_touched[j] = (uint32_t)((r.rect[2] / T + 1 - r.rect[0] / T) * (r.rect[3] / T + 1 - r.rect[1] / T));
    surfel_colour(pos + 3 * j, sh + 48 * j, cfg->sh_degree, campos, rgb + 3 * j, clamp + j);
  }
}

}  // extern "C" (3D preprocess)

extern "C" {

// TILED forward for 3D Gaussians: same walk as orc_render_fwd (O5, O6, O8), per-pair evaluation of R-3D in fp64 from the
// fp32 record (conic, c2d, rho_cut).  depth accumulates the CENTRE depth of each blended Gaussian.  A pixel is fragile when
// a decision is within the margins (rho vs rho_cut, the stop test).
double orc3d_render_fwd(int n, const OrcCamera* cam, const OrcConfig* cfg, const OrcMargins* mg, const float* conic, const float* c2d,
                        const float* rho_cut, const float* opacity, const uint32_t* depth_bits, const double* rgb, const uint32_t* ids,
                        const uint32_t* ranges, const uint8_t* mask, int wx0, int wy0, int wx1, int wy1, double* color, double* alpha,
                        double* depth, uint32_t* n_contrib, uint32_t* vis_count, double* contrib_sum, uint8_t* fragile,
                        uint32_t* fragile_touch) {
  (void)n;
  const int W = cam->width, H = cam->height, T = cfg->tile;
  const int tiles_x = (W + T - 1) / T, tiles_y = (H + T - 1) / T;
  const size_t HW = (size_t)W * H;
  double Lb = 0.0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : Lb)
  for (int t = 0; t < tiles_x * tiles_y; ++t) {
    const int tx = t % tiles_x, ty = t / tiles_x;
    const uint32_t start = ranges[2 * t], end = ranges[2 * t + 1];
    for (int y = std::max(ty * T, wy0); y < std::min({(ty + 1) * T, H, wy1}); ++y)
      for (int x = std::max(tx * T, wx0); x < std::min({(tx + 1) * T, W, wx1}); ++x) {
        double Tr = 1.0, C[3] = {0, 0, 0}, D = 0;
        uint32_t last = 0;
        bool frag = false;
        for (uint32_t pos = start; pos < end; ++pos) {
          const uint32_t j = ids[pos];
          const double dx = (double)x - (double)c2d[2 * j], dy = (double)y - (double)c2d[2 * j + 1];
          const double rho = (double)conic[3 * j] * dx * dx + 2.0 * (double)conic[3 * j + 1] * dx * dy + (double)conic[3 * j + 2] * dy * dy;
          const double rc = rho_cut[j];
          if (mg && std::fabs(rho - rc) <= mg->rho_cut_abs) frag = true;
          if (rho > rc) continue;
          const double a = std::fmin((double)cfg->alpha_max, (double)opacity[j] * std::exp(-0.5 * rho));
          const double Tn = Tr * (1.0 - a);
          if (mg && std::fabs(Tn - (double)cfg->t_min) <= mg->tmin_rel * (double)cfg->t_min) frag = true;
          if (Tn < (double)cfg->t_min) break;
          const double w = a * Tr;
          float zf; std::memcpy(&zf, &depth_bits[j], 4);
          for (int c = 0; c < 3; ++c) C[c] += w * rgb[3 * j + c];
          D += w * (double)zf;
          if (vis_count) {
#pragma omp atomic
            vis_count[j] += 1;
          }
          if (contrib_sum) {
#pragma omp atomic
            contrib_sum[j] += w;
          }
          Tr = Tn;
          last = pos - start + 1;
        }
        const size_t p = (size_t)y * W + x;
        for (int c = 0; c < 3; ++c) color[c * HW + p] = C[c] + Tr * (double)cfg->bg[c];
        alpha[p] = 1.0 - Tr;
        depth[p] = D;
        n_contrib[p] = last;
        if (fragile) fragile[p] = frag ? 1 : 0;
        if (frag && fragile_touch)
          for (uint32_t pos = start; pos < end; ++pos) {
#pragma omp atomic
            fragile_touch[ids[pos]] += 1;
          }
        const double m = mask ? (mask[p] ? 1.0 : 0.0) : 1.0;  // no mask: every pixel is object (M = 1), L_b = 0
        Lb += (1.0 - Tr) * (1.0 - m);
      }
  }
  return Lb / (double)HW;
}

// Brute force for 3D Gaussians: fp64 from the raw parameters, every (pixel, Gaussian) pair, no boxes, no tiles, exhaustive
// per-pixel sort by (fp32 centre-depth bits, id).  Knows nothing of the fp32 sequence above except the ordering key.
double orc3d_bf_render(int n, const double* pos, const double* scale, const double* quat, const double* opacity, const double* sh,
                       const OrcCamera* cam, const OrcConfig* cfg, const uint8_t* mask, int wx0, int wy0, int wx1, int wy1,
                       double* color, double* alpha, double* depth, uint32_t* n_blended, uint32_t* vis_count, double* contrib_sum) {
  const int W = cam->width, H = cam->height;
  const size_t HW = (size_t)W * H;
  const float* V = cam->view;
  double campos[3];
  cam_position(V, campos);
  struct G { bool ok; double c[2], q[3], rho_cut, o, z, rgb[3]; uint32_t key; };
  std::vector<G> gs((size_t)n);
  const double fx = cam->fx, fy = cam->fy, ox = (double)(cam->cx - 0.5f), oy = (double)(cam->cy - 0.5f);
  for (int j = 0; j < n; ++j) {
    G& g = gs[(size_t)j];
    const double* p = pos + 3 * j;
    double t[3];
    for (int k = 0; k < 3; ++k) t[k] = (double)V[4 * k] * p[0] + (double)V[4 * k + 1] * p[1] + (double)V[4 * k + 2] * p[2] + (double)V[4 * k + 3];
    const float pf[3] = {(float)p[0], (float)p[1], (float)p[2]};
    float tf[3];
    view_point(V, pf, tf);
    g.key = float_bits(tf[2]);
    g.z = (double)tf[2];  // the depth map accumulates the fp32 centre depth (the key), as the tiled path does
    g.o = opacity[j];
    g.ok = t[2] > (double)cfg->near_z && g.o >= (double)cfg->alpha_min;
    if (!g.ok) continue;
    const Rot r = rot_from_quat(quat + 4 * j);
    const double* cols[3] = {r.tu, r.tv, r.tw};
    double B[3][3];  // B[k] = s_k W R e_k
    for (int k = 0; k < 3; ++k) {
      double m[3];
      mat3_vec(V, cols[k], m);
      for (int i = 0; i < 3; ++i) B[k][i] = scale[3 * j + k] * m[i];
    }
    double S[3][3];
    for (int a = 0; a < 3; ++a)
      for (int b2 = 0; b2 < 3; ++b2) S[a][b2] = B[0][a] * B[0][b2] + B[1][a] * B[1][b2] + B[2][a] * B[2][b2];
    const double J[2][3] = {{fx / t[2], 0.0, -fx * t[0] / (t[2] * t[2])}, {0.0, fy / t[2], -fy * t[1] / (t[2] * t[2])}};
    double cov[2][2];
    for (int a = 0; a < 2; ++a)
      for (int b2 = 0; b2 < 2; ++b2) {
        double acc = 0;
        for (int k = 0; k < 3; ++k)
          for (int l = 0; l < 3; ++l) acc += J[a][k] * S[k][l] * J[b2][l];
        cov[a][b2] = acc;
      }
    cov[0][0] += 0.3; cov[1][1] += 0.3;
    const double det = cov[0][0] * cov[1][1] - cov[0][1] * cov[1][0];
    if (!(det > 0)) { g.ok = false; continue; }
    g.q[0] = cov[1][1] / det; g.q[1] = -cov[0][1] / det; g.q[2] = cov[0][0] / det;
    g.c[0] = fx * t[0] / t[2] + ox; g.c[1] = fy * t[1] / t[2] + oy;
    g.rho_cut = std::fmin((double)cfg->rho_max, 2.0 * std::log(g.o / (double)cfg->alpha_min));
    const float pff[3] = {(float)p[0], (float)p[1], (float)p[2]};
    std::vector<float> shf(48);
    for (int k = 0; k < 48; ++k) shf[(size_t)k] = (float)sh[48 * (size_t)j + k];
    uint8_t cl;
    surfel_colour(pff, shf.data(), cfg->sh_degree, campos, g.rgb, &cl);
  }
  double Lb = 0.0;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : Lb)
  for (int y = wy0; y < wy1; ++y) {
    struct Cand { uint32_t key; int j; double alpha; };
    std::vector<Cand> cands;
    for (int x = wx0; x < wx1; ++x) {
      cands.clear();
      for (int j = 0; j < n; ++j) {
        const G& g = gs[(size_t)j];
        if (!g.ok) continue;
        const double dx = x - g.c[0], dy = y - g.c[1];
        const double rho = g.q[0] * dx * dx + 2 * g.q[1] * dx * dy + g.q[2] * dy * dy;
        if (rho > g.rho_cut) continue;
        cands.push_back({g.key, j, std::fmin((double)cfg->alpha_max, g.o * std::exp(-0.5 * rho))});
      }
      std::sort(cands.begin(), cands.end(), [](const Cand& a, const Cand& b) { return a.key != b.key ? a.key < b.key : a.j < b.j; });
      double Tr = 1.0, C[3] = {0, 0, 0}, D = 0;
      uint32_t cnt = 0;
      for (const Cand& c : cands) {
        const double Tn = Tr * (1.0 - c.alpha);
        if (Tn < (double)cfg->t_min) break;
        const double w = c.alpha * Tr;
        const G& g = gs[(size_t)c.j];
        for (int k = 0; k < 3; ++k) C[k] += w * g.rgb[k];
        D += w * g.z;
        if (vis_count) {
#pragma omp atomic
          vis_count[c.j] += 1;
        }
        if (contrib_sum) {
#pragma omp atomic
          contrib_sum[c.j] += w;
        }
        Tr = Tn;
        ++cnt;
      }
      const size_t p = (size_t)y * W + x;
      for (int k = 0; k < 3; ++k) color[k * HW + p] = C[k] + Tr * (double)cfg->bg[k];
      alpha[p] = 1.0 - Tr;
      depth[p] = D;
      if (n_blended) n_blended[p] = cnt;
      const double m = mask ? (mask[p] ? 1.0 : 0.0) : 1.0;  // no mask: every pixel is object (M = 1), L_b = 0
      Lb += (1.0 - Tr) * (1.0 - m);
    }
  }
  return Lb / (double)HW;
}

}  // extern "C" (3D render)

// SH basis exposed for the orthonormality pin (tests integrate Y_i Y_j over the sphere by quadrature).
void orc_sh_basis(const double* dir, double* Y16) { sh_basis(dir, Y16, nullptr); }

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// number of OpenMP threads of the following calls (bench.py times the oracle on 1 core and on all cores); returns the value in force
int orc_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n;
  return 1;
#endif
}

}  // extern "C"
