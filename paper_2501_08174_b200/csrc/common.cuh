// common.cuh -- shared declarations of libocgs (sm_100a). Internal; the public boundary is include/ocgs.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ocgs.h"

namespace ocgs {

constexpr int kTile = 16;
// pixel block of one forward warp inside the tile (32 pixels); bit w of a list entry's `hit` byte refers to block w,
// numbered row-major.  8x4 blocks are cut by fewer splat outlines than 16x2 strips, so fewer (warp, entry) pairs are walked.
// (16x2 strips and 4x8 blocks measured slower: step 2.30 / 2.35 ms against 2.21 ms.)
constexpr int kSubW = 8, kSubH = 32 / kSubW;
constexpr int kRec = 24;  // floats per raster record (96 B = 6 x float4)
// Record layout.  With c = c2d the projected centre, A0 = M0 - cx*M2, A1 = M1 - cy*M2 (third
// components are the exact division residuals), the pixel ray (x, y) meets the surfel plane at (u,v) = (qx,qy)/qz with
//   q = (dx*M2 - A0) x (dy*M2 - A1) = R - dx*P - dy*Q,   dx = x - cx, dy = y - cy,
//   P = M2 x A1,  Q = A0 x M2,  R = A0 x A1,  and the hit depth is z = M2.(u,v,1) = D0/qz with D0 = M2.R
// (M2.P = M2.Q = 0).  P, Q, R, D0 are formed in fp64 from the fp32 M and rounded once.
//   f4[0] = (Px, Py, Pz, Qx)  f4[1] = (Qy, Qz, Rx, Ry)  f4[2] = (Rz, D0, cx, cy)
//   f4[3] = (rho_cut, z_j, bits(ix0 | iy0<<16), bits(ix1 | iy1<<16))  f4[4] = (opacity, r, g, b)  f4[5] = (nx, ny, nz, 0)
enum RecField {
  R_PX = 0, R_PY, R_PZ, R_QX, R_QY, R_QZ, R_RX, R_RY, R_RZ, R_D0, R_CX, R_CY, R_RHOCUT, R_ZJ, R_RECT0, R_RECT1, R_OPA, R_COLR,
  R_COLG, R_COLB, R_NX, R_NY, R_NZ, R_PAD
};
// gradient accumulator layout in ws.grad_rec (by rank, stride kRec): 16 "main" fields reduced by the transposing
// butterfly, 4 "extra" fields that are non-zero only with a depth gradient or when the filter term wins
enum GradField {
  G_PX = 0, G_PY, G_PZ, G_QX, G_QY, G_QZ, G_RX, G_RY, G_RZ, G_OPA, G_COLR, G_COLG, G_COLB, G_NX, G_NY, G_NZ,
  G_D0, G_ZJ, G_CX, G_CY, G_COUNT
};

#ifndef OCGS_SORT_ITEMS
#define OCGS_SORT_ITEMS 16
#endif
constexpr int kSortItems = OCGS_SORT_ITEMS;           // keys per thread in a radix pass
constexpr int kSortThreads = 256;
constexpr int kSortTile = kSortItems * kSortThreads;  // 4096 keys per block
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

struct Workspace {
  ocgs_header* header;
  uint32_t* depth_bits;
  ushort4* rect;
  uint32_t* tiles;
  uint8_t* clamp;
  float* rec_id;
  uint32_t* id_to_rank;
  uint32_t* rank_to_id;
  float* rec;
  uint32_t* offsets;
  uint32_t* tile_keys;
  uint32_t* tile_vals;
  uint32_t* ranges;
  float* grad_rec;
  float* loss_partial;
  float* final_T;
  // scratch
  uint32_t* dkeyA; uint32_t* dkeyB; uint32_t* dvalB;  // depth sort ping-pong (dvalA == rank_to_id)
  uint32_t* tkeyB; uint32_t* tvalB;                   // tile sort ping-pong
  uint2* blist;                                       // [key_capacity] per tile, at its list offset: the entries some warp blended, in list order:
                                                      // x = rank, y = (position in the tile list << 8) | bit w: warp block w blended it (fwd -> bwd)
  uint32_t* hist;                                     // [4 passes][max_blocks][kRadix] look-back status words of the radix passes
  uint32_t* digit_total;                              // [4][kRadix] global digit histograms + [4] tile tickets
  uint32_t* tcount;                                   // [N] tiles touched by rank
  uint32_t* blocksum;                                 // [ceil(N/1024)+1]
  uint32_t* tile_work;                                // [n_tiles] forward: list length; backward: number of blended entries of the tile
  uint32_t* tile_order;                               // [n_tiles] tiles in descending order of work (heavy tiles first)
  int n, width, height, tiles_x, tiles_y, n_tiles;
  size_t key_capacity;
};

// host: carve `ws` into sections. Returns false when the sizes are unsupported.
bool carve_workspace(void* ws, int n, int width, int height, size_t key_capacity, Workspace* out, ocgs_ws_layout* layout);

extern thread_local int g_last_cuda_error;
inline int cuda_fail(cudaError_t e) { g_last_cuda_error = (int)e; return OCGS_ERR_CUDA; }
#define OCGS_CUDA_OK(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) return ::ocgs::cuda_fail(_e); } while (0)
#define OCGS_LAUNCH_OK() do { cudaError_t _e = cudaGetLastError(); if (_e != cudaSuccess) return ::ocgs::cuda_fail(_e); } while (0)
// diagnostic per-launch timing (ocgs_profile_begin/end): when enabled on this thread, an event is recorded after each launch
extern thread_local bool g_prof_on;
void prof_mark(cudaStream_t st, const char* name);
#define OCGS_LAUNCHED(st, name) do { OCGS_LAUNCH_OK(); if (::ocgs::g_prof_on) ::ocgs::prof_mark(st, name); } while (0)

struct CamParams {
  float V[12];  // rows 0..2 of the view matrix
  float fx, fy, ox, oy;  // ox = cx - 1/2, oy = cy - 1/2 (Appendix A step 4)
  float campos[3];
  int W, H, tiles_x, tiles_y;
};
CamParams make_cam(const ocgs_camera& c);

// stage launchers (each returns an OCGS_* code)
int launch_preprocess(const ocgs_surfels& s, const CamParams& cam, const ocgs_config& cfg, Workspace& w, cudaStream_t st, bool colour = true);
int launch_render_stats(const CamParams& cam, const ocgs_config& cfg, const Workspace& w, uint32_t* vis_count, float* contrib_sum,
                        int prim, cudaStream_t st);
int launch_bin_sort(const CamParams& cam, Workspace& w, uint32_t* sorted_ids, cudaStream_t st);
int launch_render_fwd(const CamParams& cam, const ocgs_config& cfg, const Workspace& w, const uint8_t* mask, float* color,
                      float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg, uint32_t* vis_count,
                      float* contrib_sum, float* mom, int prim, const float* target, float* gC, float* loss_l1, cudaStream_t st);
int launch_preprocess3d(const ocgs_gaussians3d& g, const CamParams& cam, const ocgs_config& cfg, Workspace& w, cudaStream_t st);
int launch_render_bwd(const ocgs_surfels& s, const CamParams& cam, const ocgs_config& cfg, Workspace& w, const uint8_t* mask,
                      const float* final_T, const uint32_t* n_contrib, const float* gC, const float* gA, const float* gD,
                      const float* gN, const float* mom, const float* gM1, const float* gM2, float* d_pos, float* d_scale, float* d_quat, float* d_opacity, float* d_sh,
                      float* d_center2d, cudaStream_t st);

int launch_prune(const ocgs_surfels& in, uint32_t* vis_count, float* contrib_sum, const ocgs_config& cfg, uint8_t* prune_mask,
                 int32_t* remap, const ocgs_surfels_mut* out, int* n_out, int reset_stats, void* ws, cudaStream_t st);

size_t densify_workspace_bytes(int n);
int launch_densify_accumulate(const Workspace& w, const float* d_center2d, float* grad_accum, uint32_t* denom, cudaStream_t st);
int launch_densify(const ocgs_surfels& in, const float* grad_accum, const uint32_t* denom, float grad_threshold, float scale_threshold,
                   const float* xi, const ocgs_surfels_mut& out, int32_t* src, int* counts, void* ws, cudaStream_t st);
int launch_compact_rows(const float* in, const int32_t* remap, int n, int row_floats, float* out, cudaStream_t st);

int launch_masked_l1(const float* color, const float* target, const uint8_t* mask, int W, int H, float* dL_dcolor, float* loss,
                     float* partial, int n_partial, cudaStream_t st);

size_t regularizers_workspace_bytes(int W, int H);
int launch_regularizers(const float* alpha, const float* depth, const float* mom, const float* normal, const ocgs_camera& c, float w_d,
                        float w_n, float* gA, float* gD, float* gM, float* gN, float* loss, void* scratch, cudaStream_t st);
size_t photometric_workspace_bytes(int W, int H);
int launch_photometric(const float* color, const float* target, const uint8_t* mask, int W, int H, float lam, float* dL_dcolor,
                       float* loss, void* scratch, cudaStream_t st);

// tile_order <- tiles sorted by descending tile_work (bucketed; launch order of the raster CTAs)
int launch_order_tiles(const Workspace& w, bool from_ranges, cudaStream_t st, bool clear_grad_rec = false);

// stable LSD radix sort of (u32 key, u32 value) pairs on bits [0, key_bits); count is read from the device (*n_ptr, u64 or
// u32 selected by n_is_u64) and bounded by n_max for grid sizing. Result lands in (keysA, valsA) when the number of
// passes is even, else in (keysB, valsB); returns that through *result_in_B.
int radix_sort_pairs(uint32_t* keysA, uint32_t* valsA, uint32_t* keysB, uint32_t* valsB, const void* n_ptr, bool n_is_u64,
                     size_t n_max, int key_bits, uint32_t* status, uint32_t* ghist, bool* result_in_B, cudaStream_t st,
                     bool prepared = false);

#ifdef __CUDACC__
// MUFU approximations (1-2 ulp, flush-to-zero): enough for the 1e-4 / 1e-3 tolerances, no denormal fix-up code
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2_approx(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
constexpr float kNegHalfLog2e = -0.72134752044448170f;  // exp(-rho/2) = 2^(rho * -0.5 log2 e)
#endif

__host__ __device__ inline size_t div_up(size_t a, size_t b) { return (a + b - 1) / b; }

// number of SMs of the current device (queried once per thread; grids of the persistent / grid-stride kernels are multiples of it)
int sm_count();

}  // namespace ocgs
