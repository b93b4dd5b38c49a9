// raster_fwd.cu -- ocgs_render_fwd and its variants (O4-O6, O8): one CTA per 16x16 tile, one thread per pixel, warp w owns the
// kSubW x kSubH pixel block w; the tile's depth-ordered list is walked front to back in shared-memory batches of records:
// per 32 entries an entry-parallel conservative cull against the warp's block, then the pixel-parallel walk of the
// survivors; early stop per pixel, per warp and per CTA.  Fused: background loss L_b (Eq. 1), the visibility
// statistics, the compact list of blended entries handed to the backward pass, and optionally the depth
// moments (kMoments, f-2), the harness masked-L1 term (kL1, f-1) or the 3D-Gaussian pair rule (kPrim = 1, f-3).
#include <cooperative_groups.h>
#include <stdlib.h>

#include "common.cuh"

namespace ocgs {

constexpr int kFwdBatch = 256;                 // list entries staged per batch (= block size; 128 measured 2 % slower)
constexpr float kContribFix = 134217728.0f;    // 2^27: alpha*T in fixed point for the warp-wide REDUX sum

// Conservative test "can surfel (r0..r3) contribute to any pixel of the kSubW x kSubH block with first pixel (x0, y0)?", run by ONE
// lane per list entry (32 entries per warp step) so that the pixel-parallel walk below only visits survivors.
// A pair contributes iff rho = min(rho3, rho2) <= rho_cut (S6).  Per pixel row dy = y - cy:
//   rho3 <= rc  <=>  F(dx) = |S - dx P|_W^2 <= 0,  S = R - dy Q,  W = diag(1, 1, -rc)   (q = R - dx P - dy Q, rho3 = (qx^2+qy^2)/qz^2)
//   i.e. A dx^2 - 2 B dx + C <= 0 with A = P.WP, B = S.WP, C = S.WS: real roots (B -+ sqrt(B^2 - AC))/A must overlap the
//   block's dx range; rho2 <= rc is a disc of radius sqrt(rc sigma_f^2) about the centre.
// Every inequality is relaxed (rc by 1e-4 relative + 1e-4, the dx range by 0.01 px, the discriminant by 1e-5 of its
// term magnitudes), far more than the fp32 error of either this test (approximate square root included: 2^-22 relative, < 1e-3 px
// on a root interval 1000 px wide) or the per-pixel evaluation, so a pair the walk
// would blend is never culled: the images are bit-identical with and without the cull.
__device__ __forceinline__ bool block_may_contribute(const float4 r0, const float4 r1, const float4 r2, const float4 r3, int x0, int y0,
                                                     float inv_sigma2) {
  constexpr int kW = kSubW, kH = kSubH;  // the warp's pixel block (common.cuh)
  const uint32_t b0 = __float_as_uint(r3.z), b1 = __float_as_uint(r3.w);
  const int ix0 = (int)(b0 & 0xFFFFu), iy0 = (int)(b0 >> 16), ix1 = (int)(b1 & 0xFFFFu), iy1 = (int)(b1 >> 16);
  if (iy1 < y0 || iy0 > y0 + kH - 1 || ix1 < x0 || ix0 > x0 + kW - 1) return false;  // pixel rect (S7) misses the block
  const float rc = fmaf(r3.x, 1.0001f, 1e-4f);
  const float dxa = ((float)x0 - r2.z) - 0.01f, dxb = ((float)(x0 + kW - 1) - r2.z) + 0.01f;
  const float dxn = fminf(fmaxf(0.0f, dxa), dxb);  // dx of the range closest to the centre
  const float Px = r0.x, Py = r0.y, Pz = r0.z, Qx = r0.w, Qy = r1.x, Qz = r1.y, Rx = r1.z, Ry = r1.w, Rz = r2.x;
  const float Ap = fmaf(Px, Px, Py * Py), An = rc * Pz * Pz, A = Ap - An;
  bool keep = !(A > 0.0f);  // not an ellipse along x (cannot happen after the a < 0 cull): keep
#pragma unroll
  for (int row = 0; row < kH; ++row) {
    const float dy = (float)(y0 + row) - r2.w;
    keep |= fmaf(dxn, dxn, dy * dy) * inv_sigma2 <= rc;  // filter disc (S8)
    const float Sx = fmaf(-dy, Qx, Rx), Sy = fmaf(-dy, Qy, Ry), Sz = fmaf(-dy, Qz, Rz);
    const float Cp = fmaf(Sx, Sx, Sy * Sy), Cn = rc * Sz * Sz;
    const float B = fmaf(Sx, Px, fmaf(Sy, Py, -rc * Sz * Pz));
    const float disc = fmaf(B, B, -A * (Cp - Cn)) + 1e-5f * (Ap + An) * (Cp + Cn);
    const float sq = sqrt_approx(fmaxf(disc, 0.0f));  // one MUFU: sqrtf takes its slow path (a call) at 0, i.e. on every row that misses
    keep |= disc >= 0.0f && (B - sq) <= A * dxb && (B + sq) >= A * dxa;
  }
  return keep;
}

// The same conservative block test for the 3D-Gaussian variant (gaussian3d.cu): rho = a dx^2 + 2 b dx dy + c dy^2 <= rc,
// per pixel row a quadratic in dx with roots (-b dy -+ sqrt((b dy)^2 - a (c dy^2 - rc))) / a.
__device__ __forceinline__ bool block_may_contribute3d(const float4 r0, const float4 r2, const float4 r3, int x0, int y0) {
  constexpr int kW = kSubW, kH = kSubH;
  const uint32_t b0 = __float_as_uint(r3.z), b1 = __float_as_uint(r3.w);
  const int ix0 = (int)(b0 & 0xFFFFu), iy0 = (int)(b0 >> 16), ix1 = (int)(b1 & 0xFFFFu), iy1 = (int)(b1 >> 16);
  if (iy1 < y0 || iy0 > y0 + kH - 1 || ix1 < x0 || ix0 > x0 + kW - 1) return false;
  const float rc = fmaf(r3.x, 1.0001f, 1e-4f);
  const float dxa = ((float)x0 - r2.z) - 0.01f, dxb = ((float)(x0 + kW - 1) - r2.z) + 0.01f;
  const float a = r0.x, b = r0.y, c = r0.z;
  bool keep = !(a > 0.0f);
#pragma unroll
  for (int row = 0; row < kH; ++row) {
    const float dy = (float)(y0 + row) - r2.w;
    const float B = -b * dy, Cp = c * dy * dy;
    const float disc = fmaf(B, B, -a * (Cp - rc)) + 1e-5f * a * (Cp + rc);
    const float sq = sqrt_approx(fmaxf(disc, 0.0f));  // one MUFU: sqrtf takes its slow path (a call) at 0, i.e. on every row that misses
    keep |= disc >= 0.0f && (B - sq) <= a * dxb && (B + sq) >= a * dxa;
  }
  return keep;
}

// Tiles with long lists finish last, alone on their SM, where two warps per scheduler cannot hide the ~300-cycle dependent
// chain of one survivor: above kFwdHeavyLen entries the walk takes kFwdIlp survivors per iteration (measured at config 5:
// forward 2.34 -> 2.04 ms with 2, 2.07 with 4, 2.09 with 3; used for every tile it costs 3 % at config 3).
constexpr int kFwdIlp = 2;
constexpr uint32_t kFwdHeavyLen = 2048;
#ifndef OCGS_FWD_MIN_BLOCKS
#define OCGS_FWD_MIN_BLOCKS 6
#endif
constexpr int kFwdMinBlocks = OCGS_FWD_MIN_BLOCKS;  // CTAs per SM the register budget is held to (40 registers; 5 (48 registers, no spill) and 7 (32) measured
                                                    // slower at the end of round 2 too: 0.677 / 0.680 vs 0.643 ms at config 3)
// fused harness photometric term (S20): target image in, dL/dcolor and per-tile partial sums of |M (R - I)| out
struct FwdL1 { const float* target; float* gC; float* partial; float inv_norm; };

// Exact segmented compositing of heavy tiles (kSeg = 1).  A tile whose list is longer than kFwdHeavyLen is
// walked by a thread-block CLUSTER of kSegRanks CTAs on kSegRanks SMs, CTA r taking the r-th part of the list:
//   phase A  every CTA walks its part alpha-only and stop-free: P_r(p) = prod (1 - alpha) over the pairs that pass the pair rule;
//   exchange through distributed shared memory: T_in,r(p) = prod_{r' < r} P_r'(p).  The stop rule (S11) fires at the first pair
//            where the running product falls below t_min, and the product is monotone, so "a CTA in front has stopped" is
//            exactly T_in,r < t_min: every blend / stop decision is the serial walk's (up to the rounding of the regrouped product,
//            which matters only where the oracle calls the stop test fragile);
//   phase B  the ordinary walk of the part, started at T = T_in,r: blends, statistics, blended lists;
//   combine  CTA 0 adds the partial sums of the maps in list order (deterministic) through distributed shared memory, takes
//            n_contrib = the last blended position and final T = T_out of the last CTA that was still walking, runs the ordinary
//            epilogue, and packs the kSegRanks blended sub-lists into the one compact list the backward pass walks.
// The launch covers the first kSegMaxTiles positions of the heavy-first tile order; clusters whose tile is not heavy exit at
// once, and the ordinary launch skips the tiles the clusters took.
#ifndef OCGS_SEG_RANKS
#define OCGS_SEG_RANKS 8
#endif
#ifndef OCGS_SEG_LEN
#define OCGS_SEG_LEN 6144
#endif
#ifndef OCGS_SEG_MINB
#define OCGS_SEG_MINB 3
#endif
constexpr int kSegRanks = OCGS_SEG_RANKS;      // CTAs per cluster (8 is the portable maximum, 16 needs the non-portable opt-in)
constexpr uint32_t kSegLen = OCGS_SEG_LEN;     // lists longer than this are segmented
constexpr int kSegMaxTiles = 128;
namespace cg = cooperative_groups;

// kMaps = false: the visibility pass (ocgs_visibility_pass): only the statistics are produced -- no maps, no blended lists, no loss
template <bool kStats, bool kMoments, int kPrim /*0 = 2D surfel, 1 = 3D Gaussian (EWA conic record)*/, bool kL1, bool kMaps = true, int kSeg = 0>
__global__ void __launch_bounds__(256, kSeg ? OCGS_SEG_MINB : kFwdMinBlocks) render_fwd_kernel(const uint32_t* __restrict__ tile_order, uint32_t* __restrict__ tile_work,
                                                            const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ list,
                                                         const float4* __restrict__ rec, const uint32_t* __restrict__ rank_to_id,
                                                         const uint8_t* __restrict__ mask, int W, int H, int tiles_x,
                                                         ocgs_config cfg, float* __restrict__ color, float* __restrict__ alpha,
                                                         float* __restrict__ depth, float* __restrict__ normal,
                                                         uint32_t* __restrict__ n_contrib, float* __restrict__ final_T, uint2* __restrict__ blist, ocgs_header* __restrict__ header, float* __restrict__ loss_partial,
                                                         uint32_t* __restrict__ vis_count, float* __restrict__ contrib_sum, float* __restrict__ mom /*[3,H,W]: origin, m1, m2 (kMoments)*/, FwdL1 l1,
                                                         int seg_tiles /*leading positions of the tile order the segmented launch takes (0: none)*/) {
  static_assert(!kSeg || (!kMoments && kPrim == 0), "segmented compositing: surfel forward (with maps or statistics only), no depth moments");
  __shared__ float4 s_rec[kFwdBatch * 6];
  __shared__ uint32_t s_rank[kFwdBatch];
  __shared__ uint32_t s_hit[kFwdBatch];  // bit w: warp w blended the entry (read by the backward pass)
  __shared__ uint32_t s_cnt[kStats ? kFwdBatch : 1];
  __shared__ uint2 s_fix[kStats ? kFwdBatch : 1];  // sum of alpha*T in 2^-27 fixed point, as (sum of the low 16 bits, sum of the high 16 bits) of
                                                   // the warps' 32-bit terms: two native 32-bit shared atomics instead of a 64-bit CAS loop
  __shared__ float s_red[8];
  __shared__ uint32_t s_wcnt[8];

  __shared__ float s_seg[kSeg ? 11 : 1][kSeg ? 256 : 1];  // kSeg: [0] = P_r, then the CTA's partial results, read by its cluster
  __shared__ uint32_t s_segn;                              // kSeg: length of this CTA's blended sub-list
  const int pos = kSeg ? (int)blockIdx.x / kSegRanks : (int)blockIdx.x;
  const int tile = (int)tile_order[pos];  // heavy tiles are launched first
  const int tx = tile % tiles_x, ty = tile / tiles_x;
  // warp w owns the kSubW x kSubH pixel block number w of the tile (row-major over blocks), lane l pixel (l % kSubW, l / kSubW)
  const int sub = threadIdx.x >> 5, sl = threadIdx.x & 31;
  const int sub_x0 = (sub % (kTile / kSubW)) * kSubW, sub_y0 = (sub / (kTile / kSubW)) * kSubH;
  const int lx = sub_x0 + sl % kSubW, ly = sub_y0 + sl / kSubW;
  const int ix = tx * kTile + lx, iy = ty * kTile + ly;
  const bool inside = ix < W && iy < H;
  const float px = (float)ix, py = (float)iy;
  // Programmatic dependent launch: the ordinary launch follows the segmented one in the stream and needs nothing from it, so the
  // clusters let it start at once and it fills the SMs their long chains leave idle; its LAST CTA waits for the clusters before
  // it exits, so the ordinary grid -- and everything behind it in the stream -- completes only after the segmented one.
  if (kSeg) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  struct PdlJoin {
    bool on;
    __device__ ~PdlJoin() { if (on) asm volatile("griddepcontrol.wait;" ::: "memory"); }
  } pdl_join{!kSeg && seg_tiles > 0 && blockIdx.x == gridDim.x - 1};
  const uint32_t start = ranges[2 * tile], end = ranges[2 * tile + 1];
  if (kSeg ? end - start <= kSegLen : (pos < seg_tiles && end - start > kSegLen)) return;  // (uniform over the CTA / cluster)
  // kSeg: this CTA's part [rs, re) of the list, a multiple of the batch size long so that batches never straddle two parts
  const uint32_t seg_rank = kSeg ? cg::this_cluster().block_rank() : 0u;
  const uint32_t seg_len = kSeg ? (uint32_t)(div_up(div_up((size_t)(end - start), kSegRanks), kFwdBatch) * kFwdBatch) : end - start;
  const uint32_t rs = kSeg ? min(end, start + seg_rank * seg_len) : start, re = kSeg ? min(end, rs + seg_len) : end;
  const float inv_sigma2 = 1.0f / cfg.filter_sigma2;
  const int lane = threadIdx.x & 31;
  const uint32_t wbit = 1u << (threadIdx.x >> 5);
  const float near_z = cfg.near_z, alpha_max = cfg.alpha_max, t_min = cfg.t_min;

  float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f, N0 = 0.f, N1 = 0.f, N2 = 0.f;
  // kMoments: depth moments about the first blended pair's depth zc (reading R-moments): m1 = sum w (z - zc), m2 = sum w (z - zc)^2
  float zc = 0.f, M1 = 0.f, M2 = 0.f;
  uint32_t last = 0;
  uint32_t nhit = 0;  // entries of this tile blended so far (uniform across the CTA)
  bool done = !inside;
  const bool heavy = kSeg || end - start > kFwdHeavyLen;

  if (kSeg) {
    // ---- phase A: alpha-only, stop-free product over this CTA's part; a pixel may leave once P < t_min (all CTAs behind are then
    // cut off whatever the exact value) ----
    float P = 1.0f;
    bool doneA = !inside;
    for (uint32_t b0 = rs; b0 < re; b0 += kFwdBatch) {
      const int cnt = (int)min((uint32_t)kFwdBatch, re - b0);
      if (__syncthreads_and(doneA)) break;
      if ((int)threadIdx.x < cnt) s_rank[threadIdx.x] = list[b0 + threadIdx.x];
      __syncthreads();
      for (int i = threadIdx.x; i < cnt * 5; i += 256) {
        const int e = i / 5, part = i - 5 * e;
        s_rec[6 * e + part] = __ldg(rec + (size_t)s_rank[e] * 6 + part);
      }
      __syncthreads();
      for (int c0 = 0; c0 < cnt; c0 += 32) {
        const int ce = min(32, cnt - c0);
        bool keep = false;
        if (lane < ce) {
          const float4* se = s_rec + 6 * (c0 + lane);
          keep = block_may_contribute(se[0], se[1], se[2], se[3], tx * kTile + sub_x0, ty * kTile + sub_y0, inv_sigma2);
        }
        uint32_t todo = __ballot_sync(0xFFFFFFFFu, keep);
        if (__all_sync(0xFFFFFFFFu, doneA)) break;
        while (todo) {
          const int jj = __ffs(todo) - 1;
          todo &= todo - 1;
          const float4* sr = s_rec + 6 * (c0 + jj);
          const float4 r0 = sr[0], r1 = sr[1], r2 = sr[2], r3 = sr[3];
          const float dx = px - r2.z, dy = py - r2.w;
          const float qx = fmaf(-dy, r0.w, fmaf(-dx, r0.x, r1.z));
          const float qy = fmaf(-dy, r1.x, fmaf(-dx, r0.y, r1.w));
          const float qz = fmaf(-dy, r1.y, fmaf(-dx, r0.z, r2.x));
          const float inv = rcp_approx(qz);
          const float u = qx * inv, v = qy * inv;
          const float rho3 = fmaf(u, u, v * v);
          const float rho2 = fmaf(dx, dx, dy * dy) * inv_sigma2;
          const bool surf = rho3 <= rho2;
          const float rho = surf ? rho3 : rho2;
          const float z = surf ? r2.y * inv : r3.y;
          if (!doneA && qz != 0.0f && !(z < near_z) && !(rho > r3.x)) {
            const float a = fminf(alpha_max, sr[4].x * ex2_approx(rho * kNegHalfLog2e));
            P *= 1.0f - a;
            doneA = P < t_min;
          }
        }
      }
    }
    __syncthreads();
    s_seg[0][threadIdx.x] = P;
    cg::this_cluster().sync();
    for (uint32_t rr = 0; rr < seg_rank; ++rr) T *= *cg::this_cluster().map_shared_rank(&s_seg[0][threadIdx.x], rr);
    done = !inside || T < t_min;  // a CTA in front has met the stop rule (S11)
  }
  const bool done_in = done;

  for (uint32_t b0 = rs; b0 < re; b0 += kFwdBatch) {
    const int cnt = (int)min((uint32_t)kFwdBatch, re - b0);
    if (__syncthreads_and(done)) break;
    if ((int)threadIdx.x < cnt) s_rank[threadIdx.x] = list[b0 + threadIdx.x];
    if (kMaps && threadIdx.x < kFwdBatch) s_hit[threadIdx.x] = 0;
    if (kStats && threadIdx.x < kFwdBatch) { s_cnt[threadIdx.x] = 0; s_fix[threadIdx.x] = make_uint2(0u, 0u); }
    __syncthreads();
    constexpr int kParts = kMaps ? 6 : 5;  // the last 16 bytes of a record hold the normal: not read by the statistics-only walk
    for (int i = threadIdx.x; i < cnt * kParts; i += 256) {
      const int e = i / kParts, part = i - kParts * e;
      s_rec[6 * e + part] = __ldg(rec + (size_t)s_rank[e] * 6 + part);
    }
    __syncthreads();
    // the batch in chunks of 32 entries: lane jj keeps the statistics of entry c0 + jj in registers
    bool all_done = false;
    for (int c0 = 0; c0 < cnt && !all_done; c0 += 32) {
      uint32_t cntr = 0, fixr = 0;
      const int ce = min(32, cnt - c0);
      if (__all_sync(0xFFFFFFFFu, done)) { all_done = true; break; }  // once per 32 entries (before their cull): finished lanes are predicated off below
      // entry-parallel cull: lane l tests entry c0 + l against this warp's pixel block; the walk visits the survivors
      bool keep = false;
      if (lane < ce) {
        const float4* se = s_rec + 6 * (c0 + lane);
        keep = kPrim == 0 ? block_may_contribute(se[0], se[1], se[2], se[3], tx * kTile + sub_x0, ty * kTile + sub_y0, inv_sigma2)
                          : block_may_contribute3d(se[0], se[2], se[3], tx * kTile + sub_x0, ty * kTile + sub_y0);
      }
      uint32_t todo = __ballot_sync(0xFFFFFFFFu, keep);
      if (kPrim == 0 && heavy) {
        // long lists (a lone CTA on its SM at the kernel's tail): kFwdIlp survivors per iteration, evaluated without branches so
        // that their latencies overlap; the blend itself stays in list order and keeps the arithmetic of the loop below
        while (todo) {
          int jj[kFwdIlp]; bool ok[kFwdIlp]; float a[kFwdIlp], z[kFwdIlp];
#pragma unroll
          for (int k = 0; k < kFwdIlp; ++k) {
            const bool on = todo != 0;
            jj[k] = on ? __ffs(todo) - 1 : (k ? jj[0] : 0);
            todo &= todo - 1;
            const float4* sr = s_rec + 6 * (c0 + jj[k]);
            const float4 r0 = sr[0], r1 = sr[1], r2 = sr[2], r3 = sr[3];
            const float dx = px - r2.z, dy = py - r2.w;
            const float qx = fmaf(-dy, r0.w, fmaf(-dx, r0.x, r1.z));
            const float qy = fmaf(-dy, r1.x, fmaf(-dx, r0.y, r1.w));
            const float qz = fmaf(-dy, r1.y, fmaf(-dx, r0.z, r2.x));
            const float inv = rcp_approx(qz);
            const float u = qx * inv, v = qy * inv;
            const float rho3 = fmaf(u, u, v * v);
            const float rho2 = fmaf(dx, dx, dy * dy) * inv_sigma2;
            const bool surf = rho3 <= rho2;
            const float rho = surf ? rho3 : rho2;
            const float zz = surf ? r2.y * inv : r3.y;
            ok[k] = on && qz != 0.0f && !(zz < near_z) && !(rho > r3.x);
            z[k] = ok[k] ? zz : 0.0f;
            a[k] = fminf(alpha_max, sr[4].x * ex2_approx(rho * kNegHalfLog2e));
            if (!on) jj[k] = -1;
          }
#pragma unroll
          for (int k = 0; k < kFwdIlp; ++k) {
            const int j = jj[k] < 0 ? 0 : jj[k];
            const float4* sr = s_rec + 6 * (c0 + j);
            const float Tn = T * (1.0f - a[k]);
            const bool live = ok[k] && !done;
            const bool blend = live && !(Tn < t_min);
            done = done || (live && Tn < t_min);  // S11: stop before blending this pair
            const float wgt = blend ? a[k] * T : 0.0f;
            if (kMaps) {
              const float4 r4 = sr[4], r5 = sr[5];
              C0 = fmaf(wgt, r4.y, C0); C1 = fmaf(wgt, r4.z, C1); C2 = fmaf(wgt, r4.w, C2);
              D = fmaf(wgt, z[k], D);
              if (kMoments) {
                zc = (blend && last == 0) ? z[k] : zc;
                const float dz = blend ? z[k] - zc : 0.0f;
                M1 = fmaf(wgt, dz, M1);
                M2 = fmaf(wgt * dz, dz, M2);
              }
              N0 = fmaf(wgt, r5.x, N0); N1 = fmaf(wgt, r5.y, N1); N2 = fmaf(wgt, r5.z, N2);
              last = blend ? (b0 - start) + c0 + j + 1 : last;
            }
            T = blend ? Tn : T;
            const unsigned bal = __ballot_sync(0xFFFFFFFFu, blend);
            unsigned fix = 0;
            if (kStats) fix = __reduce_add_sync(0xFFFFFFFFu, (unsigned)__float2uint_rn(wgt * kContribFix));
            if (lane == jj[k]) { fixr = fix; cntr = (uint32_t)__popc(bal); }
          }
        }
      } else
      while (todo) {
        const int jj = __ffs(todo) - 1;
        todo &= todo - 1;
        const float4* sr = s_rec + 6 * (c0 + jj);
        const float4 r0 = sr[0], r1 = sr[1], r2 = sr[2], r3 = sr[3];
        const float dx = px - r2.z, dy = py - r2.w;
        float rho, z, qz;
        if (kPrim == 0) {
          // O4 from the record: q = R - dx P - dy Q, (u,v) = (qx,qy)/qz, hit depth D0/qz
          const float qx = fmaf(-dy, r0.w, fmaf(-dx, r0.x, r1.z));
          const float qy = fmaf(-dy, r1.x, fmaf(-dx, r0.y, r1.w));
          qz = fmaf(-dy, r1.y, fmaf(-dx, r0.z, r2.x));
          const float inv = rcp_approx(qz);
          const float u = qx * inv, v = qy * inv;
          const float rho3 = fmaf(u, u, v * v);
          const float rho2 = fmaf(dx, dx, dy * dy) * inv_sigma2;
          const bool surf = rho3 <= rho2;
          rho = surf ? rho3 : rho2;
          z = surf ? r2.y * inv : r3.y;
        } else {
          // R-3D: rho = d^T Sigma'^-1 d, depth of the pair = centre depth
          rho = fmaf(r0.x * dx, dx, fmaf(2.0f * r0.y * dx, dy, r0.z * dy * dy));
          z = r3.y;
          qz = 1.0f;
        }
        bool blend = false;
        float wgt = 0.f;
        unsigned fixl = 0;  // this pixel's term of contrib_sum, fixed point
        if (!done && qz != 0.0f && !(z < near_z) && !(rho > r3.x)) {
          const float4 r4 = sr[4];
          const float a = fminf(alpha_max, r4.x * ex2_approx(rho * kNegHalfLog2e));
          const float Tn = T * (1.0f - a);
          if (Tn < t_min) {
            done = true;  // S11: stop before blending this pair
          } else {
            wgt = a * T;
            if (kMaps) {
              const float4 r5 = sr[5];
              C0 = fmaf(wgt, r4.y, C0); C1 = fmaf(wgt, r4.z, C1); C2 = fmaf(wgt, r4.w, C2);
              D = fmaf(wgt, z, D);
              if (kMoments) {
                if (last == 0) zc = z;
                const float dz = z - zc;
                M1 = fmaf(wgt, dz, M1);
                M2 = fmaf(wgt * dz, dz, M2);
              }
              N0 = fmaf(wgt, r5.x, N0); N1 = fmaf(wgt, r5.y, N1); N2 = fmaf(wgt, r5.z, N2);
              last = (b0 - start) + c0 + jj + 1;
            }
            if (kStats) fixl = (unsigned)__float2uint_rn(wgt * kContribFix);
            T = Tn;
            blend = true;
          }
        }
        // no branch on "some lane blended": 87 % of the visits blend, and the test costs more than the reduction it skips
        const unsigned bal = __ballot_sync(0xFFFFFFFFu, blend);
        if (kStats) {
          const unsigned fix = __reduce_add_sync(0xFFFFFFFFu, fixl);
          if (lane == jj) fixr = fix;
        }
        if (lane == jj) cntr = (uint32_t)__popc(bal);
      }
      if (cntr) {
        if (kMaps) atomicOr(&s_hit[c0 + lane], wbit);
        if (kStats) {
          atomicAdd(&s_cnt[c0 + lane], cntr);
          atomicAdd(&s_fix[c0 + lane].x, fixr & 0xFFFFu);
          atomicAdd(&s_fix[c0 + lane].y, fixr >> 16);
        }
      }
    }
    __syncthreads();
    if (kMaps) {  // append the entries some warp blended to the tile's blended list (walked back to front by render_bwd)
      const bool hitme = (int)threadIdx.x < cnt && s_hit[threadIdx.x] != 0;
      const unsigned bal = __ballot_sync(0xFFFFFFFFu, hitme);
      if (lane == 0) s_wcnt[threadIdx.x >> 5] = (uint32_t)__popc(bal);
      __syncthreads();
      uint32_t before = 0, total = 0;
#pragma unroll
      for (int w2 = 0; w2 < 8; ++w2) {
        const uint32_t c = s_wcnt[w2];
        if (w2 < (int)(threadIdx.x >> 5)) before += c;
        total += c;
      }
      if (hitme)
        blist[rs + nhit + before + (uint32_t)__popc(bal & ((1u << lane) - 1u))] =
            make_uint2(s_rank[threadIdx.x], (((b0 - start) + threadIdx.x) << 8) | s_hit[threadIdx.x]);
      nhit += total;
    }
    if (kStats) {
      if ((int)threadIdx.x < cnt && s_cnt[threadIdx.x] > 0) {
        const uint32_t id = rank_to_id[s_rank[threadIdx.x]];
        atomicAdd(&vis_count[id], s_cnt[threadIdx.x]);
        atomicAdd(&contrib_sum[id], (float)(((unsigned long long)s_fix[threadIdx.x].y << 16) + s_fix[threadIdx.x].x) * (1.0f / kContribFix));
      }
    }
  }

  if (!kMaps) {
    // statistics only: nothing to combine (every CTA has flushed its own counts); a cluster CTA stays until its cluster has read
    // its P_r through distributed shared memory
    if (kSeg) cg::this_cluster().sync();
    return;
  }
  if (kSeg) {
    cg::cluster_group cl = cg::this_cluster();
    const int t = (int)threadIdx.x;
    s_seg[1][t] = C0; s_seg[2][t] = C1; s_seg[3][t] = C2; s_seg[4][t] = D; s_seg[5][t] = N0; s_seg[6][t] = N1; s_seg[7][t] = N2;
    s_seg[8][t] = T; s_seg[9][t] = __uint_as_float(last); s_seg[10][t] = done_in ? 1.0f : 0.0f;
    if (t == 0) s_segn = nhit;
    __threadfence();  // this CTA's part of the blended list is visible to CTA 0
    cl.sync();
    if (seg_rank != 0) { cl.sync(); return; }  // (CTA 0 has read this CTA's shared memory when the second barrier completes)
    uint32_t packed = nhit;  // blended entries in front of the sub-list being moved
    for (uint32_t rr = 1; rr < (uint32_t)kSegRanks; ++rr) {
      const float* rp = cl.map_shared_rank(&s_seg[0][0], rr);
      C0 += rp[1 * 256 + t]; C1 += rp[2 * 256 + t]; C2 += rp[3 * 256 + t]; D += rp[4 * 256 + t];
      N0 += rp[5 * 256 + t]; N1 += rp[6 * 256 + t]; N2 += rp[7 * 256 + t];
      if (rp[10 * 256 + t] == 0.0f) T = rp[8 * 256 + t];  // that CTA was still walking: its T_out is the pixel's transmittance so far
      last = max(last, __float_as_uint(rp[9 * 256 + t]));
      // its blended sub-list moves down behind the ones in front of it (never up: chunks are read before they are written)
      const uint32_t cnt_r = *cl.map_shared_rank(&s_segn, rr);
      const uint32_t src = min(end, start + rr * seg_len), dst = start + packed;
      if (dst != src)
        for (uint32_t i0 = 0; i0 < cnt_r; i0 += 256) {
          uint2 e = make_uint2(0u, 0u);
          if (i0 + t < cnt_r) e = __ldcg(blist + src + i0 + t);
          __syncthreads();
          if (i0 + t < cnt_r) blist[dst + i0 + t] = e;
          __syncthreads();
        }
      packed += cnt_r;
    }
    nhit = packed;
    cl.sync();
  }
  const float A = 1.0f - T;
  float l1sum = 0.f;
  if (inside) {
    const size_t HW = (size_t)W * H, p = (size_t)iy * W + ix;
    color[p] = fmaf(T, cfg.bg[0], C0); color[HW + p] = fmaf(T, cfg.bg[1], C1); color[2 * HW + p] = fmaf(T, cfg.bg[2], C2);
    alpha[p] = A;
    depth[p] = D;
    if (kMoments) { mom[p] = zc; mom[HW + p] = M1; mom[2 * HW + p] = M2; }
    if (kPrim == 0) { normal[p] = N0; normal[HW + p] = N1; normal[2 * HW + p] = N2; }  // the 3D variant has no normal map
    n_contrib[p] = last;
    final_T[p] = T;
    if (kL1) {  // masked L1 against the target, straight from the registers that hold the pixel's colour
      const bool m = mask == nullptr || mask[p] != 0;
      const float col[3] = {fmaf(T, cfg.bg[0], C0), fmaf(T, cfg.bg[1], C1), fmaf(T, cfg.bg[2], C2)};
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float d = m ? col[c] - l1.target[c * HW + p] : 0.f;
        l1sum += fabsf(d);
        l1.gC[c * HW + p] = d > 0.f ? l1.inv_norm : (d < 0.f ? -l1.inv_norm : 0.f);
      }
    }
  }
  if (threadIdx.x == 0) {
    tile_work[tile] = nhit;  // length of the blended list: the backward pass's loop bound and work estimate
    if (end - start >= (1u << 24)) atomicOr(&header->error, 2u);  // list positions are packed into 24 bits of blist.y
  }
  if (loss_partial) {  // Eq. 1: A (1 - M), fixed-order reduction -> deterministic
    float lb = 0.f;
    if (inside) lb = (mask != nullptr && mask[(size_t)iy * W + ix] == 0) ? A : 0.f;  // mask == NULL: M = 1 everywhere, L_b = 0 (ocgs.h)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lb += __shfl_xor_sync(0xFFFFFFFFu, lb, o);
    __syncthreads();
    if (lane == 0) s_red[threadIdx.x >> 5] = lb;
    __syncthreads();
    if (threadIdx.x == 0) {
      float s = 0.f;
#pragma unroll
      for (int w2 = 0; w2 < 8; ++w2) s += s_red[w2];
      loss_partial[tile] = s;
    }
  }
  if (kL1) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) l1sum += __shfl_xor_sync(0xFFFFFFFFu, l1sum, o);
    __syncthreads();
    if (lane == 0) s_red[threadIdx.x >> 5] = l1sum;
    __syncthreads();
    if (threadIdx.x == 0) {
      float s = 0.f;
#pragma unroll
      for (int w2 = 0; w2 < 8; ++w2) s += s_red[w2];
      l1.partial[tile] = s;
    }
  }
}

__global__ void __launch_bounds__(1024) loss_final_kernel(const float* __restrict__ partial, int n_tiles, float inv_hw,
                                                          float* __restrict__ loss_bg, const float* __restrict__ partial2, float scale2,
                                                          float* __restrict__ loss2) {
  __shared__ double s[2][1024];
  double acc = 0.0, acc2 = 0.0;
  for (int i = threadIdx.x; i < n_tiles; i += 1024) {
    if (loss_bg) acc += (double)partial[i];
    if (loss2) acc2 += (double)partial2[i];
  }
  s[0][threadIdx.x] = acc; s[1][threadIdx.x] = acc2;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) { s[0][threadIdx.x] += s[0][threadIdx.x + o]; s[1][threadIdx.x] += s[1][threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (loss_bg) *loss_bg = (float)(s[0][0] * (double)inv_hw);
    if (loss2) *loss2 = (float)(s[1][0] * (double)scale2);
  }
}

// The visibility pass: statistics only ("rendering all training views"): same pair rule, same transmittance
// chain and stop rule as the forward pass -- vis_count is bit-identical -- without the colour / depth / normal blends, the
// maps, L_b and the blended lists.
int launch_render_stats(const CamParams& cam, const ocgs_config& cfg, const Workspace& w, uint32_t* vis_count, float* contrib_sum,
                        int prim, cudaStream_t st) {
  if (w.n_tiles == 0) return OCGS_OK;
  int rc = launch_order_tiles(w, /*from_ranges=*/true, st);
  if (rc != OCGS_OK) return rc;
  FwdL1 l1 = {nullptr, nullptr, nullptr, 0.f};
  // heavy tiles (surfels): the same clusters as the full forward pass, transmittance exchange only; the ordinary launch overlaps them
  static const bool seg_on = [] { const char* e = getenv("OCGS_FWD_SEGMENTED"); return !e || atoi(e) != 0; }();
  const int seg_tiles = (prim == 0 && seg_on) ? min(w.n_tiles, kSegMaxTiles) : 0;
  if (seg_tiles > 0) {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)(seg_tiles * kSegRanks)); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = kSegRanks; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    lc.attrs = at; lc.numAttrs = 1;
    if (kSegRanks > 8) OCGS_CUDA_OK(cudaFuncSetAttribute(render_fwd_kernel<true, false, 0, false, false, 1>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    OCGS_CUDA_OK(cudaLaunchKernelEx(&lc, render_fwd_kernel<true, false, 0, false, false, 1>, (const uint32_t*)w.tile_order, w.tile_work, (const uint32_t*)w.ranges,
                                    (const uint32_t*)w.tile_vals, (const float4*)w.rec, (const uint32_t*)w.rank_to_id, (const uint8_t*)nullptr, cam.W, cam.H, cam.tiles_x, cfg,
                                    (float*)nullptr, (float*)nullptr, (float*)nullptr, (float*)nullptr, (uint32_t*)nullptr, (float*)nullptr, (uint2*)nullptr, w.header,
                                    (float*)nullptr, vis_count, contrib_sum, (float*)nullptr, l1, seg_tiles));
    OCGS_LAUNCHED(st, "render_stats_seg_kernel");
  }
  if (prim == 1)
    render_fwd_kernel<true, false, 1, false, false><<<w.n_tiles, 256, 0, st>>>(w.tile_order, w.tile_work, w.ranges, w.tile_vals, (const float4*)w.rec,
        w.rank_to_id, nullptr, cam.W, cam.H, cam.tiles_x, cfg, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, w.header, nullptr,
        vis_count, contrib_sum, nullptr, l1, 0);
  else {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)w.n_tiles); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = at; lc.numAttrs = seg_tiles > 0 ? 1 : 0;
    OCGS_CUDA_OK(cudaLaunchKernelEx(&lc, render_fwd_kernel<true, false, 0, false, false>, (const uint32_t*)w.tile_order, w.tile_work, (const uint32_t*)w.ranges,
                                    (const uint32_t*)w.tile_vals, (const float4*)w.rec, (const uint32_t*)w.rank_to_id, (const uint8_t*)nullptr, cam.W, cam.H, cam.tiles_x, cfg,
                                    (float*)nullptr, (float*)nullptr, (float*)nullptr, (float*)nullptr, (uint32_t*)nullptr, (float*)nullptr, (uint2*)nullptr, w.header,
                                    (float*)nullptr, vis_count, contrib_sum, (float*)nullptr, l1, seg_tiles));
  }
  OCGS_LAUNCHED(st, "render_stats_kernel");
  return OCGS_OK;
}

int launch_render_fwd(const CamParams& cam, const ocgs_config& cfg, const Workspace& w, const uint8_t* mask, float* color,
                      float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg, uint32_t* vis_count,
                      float* contrib_sum, float* mom, int prim, const float* target, float* gC, float* loss_l1, cudaStream_t st) {
  if (w.n_tiles == 0) return OCGS_OK;
  int rc = launch_order_tiles(w, /*from_ranges=*/true, st);  // launch order: longest lists first
  if (rc != OCGS_OK) return rc;
  const bool stats = vis_count != nullptr && contrib_sum != nullptr;
  float* lp = loss_bg ? w.loss_partial : nullptr;
  FwdL1 l1 = {target, gC, w.loss_partial + w.n_tiles, (float)(1.0 / (3.0 * (double)cam.W * (double)cam.H))};
  // heavy tiles of the surfel forward (no depth moments): clusters of kSegRanks CTAs over the first positions of the tile order
  static const bool seg_on = [] { const char* e = getenv("OCGS_FWD_SEGMENTED"); return !e || atoi(e) != 0; }();
  const int seg_tiles = (prim == 0 && !mom && seg_on) ? min(w.n_tiles, kSegMaxTiles) : 0;
#define OCGS_FWD_LAUNCH(S, M, P, L)                                                                                                \
  do {                                                                                                                             \
    cudaLaunchConfig_t lc = {};                                                                                                    \
    lc.gridDim = dim3((unsigned)w.n_tiles); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = st;                     \
    cudaLaunchAttribute at[1];                                                                                                     \
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1;          \
    lc.attrs = at; lc.numAttrs = seg_tiles > 0 ? 1 : 0;  /* overlap with the segmented launch in front (see the kernel) */      \
    OCGS_CUDA_OK(cudaLaunchKernelEx(&lc, render_fwd_kernel<S, M, P, L>, (const uint32_t*)w.tile_order, w.tile_work, (const uint32_t*)w.ranges, \
                                    (const uint32_t*)w.tile_vals, (const float4*)w.rec, (const uint32_t*)w.rank_to_id, mask, cam.W, cam.H, cam.tiles_x, cfg, \
                                    color, alpha, depth, normal, n_contrib, w.final_T, w.blist, w.header, lp, vis_count, contrib_sum, mom, l1, seg_tiles)); \
  } while (0)
#define OCGS_FWD_LAUNCH_SEG(S, L)                                                                                                  \
  do {                                                                                                                             \
    cudaLaunchConfig_t lc = {};                                                                                                    \
    lc.gridDim = dim3((unsigned)(seg_tiles * kSegRanks)); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = st;       \
    cudaLaunchAttribute at[1];                                                                                                     \
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = kSegRanks; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1; \
    lc.attrs = at; lc.numAttrs = 1;                                                                                                \
    if (kSegRanks > 8) OCGS_CUDA_OK(cudaFuncSetAttribute(render_fwd_kernel<S, false, 0, L, true, 1>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1)); \
    OCGS_CUDA_OK(cudaLaunchKernelEx(&lc, render_fwd_kernel<S, false, 0, L, true, 1>, (const uint32_t*)w.tile_order, w.tile_work, (const uint32_t*)w.ranges, \
                                    (const uint32_t*)w.tile_vals, (const float4*)w.rec, (const uint32_t*)w.rank_to_id, mask, cam.W, cam.H, cam.tiles_x, cfg, \
                                    color, alpha, depth, normal, n_contrib, w.final_T, w.blist, w.header, lp, vis_count, contrib_sum, mom, l1, seg_tiles)); \
    OCGS_LAUNCHED(st, "render_fwd_seg_kernel");                                                                                    \
  } while (0)
  if (seg_tiles > 0) {
    if (target) { if (stats) OCGS_FWD_LAUNCH_SEG(true, true); else OCGS_FWD_LAUNCH_SEG(false, true); }
    else        { if (stats) OCGS_FWD_LAUNCH_SEG(true, false); else OCGS_FWD_LAUNCH_SEG(false, false); }
  }
#undef OCGS_FWD_LAUNCH_SEG
  if (prim == 1) {  // 3D Gaussians: forward + statistics only (no moment maps)
    if (mom || target) return OCGS_ERR_UNSUPPORTED;
    if (stats) OCGS_FWD_LAUNCH(true, false, 1, false); else OCGS_FWD_LAUNCH(false, false, 1, false);
  } else if (target) {  // fused masked L1 (no moment maps in this variant)
    if (mom || !gC) return OCGS_ERR_UNSUPPORTED;
    if (stats) OCGS_FWD_LAUNCH(true, false, 0, true); else OCGS_FWD_LAUNCH(false, false, 0, true);
  } else if (stats) { if (mom) OCGS_FWD_LAUNCH(true, true, 0, false); else OCGS_FWD_LAUNCH(true, false, 0, false); }
  else              { if (mom) OCGS_FWD_LAUNCH(false, true, 0, false); else OCGS_FWD_LAUNCH(false, false, 0, false); }
#undef OCGS_FWD_LAUNCH
  OCGS_LAUNCHED(st, "render_fwd_kernel");
  float* l1_out = target ? loss_l1 : nullptr;
  if (loss_bg || l1_out) {
    loss_final_kernel<<<1, 1024, 0, st>>>(w.loss_partial, w.n_tiles, (float)(1.0 / ((double)cam.W * (double)cam.H)), loss_bg,
                                          w.loss_partial + w.n_tiles, l1.inv_norm, l1_out);
    OCGS_LAUNCHED(st, "loss_final_kernel");
  }
  return OCGS_OK;
}

}  // namespace ocgs
