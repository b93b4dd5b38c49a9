// raster_bwd.cu -- ocgs_render_bwd (O7).
//  (a) render_bwd_kernel: one CTA per tile, two pixels per thread, the tile's compact list of BLENDED entries (written by
//      the forward pass) walked BACK to FRONT; per pair the chain rule through compositing and the ray-splat intersection
//      gives 16 + 4 record gradients, reduced across the warp by a transposing butterfly (16 values, 8+4+2+1+1 shuffles),
//      stored per warp in shared memory, combined across the CTA and flushed with one global RED per (tile, entry, field).
//  (b) project_bwd_kernel: one thread per surfel, record gradients -> (pos, scale, quat, opacity, sh) gradients.
#include <cooperative_groups.h>
#include <stdlib.h>

#include "projection.cuh"

namespace ocgs {

constexpr int kBwdBatch = 64;
constexpr int kNG = G_COUNT;  // 20 accumulated fields per list entry

// sum of v[0..15] over the 32 lanes (16 shuffles); afterwards v[0] of lane L holds the total of value index
// 8*bit4(L) + 4*bit3(L) + 2*bit2(L) + bit1(L), i.e. index L >> 1
// kLast3Zero: v[13..15] are identically zero and their totals are not wanted (the colour / alpha-only backward instance): the
// first step then needs no selects for the pairs (5,13), (6,14), (7,15) -- the upper half-warp ends up with copies of the
// totals of 5..7 in the slots of 13..15, which the caller does not store.
template <bool kLast3Zero = false>
__device__ __forceinline__ void warp_transpose_reduce16(float* v, int lane) {
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const bool up = lane & 16;
    if (kLast3Zero && i >= 5) { v[i] += __shfl_xor_sync(0xFFFFFFFFu, v[i], 16); continue; }
    const float send = up ? v[i] : v[i + 8], keep = up ? v[i + 8] : v[i];
    v[i] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const bool up = lane & 8;
    const float send = up ? v[i] : v[i + 4], keep = up ? v[i + 4] : v[i];
    v[i] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 8);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const bool up = lane & 4;
    const float send = up ? v[i] : v[i + 2], keep = up ? v[i + 2] : v[i];
    v[i] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 4);
  }
  {
    const bool up = lane & 2;
    const float send = up ? v[0] : v[1], keep = up ? v[1] : v[0];
    v[0] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 2);
  }
  v[0] += __shfl_xor_sync(0xFFFFFFFFu, v[0], 1);
}

// sum of e[0..3] over the 32 lanes (6 shuffles); afterwards e[0] of lane L holds the total of value index 2*bit4(L) + bit3(L)
__device__ __forceinline__ void warp_transpose_reduce4(float* e, int lane) {
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const bool up = lane & 16;
    const float send = up ? e[i] : e[i + 2], keep = up ? e[i + 2] : e[i];
    e[i] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 16);
  }
  {
    const bool up = lane & 8;
    const float send = up ? e[0] : e[1], keep = up ? e[1] : e[0];
    e[0] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, 8);
  }
  e[0] += __shfl_xor_sync(0xFFFFFFFFu, e[0], 4);
  e[0] += __shfl_xor_sync(0xFFFFFFFFu, e[0], 2);
  e[0] += __shfl_xor_sync(0xFFFFFFFFu, e[0], 1);
}

// per-pixel state of the back-to-front walk
struct BwdPixel {
  float px, py;
  float T;                         // running transmittance T_i
  float GS;                        // sum_c g_c S_c - gA T_final: upstream gradients dotted with the suffix sums behind the pair
  float gc0, gc1, gc2, gd, gn0, gn1, gn2;
  float zc, gm1, gm2;              // kMoments: origin of the depth moments and the upstream gradients of m1, m2
  uint32_t last;                   // n_contrib (0 for pixels outside the image)
};

struct BwdConsts { float near_z, alpha_max, inv_sigma2; };

// One (pixel, entry) pair: recompute O4, and if the pair was blended add its 20 record-gradient terms into v / ex.
// With Q_c the accumulated maps, q_c this pair's values (rgb, z, n), S_c the suffix sums behind it (O7):
//   dL/dalpha_i = sum_c g_c (q_c T_i - S_c/(1-alpha_i)) + gA T_final/(1-alpha_i) = T_i (g.q) - (g.S - gA T_final)/(1-alpha_i),
// and g.S advances by w_i (g.q): one running scalar GS replaces the seven suffix sums.
// kGeo = false: no upstream gradient on the depth / normal / moment maps (gD, gN null: the masked-L1 + L_b step), so the
// terms they multiply are identically zero and are not evaluated.
template <bool kMoments, bool kGeo>
__device__ __forceinline__ bool bwd_pair(BwdPixel& s, uint32_t idx, const float4 r0, const float4 r1, const float4 r2, const float4 r3,
                                         const float4* __restrict__ sr, const BwdConsts& k, float* v, float* ex) {
  const float dx = s.px - r2.z, dy = s.py - r2.w;
  const float qx = fmaf(-dy, r0.w, fmaf(-dx, r0.x, r1.z));
  const float qy = fmaf(-dy, r1.x, fmaf(-dx, r0.y, r1.w));
  const float qz = fmaf(-dy, r1.y, fmaf(-dx, r0.z, r2.x));
  const float inv = rcp_approx(qz);
  const float u = qx * inv, vv = qy * inv;
  const float rho3 = fmaf(u, u, vv * vv);
  const float rho2 = fmaf(dx, dx, dy * dy) * k.inv_sigma2;
  const bool surf = rho3 <= rho2;
  const float rho = surf ? rho3 : rho2;
  const float z = surf ? r2.y * inv : r3.y;
  const bool contributes = idx < s.last && qz != 0.0f && !(z < k.near_z) && !(rho > r3.x);
  if (contributes) {
    const float4 r4 = sr[4], r5 = kGeo ? sr[5] : make_float4(0.f, 0.f, 0.f, 0.f);
    const float G = ex2_approx(rho * kNegHalfLog2e);
    const float araw = r4.x * G;
    const bool capped = araw > k.alpha_max;
    const float a = capped ? k.alpha_max : araw;
    const float inv1ma = rcp_approx(1.0f - a);
    s.T *= inv1ma;  // T_i = T_{i+1} / (1 - alpha_i)
    const float T = s.T, w = a * T;
    float gq = kGeo ? s.gd * z : 0.f;
    const float dz = z - s.zc;
    if (kMoments) gq = fmaf(s.gm2 * dz, dz, fmaf(s.gm1, dz, gq));  // m1, m2 behave like blended channels with values dz, dz^2
    gq = fmaf(s.gc0, r4.y, gq); gq = fmaf(s.gc1, r4.z, gq); gq = fmaf(s.gc2, r4.w, gq);
    if (kGeo) { gq = fmaf(s.gn0, r5.x, gq); gq = fmaf(s.gn1, r5.y, gq); gq = fmaf(s.gn2, r5.z, gq); }
    const float galpha = fmaf(T, gq, -s.GS * inv1ma);
    s.GS = fmaf(w, gq, s.GS);
    v[10] = fmaf(w, s.gc0, v[10]); v[11] = fmaf(w, s.gc1, v[11]); v[12] = fmaf(w, s.gc2, v[12]);
    if (kGeo) { v[13] = fmaf(w, s.gn0, v[13]); v[14] = fmaf(w, s.gn1, v[14]); v[15] = fmaf(w, s.gn2, v[15]); }
    float gz = kGeo ? w * s.gd : 0.f;
    if (kMoments) gz = fmaf(w, fmaf(2.0f * dz, s.gm2, s.gm1), gz);  // ... and depend on z directly (the origin is a constant)
    float grho = 0.f;
    if (!capped) { v[9] = fmaf(G, galpha, v[9]); grho = -0.5f * G * r4.x * galpha; }  // S12: zero through the cap
    if (surf) {
      // rho = u^2+v^2, z = D0/qz, (u,v) = (qx,qy)/qz, q = R - dx P - dy Q
      const float gu = 2.0f * u * grho, gv = 2.0f * vv * grho;
      const float gq0 = gu * inv, gq1 = gv * inv, gq2 = -(fmaf(gu, u, fmaf(gv, vv, kGeo ? gz * z : 0.f))) * inv;
      v[0] = fmaf(-dx, gq0, v[0]); v[1] = fmaf(-dx, gq1, v[1]); v[2] = fmaf(-dx, gq2, v[2]);
      v[3] = fmaf(-dy, gq0, v[3]); v[4] = fmaf(-dy, gq1, v[4]); v[5] = fmaf(-dy, gq2, v[5]);
      v[6] += gq0; v[7] += gq1; v[8] += gq2;
      if (kGeo) ex[0] = fmaf(gz, inv, ex[0]);
    } else {
      if (kGeo) ex[1] += gz;  // z = z_j
      ex[2] = fmaf(-2.0f * dx * k.inv_sigma2, grho, ex[2]);
      ex[3] = fmaf(-2.0f * dy * k.inv_sigma2, grho, ex[3]);
    }
  }
  return contributes;
}

// CTA = one 16x16 tile, 128 threads, TWO pixels per thread: warp w owns two vertically adjacent pixel blocks of the forward
// kernel (kSubW x kSubH each, common.cuh), lane l one pixel in each.  The two pixels' gradient terms are added in registers
// (free: the adds fold into FMAs) before the 32-lane transposing reduction, which is therefore paid once per 64 pixels
// (four pixels per thread in 64-thread CTAs measured slower: 1.21 vs 1.13 ms).  Each warp owns a slice of the batch
// accumulator and visits an entry at most once per batch, so its totals are plain stores (shared float atomics are CAS
// loops); the flush adds the slices of the warps whose forward hit bits are set.
constexpr int kBwdMinBlocks = 5;  // 4, 6, 7 measured slower
// A tile's blended list is walked by one CTA, each warp's part of it strictly in order: when lists are long and never
// saturate (config 5) the kernel's time is the chain of its heaviest tiles.  Tiles among the first kBwdSplitMax of the launch
// order whose blended list is longer than kBwdHeavyLen are therefore walked by TWO CTAs, one pixel per thread, each warp
// owning one forward block: a warp then visits only the entries its single block blended (about half as many).
constexpr int kBwdSplitMax = 512;
constexpr uint32_t kBwdHeavyLen = 2048;
#ifndef OCGS_BWD_LEAN_BLOCKS
#define OCGS_BWD_LEAN_BLOCKS 6
#endif
constexpr int kBwdLeanMinBlocks = OCGS_BWD_LEAN_BLOCKS;  // the colour / alpha-only instance (72 registers: 7 resident blocks)
// Segmented walk of heavy tiles (kSegB; the backward half of DESIGN.md "heavy tiles").  A tile whose BLENDED list is longer
// than kBwdSegLen is walked by a cluster of 8 CTAs = kBwdSegParts parts of the list x the two pixel halves of the split walk.
// The back-to-front chain needs, at the back of part r, the transmittance there and the running dot product g.S of everything
// behind it.  Both follow from one cheap pre-pass over the part (no gradient terms, no reduction): with the part's own
//   P_r = prod (1 - alpha_i),   G'_r = sum_i alpha_i T'_i (g.q_i),  T'_i = the product inside the part in front of pair i
// (Horner from the back: G' <- alpha (g.q) + (1 - alpha) G'), the true values are linear in the transmittance in front of the
// part, T_front,r = prod_{r' < r} P_r':   g.S at the back of part r = g.S_tail + sum_{r' > r} T_front,r' G'_r', T there = T_front,r+1.
// P and G' travel through distributed shared memory; then every CTA runs the ordinary walk of its part.
#ifndef OCGS_BWD_SEG_LEN
#define OCGS_BWD_SEG_LEN 3072
#endif
#ifndef OCGS_BWD_SEG_TILES
#define OCGS_BWD_SEG_TILES 128
#endif
constexpr int kBwdSegParts = 4;
constexpr uint32_t kBwdSegLen = OCGS_BWD_SEG_LEN;
constexpr int kBwdSegMaxTiles = OCGS_BWD_SEG_TILES;
namespace cg = cooperative_groups;

template <bool kMoments, bool kGeo, bool kSegB = false>
__global__ void __launch_bounds__(128, kGeo ? kBwdMinBlocks : kBwdLeanMinBlocks) render_bwd_kernel(const uint32_t* __restrict__ tile_order, const uint32_t* __restrict__ tile_work,
                                                            const uint32_t* __restrict__ ranges, const uint32_t* __restrict__ list,
                                                            const float4* __restrict__ rec, const uint2* __restrict__ blist, const uint8_t* __restrict__ mask,
                                                            const float* __restrict__ final_T, const uint32_t* __restrict__ n_contrib,
                                                            const float* __restrict__ gC, const float* __restrict__ gA,
                                                            const float* __restrict__ gD, const float* __restrict__ gN, const float* __restrict__ mom, const float* __restrict__ gM1, const float* __restrict__ gM2, int W, int H,
                                                            int tiles_x, int n_tiles, ocgs_config cfg, float gamma_over_hw, float* __restrict__ grad_rec,
                                                            int seg_tiles /*leading positions of the tile order the segmented launch takes (0: none)*/) {
  __shared__ float s_seg[kSegB ? 2 : 1][kSegB ? 128 : 1];  // kSegB: P_r and G'_r of this CTA's pixels, read by its cluster
  __shared__ float4 s_rec[kBwdBatch * 6];
  __shared__ uint32_t s_rank[kBwdBatch];
  __shared__ uint8_t s_mask[kBwdBatch];
  __shared__ uint32_t s_idx[kBwdBatch];   // position of the entry in the tile's full list (n_contrib counts those)
  __shared__ __align__(16) float s_acc[4][kBwdBatch * kNG];
  static_assert(kBwdBatch == 64, "the per-warp entry masks below cover two 32-entry halves");
  // launch order: heavy tiles first (tile_order); the first `n_split` positions own two consecutive blocks each, so that a
  // tile with a long blended list can be walked by two CTAs (see kBwdHeavyLen)
  // programmatic dependent launch, as in the forward pass: the ordinary launch overlaps the clusters and its last CTA joins them
  if (kSegB) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  struct PdlJoin {
    bool on;
    __device__ ~PdlJoin() { if (on) asm volatile("griddepcontrol.wait;" ::: "memory"); }
  } pdl_join{!kSegB && seg_tiles > 0 && blockIdx.x == gridDim.x - 1};
  const int n_split = min(n_tiles, kBwdSplitMax);
  const int crank = kSegB ? (int)cg::this_cluster().block_rank() : 0;  // kSegB: cluster rank = 2 * list part + pixel half
  const int pos = kSegB ? (int)blockIdx.x / (2 * kBwdSegParts) : ((int)blockIdx.x < 2 * n_split ? (int)(blockIdx.x >> 1) : (int)blockIdx.x - n_split);
  const int part = kSegB ? (crank & 1) : ((int)blockIdx.x < 2 * n_split ? (int)(blockIdx.x & 1u) : 0);
  const int lpart = crank >> 1;
  const int tile = (int)tile_order[pos];
  const uint32_t mx = tile_work[tile];           // length of the tile's blended list (written by the forward pass)
  const bool split = kSegB || (pos < n_split && mx > kBwdHeavyLen);
  if (kSegB ? mx <= kBwdSegLen : (pos < seg_tiles && mx > kBwdSegLen)) return;  // (uniform over the CTA / cluster)
  if (mx == 0 || (part && !split)) return;
  const int tx = tile % tiles_x, ty = tile / tiles_x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t start = ranges[2 * tile];
  // this warp's two forward blocks: vertically adjacent, block ids differ by the number of blocks per tile row; in a split
  // tile the warp owns ONE forward block (CTA `part` takes blocks 4 part .. 4 part + 3) and the second pixel is switched off
  constexpr int kBX = kTile / kSubW;  // forward blocks per tile row
  static_assert((kTile / kSubW) * (kTile / kSubH) == 8, "a split tile gives four of its eight forward blocks to each CTA");
  const int fb = split ? 4 * part + warp : 2 * (warp / kBX) * kBX + warp % kBX;  // the warp's (first) forward block
  const int bcol = fb % kBX, brow = fb / kBX;
  const uint32_t bit0 = 1u << fb, bit1 = split ? 0u : bit0 << kBX;
  const size_t HW = (size_t)W * H;
  BwdConsts kc = {cfg.near_z, cfg.alpha_max, 1.0f / cfg.filter_sigma2};
  float* acc = s_acc[warp];

  BwdPixel ps[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const int ix = tx * kTile + bcol * kSubW + lane % kSubW, iy = ty * kTile + (brow + q) * kSubH + lane / kSubW;
    BwdPixel& s = ps[q];
    s.px = (float)ix; s.py = (float)iy;
    s.last = 0;
    float Tfin = 1.0f, ga = 0.f;
    s.gc0 = s.gc1 = s.gc2 = s.gd = s.gn0 = s.gn1 = s.gn2 = s.zc = s.gm1 = s.gm2 = 0.f;
    if (ix < W && iy < H && !(split && q)) {
      const size_t p = (size_t)iy * W + ix;
      s.last = n_contrib[p];
      Tfin = final_T[p];
      if (gC) { s.gc0 = gC[p]; s.gc1 = gC[HW + p]; s.gc2 = gC[2 * HW + p]; }
      if (gA) ga = gA[p];
      if (kGeo && gD) s.gd = gD[p];
      if (kMoments) { s.zc = mom[p]; s.gm1 = gM1[p]; s.gm2 = gM2[p]; }
      if (kGeo && gN) { s.gn0 = gN[p]; s.gn1 = gN[HW + p]; s.gn2 = gN[2 * HW + p]; }
      if (mask && mask[p] == 0) ga += gamma_over_hw;  // d(gamma L_b)/dA = gamma (1-M)/(HW), Eq. 1 / Eq. 3
    }
    s.T = Tfin;
    // behind the last pair only the background term T_final bg_c is left (O5); dA/dalpha_i = T_final/(1-alpha_i)
    s.GS = Tfin * (fmaf(s.gc0, cfg.bg[0], fmaf(s.gc1, cfg.bg[1], s.gc2 * cfg.bg[2])) - ga);
  }
  const int nbatch = (int)((mx + kBwdBatch - 1) / kBwdBatch);
  // kSegB: this CTA's part of the list, in whole batches
  const int per = kSegB ? (nbatch + kBwdSegParts - 1) / kBwdSegParts : nbatch;
  const int b_lo = kSegB ? min(nbatch, lpart * per) : 0, b_hi = kSegB ? min(nbatch, b_lo + per) : nbatch;
  uint32_t lo0 = 0, lo1 = 0, hi0 = 0, hi1 = 0;
  // stage batch bi: its entries of the blended list, their records, and the warp's hit masks (two barriers inside, one in front)
  auto stage = [&](int bi) -> int {
    const uint32_t b0 = (uint32_t)bi * kBwdBatch;
    const int cnt = (int)min((uint32_t)kBwdBatch, mx - b0);
    __syncthreads();  // previous batch fully flushed before s_rank / s_mask / s_acc are reused
    if ((int)threadIdx.x < cnt) {
      const uint2 be = blist[start + b0 + threadIdx.x];
      s_rank[threadIdx.x] = be.x;
      s_mask[threadIdx.x] = (uint8_t)(be.y & 0xFFu);  // bit w: warp block w of the tile blended this entry in the forward pass
      s_idx[threadIdx.x] = be.y >> 8;
    }
    __syncthreads();
    constexpr int kParts = kGeo ? 6 : 5;  // the last 16 bytes of a record hold the normal: not read without dL/dnormal
    for (int i = threadIdx.x; i < cnt * kParts; i += 128) {
      const int e = i / kParts, part = i - kParts * e;
      s_rec[6 * e + part] = __ldg(rec + (size_t)s_rank[e] * 6 + part);
    }
    // per warp: which entries of the batch did its two pixel blocks blend (bit e of lo: entry e, of hi: entry 32 + e)
    const uint32_t mlo = lane < cnt ? s_mask[lane] : 0u, mhi = lane + 32 < cnt ? s_mask[lane + 32] : 0u;
    lo0 = __ballot_sync(0xFFFFFFFFu, mlo & bit0); lo1 = __ballot_sync(0xFFFFFFFFu, mlo & bit1);
    hi0 = __ballot_sync(0xFFFFFFFFu, mhi & bit0); hi1 = __ballot_sync(0xFFFFFFFFu, mhi & bit1);
    __syncthreads();
    return cnt;
  };
  if (kSegB) {
    // ---- pre-pass over this CTA's part (one pixel per thread: the split walk), back to front ----
    BwdPixel& s = ps[0];
    float P = 1.0f, Gp = 0.0f;
    for (int bi = b_hi - 1; bi >= b_lo; --bi) {
      stage(bi);
#pragma unroll 1
      for (int half = 1; half >= 0; --half) {
        uint32_t todo = half ? hi0 : lo0;
        while (todo) {
          const int jb = 31 - __clz(todo);
          todo &= ~(1u << jb);
          const int j = 32 * half + jb;
          const float4* sr = s_rec + 6 * j;
          const float4 r0 = sr[0], r1 = sr[1], r2 = sr[2], r3 = sr[3];
          const float dx = s.px - r2.z, dy = s.py - r2.w;
          const float qx = fmaf(-dy, r0.w, fmaf(-dx, r0.x, r1.z));
          const float qy = fmaf(-dy, r1.x, fmaf(-dx, r0.y, r1.w));
          const float qz = fmaf(-dy, r1.y, fmaf(-dx, r0.z, r2.x));
          const float inv = rcp_approx(qz);
          const float u = qx * inv, vv = qy * inv;
          const float rho3 = fmaf(u, u, vv * vv);
          const float rho2 = fmaf(dx, dx, dy * dy) * kc.inv_sigma2;
          const bool surf = rho3 <= rho2;
          const float rho = surf ? rho3 : rho2;
          const float z = surf ? r2.y * inv : r3.y;
          if (s_idx[j] < s.last && qz != 0.0f && !(z < kc.near_z) && !(rho > r3.x)) {
            const float4 r4 = sr[4], r5 = kGeo ? sr[5] : make_float4(0.f, 0.f, 0.f, 0.f);
            const float a = fminf(kc.alpha_max, r4.x * ex2_approx(rho * kNegHalfLog2e));
            float gq = kGeo ? s.gd * z : 0.f;
            const float dz = z - s.zc;
            if (kMoments) gq = fmaf(s.gm2 * dz, dz, fmaf(s.gm1, dz, gq));
            gq = fmaf(s.gc0, r4.y, gq); gq = fmaf(s.gc1, r4.z, gq); gq = fmaf(s.gc2, r4.w, gq);
            if (kGeo) { gq = fmaf(s.gn0, r5.x, gq); gq = fmaf(s.gn1, r5.y, gq); gq = fmaf(s.gn2, r5.z, gq); }
            Gp = fmaf(1.0f - a, Gp, a * gq);
            P *= 1.0f - a;
          }
        }
      }
    }
    __syncthreads();
    s_seg[0][threadIdx.x] = P; s_seg[1][threadIdx.x] = Gp;
    cg::cluster_group cl = cg::this_cluster();
    cl.sync();
    // T_front of every part, then this part's state at its back: T = T_front of the next part (the forward pass's exact T_final for
    // the last one), g.S = the tail term + the parts behind
    float Tf = 1.0f, Tback = s.T, GS = s.GS;
    for (int r = 0; r < kBwdSegParts; ++r) {
      const float* rp = cl.map_shared_rank(&s_seg[0][0], (unsigned)(2 * r + part));
      const float Pr = rp[threadIdx.x], Gr = rp[128 + threadIdx.x];
      if (r > lpart) GS = fmaf(Tf, Gr, GS);
      Tf *= Pr;
      if (r == lpart && lpart < kBwdSegParts - 1) Tback = Tf;
    }
    s.T = Tback; s.GS = GS;
    cl.sync();  // nobody leaves (or restages) while its shared memory may still be read
  }
  for (int bi = b_hi - 1; bi >= b_lo; --bi) {
    const int cnt = stage(bi);
#pragma unroll 1
    for (int half = 1; half >= 0; --half) {
      const uint32_t m0 = half ? hi0 : lo0, m1 = half ? hi1 : lo1;
      uint32_t todo = m0 | m1;
      while (todo) {
        const int jb = 31 - __clz(todo);  // back to front
        todo &= ~(1u << jb);
        const int j = 32 * half + jb;
        const float4* sr = s_rec + 6 * j;
        const uint32_t idx = s_idx[j];
        const float4 r0 = sr[0], r1 = sr[1], r2 = sr[2], r3 = sr[3];
        float v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = 0.f;
        float ex[4] = {0.f, 0.f, 0.f, 0.f};  // gD0, gzj, gcx, gcy
        if ((m0 >> jb) & 1u) bwd_pair<kMoments, kGeo>(ps[0], idx, r0, r1, r2, r3, sr, kc, v, ex);
        if ((m1 >> jb) & 1u) bwd_pair<kMoments, kGeo>(ps[1], idx, r0, r1, r2, r3, sr, kc, v, ex);
        float* dst = acc + j * kNG;
        warp_transpose_reduce16<!kGeo>(v, lane);
        if ((lane & 1) == 0 && (kGeo || lane < 26)) dst[lane >> 1] = v[0];  // !kGeo: fields 13..15 are zero and never read
        if (__any_sync(0xFFFFFFFFu, kGeo ? (ex[0] != 0.f) | (ex[1] != 0.f) | (ex[2] != 0.f) | (ex[3] != 0.f) : (ex[2] != 0.f) | (ex[3] != 0.f)))
          warp_transpose_reduce4(ex, lane);
        if ((lane & 7) == 0 && (kGeo || lane >= 16)) dst[16 + (lane >> 3)] = ex[0];  // without the reduction every lane's ex[0] is zero
      }
    }
    __syncthreads();
    // flush: one 16-byte vector RED per (tile, entry, group of four fields); !kGeo: fields 13..17 (normal, D0, z_j) are
    // identically zero and were never stored, so they are blanked here
    static_assert(kNG % 4 == 0, "fields are flushed in groups of four");
    constexpr int kNV = kNG / 4;
    for (int i = threadIdx.x; i < cnt * kNV; i += 128) {
      const int e = i / kNV, g4 = i - kNV * e;
      const uint32_t m = s_mask[e];
      float4 val = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int w2 = 0; w2 < 4; ++w2)
        if (m & (split ? 1u << (4 * part + w2) : ((1u << kBX) | 1u) << ((2 * (w2 / kBX)) * kBX + w2 % kBX))) {
          const float4 a = *reinterpret_cast<const float4*>(&s_acc[w2][e * kNG + 4 * g4]);
          val.x += a.x; val.y += a.y; val.z += a.z; val.w += a.w;
        }
      if (!kGeo) {
        if (g4 == 3) val.y = val.z = val.w = 0.f;
        if (g4 == 4) val.x = val.y = 0.f;
      }
      if (val.x != 0.f || val.y != 0.f || val.z != 0.f || val.w != 0.f)
        atomicAdd(reinterpret_cast<float4*>(grad_rec + (size_t)s_rank[e] * kRec + 4 * g4), val);
    }
  }
}

// the record-gradient accumulator is indexed by depth rank: only the first n_vis rows are ever touched
__global__ void __launch_bounds__(256) clear_grad_rec_kernel(const ocgs_header* __restrict__ header, float4* __restrict__ grad_rec) {
  const size_t n4 = (size_t)header->n_vis * 6;
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n4; i += (size_t)gridDim.x * 256) grad_rec[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

// ---- per-surfel: record gradients -> parameter gradients -------------------------------------------------------
__global__ void __launch_bounds__(128) project_bwd_kernel(const float* __restrict__ pos, const float2* __restrict__ scale,
                                                          const float4* __restrict__ quat, const float* __restrict__ opacity,
                                                          const float4* __restrict__ sh, int n, CamParams cam, ocgs_config cfg,
                                                          const ocgs_header* __restrict__ header, const uint32_t* __restrict__ id_to_rank,
                                                          const uint32_t* __restrict__ rank_to_id, const uint8_t* __restrict__ clamp_bits,
                                                          const float* __restrict__ grad_rec, float* __restrict__ d_pos,
                                                          float2* __restrict__ d_scale, float4* __restrict__ d_quat,
                                                          float* __restrict__ d_opacity, float4* __restrict__ d_sh,
                                                          float2* __restrict__ d_center2d) {
  // (1) by id: zero gradients of the surfels this view culled, written warp-cooperatively so that runs of culled
  //     surfels become full-line stores (71 % of the surfels at config 3)
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  {
    const int jw = t - lane;  // first id of this warp
    const bool culled = t < n && id_to_rank[t] == 0xFFFFFFFFu;
    const unsigned cm = __ballot_sync(0xFFFFFFFFu, culled);
    if (cm) {
      if (culled) {
        d_scale[t] = make_float2(0.f, 0.f);
        d_quat[t] = make_float4(0.f, 0.f, 0.f, 0.f);
        d_opacity[t] = 0.f;
        if (d_center2d) d_center2d[t] = make_float2(0.f, 0.f);
      }
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        const int f = i * 32 + lane;
        if ((cm >> (f / 3)) & 1u) d_pos[(size_t)jw * 3 + f] = 0.f;
      }
#pragma unroll
      for (int i = 0; i < 12; ++i) {
        const int f = i * 32 + lane;
        if ((cm >> (f / 12)) & 1u) d_sh[(size_t)jw * 12 + f] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
  }
  // (2) by id, compacted per block, so that the warps that do the arithmetic are full AND the parameter reads and gradient
  //     writes of a block stay inside its own window of ids, next to the zero rows written above (by depth rank, thread t =
  //     rank t, the same arithmetic took 103 us instead of 80: its scattered partial-sector writes cost more than the
  //     gathered 80-byte reads of grad_rec do now)
  __shared__ uint32_t s_list[128];
  __shared__ uint32_t s_wc[4];
  const bool vis = t < n && id_to_rank[t] != 0xFFFFFFFFu;
  const unsigned bv = __ballot_sync(0xFFFFFFFFu, vis);
  if (lane == 0) s_wc[threadIdx.x >> 5] = (uint32_t)__popc(bv);
  __syncthreads();
  uint32_t before = 0, total = 0;
#pragma unroll
  for (int w2 = 0; w2 < 4; ++w2) { const uint32_t c = s_wc[w2]; if (w2 < (int)(threadIdx.x >> 5)) before += c; total += c; }
  if (vis) s_list[before + (uint32_t)__popc(bv & ((1u << lane) - 1u))] = (uint32_t)t;
  __syncthreads();
  if (threadIdx.x >= total) return;
  const int j = (int)s_list[threadIdx.x];
  const uint32_t rank = id_to_rank[j];
  float4* dsh = d_sh + (size_t)j * 12;
  float g[kRec];
  const float4* gr = (const float4*)(grad_rec + (size_t)rank * kRec);
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const float4 t = gr[i];
    g[4 * i] = t.x; g[4 * i + 1] = t.y; g[4 * i + 2] = t.z; g[4 * i + 3] = t.w;
  }
  const float p[3] = {pos[3 * j], pos[3 * j + 1], pos[3 * j + 2]};
  const float2 s = scale[j];
  const float4 q = quat[j];
  Projected pr;
  project_surfel(p, s.x, s.y, q, opacity[j], cam, cfg, pr);
  const float* M = pr.M;
  const float M22 = M[8];
  // forward quantities of the record (common.cuh): A0, A1, R
  const float m2[3] = {M[6], M[7], M[8]};
  const float a0[3] = {fmaf(-pr.cx, m2[0], M[0]), fmaf(-pr.cx, m2[1], M[1]), fmaf(-pr.cx, m2[2], M[2])};
  const float a1[3] = {fmaf(-pr.cy, m2[0], M[3]), fmaf(-pr.cy, m2[1], M[4]), fmaf(-pr.cy, m2[2], M[5])};
  const float R[3] = {a0[1] * a1[2] - a0[2] * a1[1], a0[2] * a1[0] - a0[0] * a1[2], a0[0] * a1[1] - a0[1] * a1[0]};
  const float gP[3] = {g[G_PX], g[G_PY], g[G_PZ]}, gQ[3] = {g[G_QX], g[G_QY], g[G_QZ]};
  const float gD0 = g[G_D0];
  const float gR[3] = {g[G_RX] + gD0 * m2[0], g[G_RY] + gD0 * m2[1], g[G_RZ] + gD0 * m2[2]};  // D0 = M2 . R
  // c = a x b: ga = b x gc, gb = gc x a
  auto cross = [](const float* a, const float* b, float* o) {
    o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
  };
  float t1[3], t2[3], gA0[3], gA1[3], gM2c[3];
  cross(m2, gQ, t1); cross(a1, gR, t2);      // Q = A0 x M2, R = A0 x A1
  for (int i = 0; i < 3; ++i) gA0[i] = t1[i] + t2[i];
  cross(gP, m2, t1); cross(gR, a0, t2);      // P = M2 x A1
  for (int i = 0; i < 3; ++i) gA1[i] = t1[i] + t2[i];
  cross(a1, gP, t1); cross(gQ, a0, t2);      // dL/dM2 through P, Q and D0 (the -c*gA parts are folded in below)
  for (int i = 0; i < 3; ++i) gM2c[i] = t1[i] + t2[i] + gD0 * R[i];
  gM2c[2] += g[G_ZJ];                        // z_j = M22
  // A0 = M0 - cx M2, A1 = M1 - cy M2 (c constant: the intersection does not depend on it) and c2d = (M02, M12)/M22
  const float ex = pr.cx - cam.ox, ey = pr.cy - cam.oy;
  const float f0 = g[G_CX] / M22, f1 = g[G_CY] / M22;
  const float m0[3] = {gA0[0], gA0[1], gA0[2] + f0};  // dL/dM0
  const float m1[3] = {gA1[0], gA1[1], gA1[2] + f1};  // dL/dM1
  float gcol[3][3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    gcol[i][0] = cam.fx * m0[i];
    gcol[i][1] = cam.fy * m1[i];
    // ox m0 + oy m1 + dL/dM2 with dL/dM2 = gM2c - cx gA0 - cy gA1 (- (f0 cx + f1 cy) on i = 2), combined to avoid cancellation
    gcol[i][2] = gM2c[i] - ex * m0[i] - ey * m1[i];
  }
  if (d_center2d) d_center2d[j] = make_float2(M22 * m0[2], M22 * m1[2]);
  const float* V = cam.V;
  d_scale[j] = make_float2(gcol[0][0] * pr.vu[0] + gcol[0][1] * pr.vu[1] + gcol[0][2] * pr.vu[2],
                           gcol[1][0] * pr.vv[0] + gcol[1][1] * pr.vv[1] + gcol[1][2] * pr.vv[2]);
  float gtu[3], gtv[3], gtw[3], gp[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {  // R_wc^T g
    gtu[k] = s.x * (V[k] * gcol[0][0] + V[4 + k] * gcol[0][1] + V[8 + k] * gcol[0][2]);
    gtv[k] = s.y * (V[k] * gcol[1][0] + V[4 + k] * gcol[1][1] + V[8 + k] * gcol[1][2]);
    gp[k] = V[k] * gcol[2][0] + V[4 + k] * gcol[2][1] + V[8 + k] * gcol[2][2];
  }
  const float w = q.x, x = q.y, y = q.z, z = q.w;
  {
    const float tw0 = 2.0f * (x * z + w * y), tw1 = 2.0f * (y * z - w * x), tw2 = 1.0f - 2.0f * (x * x + y * y);
    const float nx = V[0] * tw0 + V[1] * tw1 + V[2] * tw2, ny = V[4] * tw0 + V[5] * tw1 + V[6] * tw2,
                nz = V[8] * tw0 + V[9] * tw1 + V[10] * tw2;
    const float sgn = (nx * pr.pc[0] + ny * pr.pc[1] + nz * pr.pc[2] > 0.0f) ? -1.0f : 1.0f;
#pragma unroll
    for (int k = 0; k < 3; ++k) gtw[k] = sgn * (V[k] * g[G_NX] + V[4 + k] * g[G_NY] + V[8 + k] * g[G_NZ]);
  }
  d_quat[j] = make_float4(
      2.0f * (z * gtu[1] - y * gtu[2] - z * gtv[0] + x * gtv[2] + y * gtw[0] - x * gtw[1]),
      2.0f * (y * gtu[1] + z * gtu[2] + y * gtv[0] - 2.0f * x * gtv[1] + w * gtv[2] + z * gtw[0] - w * gtw[1] - 2.0f * x * gtw[2]),
      2.0f * (-2.0f * y * gtu[0] + x * gtu[1] - w * gtu[2] + x * gtv[0] + z * gtv[2] + w * gtw[0] + z * gtw[1] - 2.0f * y * gtw[2]),
      2.0f * (-2.0f * z * gtu[0] + w * gtu[1] + x * gtu[2] - w * gtv[0] - 2.0f * z * gtv[1] + y * gtv[2] + x * gtw[0] + y * gtw[1]));
  d_opacity[j] = g[G_OPA];
  // colour
  float dx = p[0] - cam.campos[0], dy = p[1] - cam.campos[1], dz = p[2] - cam.campos[2];
  const float inv = rsqrtf(dx * dx + dy * dy + dz * dz);
  dx *= inv; dy *= inv; dz *= inv;
  float Y[16];
  sh_basis(dx, dy, dz, cfg.sh_degree, Y);
  const int nb = (cfg.sh_degree + 1) * (cfg.sh_degree + 1);
  const uint8_t cl = clamp_bits[j];
  const float gcolr[3] = {(cl & 1) ? 0.f : g[G_COLR], (cl & 2) ? 0.f : g[G_COLG], (cl & 4) ? 0.f : g[G_COLB]};
  float a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = 0.f;
  const float4* shj = sh + (size_t)j * 12;
  // the surfel's SH row in two batches of six 16-byte loads, each batch in flight together (as in sh_colour_rn)
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    float4 fb[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) fb[i] = 4 * (6 * h + i) < 3 * nb ? __ldg(shj + 6 * h + i) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const int v4 = 6 * h + i;
      const float ff[4] = {fb[i].x, fb[i].y, fb[i].z, fb[i].w};
      float oo[4];
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int idx = 4 * v4 + e, k = idx / 3, c = idx - 3 * k;
        oo[e] = 0.f;
        if (idx < 3 * nb) {
          oo[e] = Y[k] * gcolr[c];
          a[k] = fmaf(ff[e], gcolr[c], a[k]);
        }
      }
      dsh[v4] = make_float4(oo[0], oo[1], oo[2], oo[3]);
    }
  }
  float gdir[3];
  sh_basis_grad(dx, dy, dz, cfg.sh_degree, a, gdir);
  const float dd = dx * gdir[0] + dy * gdir[1] + dz * gdir[2];
  gp[0] += (gdir[0] - dx * dd) * inv; gp[1] += (gdir[1] - dy * dd) * inv; gp[2] += (gdir[2] - dz * dd) * inv;
  d_pos[3 * j] = gp[0]; d_pos[3 * j + 1] = gp[1]; d_pos[3 * j + 2] = gp[2];
}

int launch_render_bwd(const ocgs_surfels& s, const CamParams& cam, const ocgs_config& cfg, Workspace& w, const uint8_t* mask,
                      const float* final_T, const uint32_t* n_contrib, const float* gC, const float* gA, const float* gD,
                      const float* gN, const float* mom, const float* gM1, const float* gM2, float* d_pos, float* d_scale, float* d_quat, float* d_opacity, float* d_sh,
                      float* d_center2d, cudaStream_t st) {
  if (s.n == 0) return OCGS_OK;
  if (w.n_tiles == 0) {
    clear_grad_rec_kernel<<<(unsigned)min(div_up((size_t)s.n * 6, 256), (size_t)sm_count() * 16), 256, 0, st>>>(w.header, (float4*)w.grad_rec);
    OCGS_LAUNCHED(st, "clear_grad_rec_kernel");
  } else {
    // tile_work = length of each tile's blended list, from the forward pass; the same launch clears grad_rec
    int rc = launch_order_tiles(w, /*from_ranges=*/false, st, /*clear_grad_rec=*/true);
    if (rc != OCGS_OK) return rc;
    const float goh = mask ? (float)((double)cfg.gamma_bg / ((double)cam.W * (double)cam.H)) : 0.f;
    static const bool seg_on = [] { const char* e = getenv("OCGS_BWD_SEGMENTED"); return !e || atoi(e) != 0; }();
    const int seg_tiles = seg_on ? min(w.n_tiles, kBwdSegMaxTiles) : 0;
    const float* momp = (mom && gM1 && gM2) ? mom : nullptr;
    const bool geo = momp || gD || gN;  // colour / alpha gradients only (masked L1 + L_b): the depth and normal terms are identically zero
#define OCGS_BWD_LAUNCH(M, G, SEG)                                                                                                 \
  do {                                                                                                                             \
    cudaLaunchConfig_t lc = {};                                                                                                    \
    lc.gridDim = dim3(SEG ? (unsigned)(seg_tiles * 2 * kBwdSegParts) : (unsigned)(w.n_tiles + min(w.n_tiles, kBwdSplitMax)));      \
    lc.blockDim = dim3(128); lc.dynamicSmemBytes = 0; lc.stream = st;                                                              \
    cudaLaunchAttribute at[1];                                                                                                     \
    if (SEG) { at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = 2 * kBwdSegParts; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1; } \
    else { at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[0].val.programmaticStreamSerializationAllowed = 1; }  \
    lc.attrs = at; lc.numAttrs = (SEG || seg_tiles > 0) ? 1 : 0;                                                                   \
    OCGS_CUDA_OK(cudaLaunchKernelEx(&lc, render_bwd_kernel<M, G, SEG>, (const uint32_t*)w.tile_order, (const uint32_t*)w.tile_work, (const uint32_t*)w.ranges, \
                                    (const uint32_t*)w.tile_vals, (const float4*)w.rec, (const uint2*)w.blist, mask, final_T, n_contrib, gC, gA, \
                                    geo ? gD : (const float*)nullptr, geo ? gN : (const float*)nullptr, momp, momp ? gM1 : (const float*)nullptr, \
                                    momp ? gM2 : (const float*)nullptr, cam.W, cam.H, cam.tiles_x, w.n_tiles, cfg, goh, w.grad_rec, seg_tiles)); \
  } while (0)
    for (int seg = seg_tiles > 0 ? 1 : 0; seg >= 0; --seg) {  // the clusters first, then the ordinary launch
      if (momp) { if (seg) OCGS_BWD_LAUNCH(true, true, true); else OCGS_BWD_LAUNCH(true, true, false); }
      else if (geo) { if (seg) OCGS_BWD_LAUNCH(false, true, true); else OCGS_BWD_LAUNCH(false, true, false); }
      else { if (seg) OCGS_BWD_LAUNCH(false, false, true); else OCGS_BWD_LAUNCH(false, false, false); }
      if (seg) OCGS_LAUNCHED(st, "render_bwd_seg_kernel");
    }
#undef OCGS_BWD_LAUNCH
    OCGS_LAUNCHED(st, "render_bwd_kernel");
  }
  project_bwd_kernel<<<(unsigned)div_up((size_t)s.n, 128), 128, 0, st>>>(s.pos, (const float2*)s.scale, (const float4*)s.quat, s.opacity,
                                                                        (const float4*)s.sh, s.n, cam, cfg, w.header, w.id_to_rank, w.rank_to_id, w.clamp,
                                                                        w.grad_rec, d_pos, (float2*)d_scale, (float4*)d_quat, d_opacity,
                                                                        (float4*)d_sh, (float2*)d_center2d);
  OCGS_LAUNCHED(st, "project_bwd_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
