// sort.cu -- ocgs_bin_sort (O2/O3): depth-ordered tile binning.
//
// The order (tile id, centre-depth bits, surfel id) is produced by two stable LSD radix sorts instead of one sort of
// 64-bit (tile, depth) keys:
//   1. all N surfels by depth bits (32-bit keys; culled surfels carry 0xFFFFFFFF); the input is in id order and the
//      sort is stable, so ties keep ascending id.  Output: rank_to_id.
//   2. records are gathered into rank order, tiles-touched is scanned in rank order, keys (tile id, rank) are emitted
//      in rank order, and a stable sort by tile id alone (ceil(log2 n_tiles) bits) gives the per-tile lists.
// All counts (n_vis, K) stay on the device; grids are sized by capacities and blocks beyond the count exit.
#include "common.cuh"

namespace ocgs {

__device__ __forceinline__ unsigned long long load_count(const void* n_ptr, bool is_u64) {
  if (!n_ptr) return ~0ull;  // count known on the host: the capacity is the count
  return is_u64 ? *(const unsigned long long*)n_ptr : (unsigned long long)*(const unsigned int*)n_ptr;
}

// ---- radix pass, kernel 1: per-block digit histogram, stored digit-major: hist[d * nblk + b] ----------------------
__global__ void __launch_bounds__(kSortThreads) radix_hist_kernel(const uint32_t* __restrict__ keys, const void* n_ptr,
                                                                  bool n_is_u64, size_t n_cap, int shift, uint32_t mask,
                                                                  uint32_t* __restrict__ hist) {
  const unsigned long long n = min(load_count(n_ptr, n_is_u64), (unsigned long long)n_cap);
  const unsigned nblk = (unsigned)div_up((size_t)n, kSortTile);
  if (blockIdx.x >= nblk) return;
  __shared__ uint32_t h[kRadix];
  for (int i = threadIdx.x; i < kRadix; i += kSortThreads) h[i] = 0;
  __syncthreads();
  const size_t base = (size_t)blockIdx.x * kSortTile;
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const size_t i = base + (size_t)r * kSortThreads + threadIdx.x;
    const bool valid = i < n;
    const uint32_t d = valid ? ((keys[i] >> shift) & mask) : (0x100u + (threadIdx.x & 31));
    const unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
    if (valid && (threadIdx.x & 31) == (unsigned)(__ffs(peers) - 1)) atomicAdd(&h[d], (uint32_t)__popc(peers));
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kRadix; i += kSortThreads) hist[(size_t)i * nblk + blockIdx.x] = h[i];
}

// ---- kernel 2: block d scans row d of the histogram in place (exclusive) and writes the digit total --------------
__global__ void __launch_bounds__(1024) radix_rowscan_kernel(uint32_t* __restrict__ hist, const void* n_ptr, bool n_is_u64,
                                                             size_t n_cap, uint32_t* __restrict__ digit_total) {
  const unsigned long long n = min(load_count(n_ptr, n_is_u64), (unsigned long long)n_cap);
  const unsigned nblk = (unsigned)div_up((size_t)n, kSortTile);
  uint32_t* row = hist + (size_t)blockIdx.x * nblk;
  __shared__ uint32_t warp_sums[32];
  __shared__ uint32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (unsigned base = 0; base < nblk; base += 1024) {
    const unsigned i = base + threadIdx.x;
    const uint32_t v = i < nblk ? row[i] : 0;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      uint32_t ws = warp_sums[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, ws, o);
        if (lane >= o) ws += t;
      }
      warp_sums[lane] = ws;  // inclusive
    }
    __syncthreads();
    const uint32_t c = carry;
    const uint32_t wpre = wid ? warp_sums[wid - 1] : 0;
    if (i < nblk) row[i] = c + wpre + inc - v;
    __syncthreads();
    if (threadIdx.x == 0) carry = c + warp_sums[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) digit_total[blockIdx.x] = carry;
}

// ---- kernel 3: stable scatter --------------------------------------------------------------------------------------
// Items of a block are owned warp-by-warp (warp w: items [w*512, w*512+512), round r, lane l -> w*512 + r*32 + l), so
// the block-local rank of a key is (same digit in earlier warps) + (same digit in this warp, earlier rounds) +
// (same digit, lower lanes of this round): the order the keys had in memory.
__global__ void __launch_bounds__(kSortThreads) radix_scatter_kernel(const uint32_t* __restrict__ keys_in,
                                                                     const uint32_t* __restrict__ vals_in,
                                                                     uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                                     const void* n_ptr, bool n_is_u64, size_t n_cap, int shift,
                                                                     uint32_t mask, const uint32_t* __restrict__ hist,
                                                                     const uint32_t* __restrict__ digit_total) {
  const unsigned long long n = min(load_count(n_ptr, n_is_u64), (unsigned long long)n_cap);
  const unsigned nblk = (unsigned)div_up((size_t)n, kSortTile);
  if (blockIdx.x >= nblk) return;
  constexpr int kWarps = kSortThreads / 32;
  __shared__ uint32_t cnt[kWarps][kRadix];
  __shared__ uint32_t gbase[kRadix];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < kWarps * kRadix; i += kSortThreads) (&cnt[0][0])[i] = 0;
  // exclusive scan of the 256 digit totals (one warp, 8 per lane)
  if (wid == 0) {
    uint32_t loc[8], s = 0;
#pragma unroll
    for (int e = 0; e < 8; ++e) { loc[e] = digit_total[lane * 8 + e]; s += loc[e]; }
    uint32_t inc = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    uint32_t run = inc - s;
#pragma unroll
    for (int e = 0; e < 8; ++e) { gbase[lane * 8 + e] = run; run += loc[e]; }
  }
  __syncthreads();
  const size_t base = (size_t)blockIdx.x * kSortTile + (size_t)wid * (kSortItems * 32);
  uint32_t key[kSortItems], val[kSortItems];
  uint16_t rank[kSortItems];
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const size_t i = base + (size_t)r * 32 + lane;
    const bool valid = i < n;
    key[r] = valid ? keys_in[i] : 0xFFFFFFFFu;
    val[r] = valid ? vals_in[i] : 0u;
    const uint32_t d = valid ? ((key[r] >> shift) & mask) : (0x100u + lane);
    const unsigned peers = __match_any_sync(0xFFFFFFFFu, d);
    uint32_t pre = 0;
    if (valid) pre = cnt[wid][d];
    __syncwarp();
    if (valid && lane == (__ffs(peers) - 1)) cnt[wid][d] = pre + (uint32_t)__popc(peers);
    __syncwarp();
    rank[r] = (uint16_t)(pre + (uint32_t)__popc(peers & lt));
  }
  __syncthreads();
  // per digit: exclusive prefix over warps, plus this block's global base
  {
    const int d = threadIdx.x;  // kSortThreads == kRadix
    uint32_t run = gbase[d] + hist[(size_t)d * nblk + blockIdx.x];
#pragma unroll
    for (int w2 = 0; w2 < kWarps; ++w2) {
      const uint32_t t = cnt[w2][d];
      cnt[w2][d] = run;
      run += t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const size_t i = base + (size_t)r * 32 + lane;
    if (i < n) {
      const uint32_t d = (key[r] >> shift) & mask;
      const uint32_t p = cnt[wid][d] + rank[r];
      keys_out[p] = key[r];
      vals_out[p] = val[r];
    }
  }
}

int radix_sort_pairs(uint32_t* keysA, uint32_t* valsA, uint32_t* keysB, uint32_t* valsB, const void* n_ptr, bool n_is_u64,
                     size_t n_max, int key_bits, uint32_t* hist, uint32_t* digit_total, bool* result_in_B, cudaStream_t st) {
  static_assert(kSortThreads == kRadix, "scatter kernel maps one thread per digit");
  const int passes = (key_bits + kRadixBits - 1) / kRadixBits;
  const unsigned grid = (unsigned)div_up(n_max, kSortTile);
  uint32_t *kin = keysA, *vin = valsA, *kout = keysB, *vout = valsB;
  for (int p = 0; p < passes && grid > 0; ++p) {
    const int shift = p * kRadixBits;
    const int bits = min(kRadixBits, key_bits - shift);
    const uint32_t mask = (1u << bits) - 1u;
    radix_hist_kernel<<<grid, kSortThreads, 0, st>>>(kin, n_ptr, n_is_u64, n_max, shift, mask, hist);
    OCGS_LAUNCHED(st, "radix_hist_kernel");
    radix_rowscan_kernel<<<kRadix, 1024, 0, st>>>(hist, n_ptr, n_is_u64, n_max, digit_total);
    OCGS_LAUNCHED(st, "radix_rowscan_kernel");
    radix_scatter_kernel<<<grid, kSortThreads, 0, st>>>(kin, vin, kout, vout, n_ptr, n_is_u64, n_max, shift, mask, hist, digit_total);
    OCGS_LAUNCHED(st, "radix_scatter_kernel");
    uint32_t* t = kin; kin = kout; kout = t;
    t = vin; vin = vout; vout = t;
  }
  *result_in_B = (passes & 1) != 0;
  return OCGS_OK;
}

// ---- gather records into rank order, tiles-touched by rank, block sums -----------------------------------------
constexpr int kScanBlock = 1024;

__global__ void __launch_bounds__(kScanBlock) reorder_kernel(const uint32_t* __restrict__ rank_to_id, const ocgs_header* __restrict__ header,
                                                             const uint32_t* __restrict__ tiles, const float4* __restrict__ rec_id,
                                                             uint32_t* __restrict__ id_to_rank, float4* __restrict__ rec,
                                                             uint32_t* __restrict__ tcount, uint32_t* __restrict__ blocksum) {
  const unsigned n_vis = header->n_vis;
  const unsigned r = blockIdx.x * kScanBlock + threadIdx.x;
  if (blockIdx.x * kScanBlock >= n_vis) return;
  uint32_t t = 0;
  if (r < n_vis) {
    const uint32_t id = rank_to_id[r];
    id_to_rank[id] = r;
    t = tiles[id];
    tcount[r] = t;
    const float4* src = rec_id + (size_t)id * 6;
    float4* dst = rec + (size_t)r * 6;
    const float4 a = src[0], b = src[1], c = src[2], d = src[3], e = src[4], f = src[5];
    dst[0] = a; dst[1] = b; dst[2] = c; dst[3] = d; dst[4] = e; dst[5] = f;
  }
  // block sum
  __shared__ uint32_t ws[32];
  uint32_t s = t;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x < 32) {
    s = ws[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = s;
  }
}

// single block: exclusive scan of the block sums (64-bit running total), K, capacity check
__global__ void __launch_bounds__(1024) scan_blocksums_kernel(uint32_t* __restrict__ blocksum, ocgs_header* __restrict__ header,
                                                              size_t key_capacity, uint32_t* __restrict__ offsets) {
  const unsigned n_vis = header->n_vis;
  const unsigned nb = (unsigned)div_up((size_t)n_vis, kScanBlock);
  __shared__ unsigned long long warp_sums[32];
  __shared__ unsigned long long carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (unsigned base = 0; base < nb; base += 1024) {
    const unsigned i = base + threadIdx.x;
    const unsigned long long v = i < nb ? blocksum[i] : 0;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      unsigned long long w = warp_sums[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xFFFFFFFFu, w, o);
        if (lane >= o) w += t;
      }
      warp_sums[lane] = w;
    }
    __syncthreads();
    const unsigned long long c = carry;
    const unsigned long long ex = c + (wid ? warp_sums[wid - 1] : 0) + inc - v;
    if (i < nb) blocksum[i] = (uint32_t)min(ex, 0xFFFFFFFFull);
    __syncthreads();
    if (threadIdx.x == 0) carry = c + warp_sums[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const unsigned long long K = carry;
    header->K = K;
    if (K > (unsigned long long)key_capacity || K > 0xFFFFFFF0ull) header->error |= 1u;
    offsets[n_vis] = (uint32_t)min(K, 0xFFFFFFFFull);
  }
}

__global__ void __launch_bounds__(kScanBlock) scan_apply_kernel(const uint32_t* __restrict__ tcount, const uint32_t* __restrict__ blocksum,
                                                                const ocgs_header* __restrict__ header, uint32_t* __restrict__ offsets) {
  const unsigned n_vis = header->n_vis;
  if (blockIdx.x * kScanBlock >= n_vis) return;
  const unsigned r = blockIdx.x * kScanBlock + threadIdx.x;
  const uint32_t v = r < n_vis ? tcount[r] : 0;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __shared__ uint32_t ws[32];
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) ws[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = ws[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, w, o);
      if (lane >= o) w += t;
    }
    ws[lane] = w;
  }
  __syncthreads();
  if (r < n_vis) offsets[r] = blocksum[blockIdx.x] + (wid ? ws[wid - 1] : 0) + inc - v;
}

// ---- key emission: one thread per key, the owning surfel found by binary search in a shared slice of `offsets` -----
constexpr int kEmitThreads = 256;
constexpr int kEmitPerThread = 8;
constexpr int kEmitTile = kEmitThreads * kEmitPerThread;  // 2048 keys -> at most 2049 offsets entries

__global__ void __launch_bounds__(kEmitThreads) emit_keys_kernel(const ocgs_header* __restrict__ header, const uint32_t* __restrict__ offsets,
                                                                 const uint32_t* __restrict__ rank_to_id, const ushort4* __restrict__ rect,
                                                                 int tiles_x, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals) {
  if (header->error) return;
  const unsigned K = (unsigned)header->K;
  const unsigned n_vis = header->n_vis;
  const unsigned k0 = blockIdx.x * kEmitTile;
  if (k0 >= K) return;
  const unsigned k1 = min(k0 + kEmitTile, K);
  __shared__ uint32_t s_off[kEmitTile + 2];
  __shared__ unsigned s_r0, s_cnt;
  if (threadIdx.x == 0) {
    // r_lo = last rank with offsets[r] <= k0; r_hi = last rank with offsets[r] <= k1-1
    unsigned lo = 0, hi = n_vis;  // offsets has n_vis+1 entries, offsets[n_vis] = K > k0
    while (hi - lo > 1) { const unsigned mid = (lo + hi) >> 1; if (offsets[mid] <= k0) lo = mid; else hi = mid; }
    const unsigned r_lo = lo;
    lo = r_lo; hi = n_vis;
    while (hi - lo > 1) { const unsigned mid = (lo + hi) >> 1; if (offsets[mid] <= k1 - 1) lo = mid; else hi = mid; }
    s_r0 = r_lo;
    s_cnt = lo - r_lo + 1;
  }
  __syncthreads();
  const unsigned r0 = s_r0, cnt = s_cnt;  // surfels r0 .. r0+cnt-1 own the keys of this block (cnt <= kEmitTile)
  for (unsigned i = threadIdx.x; i <= cnt; i += kEmitThreads) s_off[i] = offsets[r0 + i];
  __syncthreads();
  for (unsigned k = k0 + threadIdx.x; k < k1; k += kEmitThreads) {
    unsigned lo = 0, hi = cnt;
    while (hi - lo > 1) { const unsigned mid = (lo + hi) >> 1; if (s_off[mid] <= k) lo = mid; else hi = mid; }
    // skip surfels with zero tiles cannot happen: visible surfels touch >= 1 tile, so s_off is strictly increasing
    const unsigned r = r0 + lo;
    const unsigned local = k - s_off[lo];
    const ushort4 rc = rect[rank_to_id[r]];
    const unsigned tx0 = rc.x >> 4, ty0 = rc.y >> 4, wdt = (rc.z >> 4) + 1 - tx0;
    const unsigned ty = ty0 + local / wdt, tx = tx0 + local % wdt;
    keys[k] = ty * (unsigned)tiles_x + tx;
    vals[k] = r;
  }
}

// ---- per-tile ranges from the sorted tile keys ----------------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_ranges_kernel(const ocgs_header* __restrict__ header, const uint32_t* __restrict__ keys,
                                                          int n_tiles, uint32_t* __restrict__ ranges) {
  const unsigned K = header->error ? 0u : (unsigned)header->K;
  const size_t stride = (size_t)gridDim.x * 256;
  if (K == 0) {
    for (size_t t = (size_t)blockIdx.x * 256 + threadIdx.x; t < (size_t)n_tiles; t += stride) { ranges[2 * t] = 0; ranges[2 * t + 1] = 0; }
    return;
  }
  for (size_t k = (size_t)blockIdx.x * 256 + threadIdx.x; k < K; k += stride) {
    const int cur = (int)keys[k];
    const int prev = k == 0 ? -1 : (int)keys[k - 1];
    for (int t = prev + 1; t <= cur; ++t) {  // tiles in (prev, cur] start at k; the tile before each of them ends at k
      ranges[2 * t] = (uint32_t)k;
      if (t >= 1) ranges[2 * (t - 1) + 1] = (uint32_t)k;
    }
    if (k == K - 1) {
      for (int t = cur + 1; t < n_tiles; ++t) { ranges[2 * t] = K; ranges[2 * (t - 1) + 1] = K; }
      ranges[2 * (n_tiles - 1) + 1] = K;
    }
  }
}

__global__ void __launch_bounds__(256) gather_ids_kernel(const ocgs_header* __restrict__ header, const uint32_t* __restrict__ vals,
                                                         const uint32_t* __restrict__ rank_to_id, uint32_t* __restrict__ out) {
  const unsigned K = header->error ? 0u : (unsigned)header->K;
  const size_t k = (size_t)blockIdx.x * 256 + threadIdx.x;
  if (k < K) out[k] = rank_to_id[vals[k]];
}

__global__ void copy_u32_kernel(const uint32_t* __restrict__ src, uint32_t* __restrict__ dst, const ocgs_header* __restrict__ header) {
  const unsigned K = header->error ? 0u : (unsigned)header->K;
  for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < K; k += (size_t)gridDim.x * blockDim.x) dst[k] = src[k];
}

int launch_bin_sort(const CamParams& cam, Workspace& w, uint32_t* sorted_ids, cudaStream_t st) {
  const int n = w.n;
  if (n > 0) {
    // stage 1: all surfels by depth bits (stable; 4 passes end in the A buffers = dkeyA / rank_to_id)
    bool inB = false;
    int rc = radix_sort_pairs(w.dkeyA, w.rank_to_id, w.dkeyB, w.dvalB, nullptr, false, (size_t)n, 32, w.hist,
                              w.digit_total, &inB, st);
    if (rc != OCGS_OK) return rc;
  }
  const unsigned nblk = (unsigned)div_up((size_t)max(n, 1), kScanBlock);
  if (n > 0) {
    reorder_kernel<<<nblk, kScanBlock, 0, st>>>(w.rank_to_id, w.header, w.tiles, (const float4*)w.rec_id, w.id_to_rank, (float4*)w.rec,
                                                w.tcount, w.blocksum);
    OCGS_LAUNCHED(st, "reorder_kernel");
  }
  scan_blocksums_kernel<<<1, 1024, 0, st>>>(w.blocksum, w.header, w.key_capacity, w.offsets);
  OCGS_LAUNCHED(st, "scan_blocksums_kernel");
  if (n > 0) {
    scan_apply_kernel<<<nblk, kScanBlock, 0, st>>>(w.tcount, w.blocksum, w.header, w.offsets);
    OCGS_LAUNCHED(st, "scan_apply_kernel");
  }
  const size_t cap = w.key_capacity;
  if (cap > 0 && n > 0) {
    emit_keys_kernel<<<(unsigned)div_up(cap, kEmitTile), kEmitThreads, 0, st>>>(w.header, w.offsets, w.rank_to_id, w.rect, cam.tiles_x,
                                                                                w.tile_keys, w.tile_vals);
    OCGS_LAUNCHED(st, "emit_keys_kernel");
    int bits = 1;
    while ((1 << bits) < w.n_tiles) ++bits;
    bool inB = false;
    int rc = radix_sort_pairs(w.tile_keys, w.tile_vals, w.tkeyB, w.tvalB, &w.header->K, true, cap, bits, w.hist, w.digit_total, &inB, st);
    if (rc != OCGS_OK) return rc;
    if (inB) {  // odd number of passes: bring the result back to the documented sections
      const unsigned g = (unsigned)min(div_up(cap, 1024), (size_t)148 * 8);
      copy_u32_kernel<<<g, 1024, 0, st>>>(w.tkeyB, w.tile_keys, w.header);
      copy_u32_kernel<<<g, 1024, 0, st>>>(w.tvalB, w.tile_vals, w.header);
      OCGS_LAUNCHED(st, "copy_u32_kernel");
    }
  }
  const unsigned rgrid = (unsigned)min(max(div_up(max(cap, (size_t)1), 256), div_up((size_t)w.n_tiles, 256)), (size_t)148 * 16);
  tile_ranges_kernel<<<rgrid, 256, 0, st>>>(w.header, w.tile_keys, w.n_tiles, w.ranges);
  OCGS_LAUNCHED(st, "tile_ranges_kernel");
  if (sorted_ids && cap > 0) {
    gather_ids_kernel<<<(unsigned)div_up(cap, 256), 256, 0, st>>>(w.header, w.tile_vals, w.rank_to_id, sorted_ids);
    OCGS_LAUNCHED(st, "gather_ids_kernel");
  }
  return OCGS_OK;
}

}  // namespace ocgs

// ---- launch order of the raster CTAs: heavy tiles first (longest-processing-time-first keeps the tail short) -----------
namespace ocgs {

__global__ void __launch_bounds__(1024) order_tiles_kernel(const uint32_t* __restrict__ ranges, uint32_t* __restrict__ work, int n_tiles,
                                                           bool from_ranges, uint32_t* __restrict__ order) {
  constexpr int kBuckets = 1024;
  __shared__ uint32_t s_cnt[kBuckets];
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_maxw;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  uint32_t mx = 0;
  for (int t = tid; t < n_tiles; t += 1024) {
    uint32_t wk = from_ranges ? ranges[2 * t + 1] - ranges[2 * t] : work[t];
    if (from_ranges) work[t] = wk;
    mx = max(mx, wk);
  }
  s_cnt[tid] = 0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = max(mx, __shfl_xor_sync(0xFFFFFFFFu, mx, o));
  if (lane == 0) s_warp[wid] = mx;
  __syncthreads();
  if (tid == 0) {
    uint32_t m = 0;
    for (int i = 0; i < 32; ++i) m = max(m, s_warp[i]);
    s_maxw = m;
  }
  __syncthreads();
  const unsigned long long maxw = (unsigned long long)s_maxw + 1ull;
  // bucket 0 = heaviest
  for (int t = tid; t < n_tiles; t += 1024) {
    const uint32_t b = (kBuckets - 1) - (uint32_t)(((unsigned long long)work[t] * kBuckets) / maxw);
    atomicAdd(&s_cnt[b], 1u);
  }
  __syncthreads();
  // exclusive scan of the 1024 bucket counts
  const uint32_t c = s_cnt[tid];
  uint32_t inc = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, inc, o);
    if (lane >= o) inc += x;
  }
  if (lane == 31) s_warp[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t x = s_warp[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, o);
      if (lane >= o) x += y;
    }
    s_warp[lane] = x;
  }
  __syncthreads();
  s_cnt[tid] = (wid ? s_warp[wid - 1] : 0) + inc - c;
  __syncthreads();
  for (int t = tid; t < n_tiles; t += 1024) {
    const uint32_t b = (kBuckets - 1) - (uint32_t)(((unsigned long long)work[t] * kBuckets) / maxw);
    order[atomicAdd(&s_cnt[b], 1u)] = (uint32_t)t;
  }
}

int launch_order_tiles(const Workspace& w, bool from_ranges, cudaStream_t st) {
  if (w.n_tiles == 0) return OCGS_OK;
  order_tiles_kernel<<<1, 1024, 0, st>>>(w.ranges, w.tile_work, w.n_tiles, from_ranges, w.tile_order);
  OCGS_LAUNCHED(st, "order_tiles_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
