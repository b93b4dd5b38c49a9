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

// ---- stable LSD radix sort, onesweep style ------------------------------------------------------------------------
// One kernel reads the keys once and builds the global digit histograms of ALL passes; then each pass is ONE kernel:
// a block takes the next 4096-key tile (atomic ticket, so a tile only ever waits on tiles that are already running),
// ranks its keys, publishes its per-digit counts, finds its global offsets by decoupled look-back over the preceding
// tiles' status words (thread d owns digit d), reorders the tile by digit in shared memory and writes it out in runs.
// Status word = 2 flag bits | 30-bit count, so a plain 32-bit store/load carries flag and value together.
constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kFlagMask = 3u << 30, kValMask = (1u << 30) - 1u;
constexpr int kMaxPasses = 4;
#ifndef OCGS_SORT_LOOKBACK_WIDTH
#define OCGS_SORT_LOOKBACK_WIDTH 4
#endif
// Predecessors whose status words one step of the look-back loads at once (independent, coalesced loads): the look-back is a chain
// of dependent L2 round trips and a pass, one wave of blocks at these sizes, is as long as that chain
// (profiles/r02_config3_radix_passes_full.md); width 1 is the textbook walk.
constexpr int kLookbackWidth = OCGS_SORT_LOOKBACK_WIDTH;
constexpr int kHistItems = 4;  // keys per thread and unit of work of the histogram kernel (finer than a sort tile: more blocks in flight)
__global__ void __launch_bounds__(kSortThreads) radix_hist_all_kernel(const uint32_t* __restrict__ keys, const void* n_ptr, bool n_is_u64,
                                                                      size_t n_cap, int key_bits, int passes, uint32_t* __restrict__ ghist,
                                                                      uint32_t* __restrict__ status, size_t status_stride) {
  const unsigned long long n = min(load_count(n_ptr, n_is_u64), (unsigned long long)n_cap);
  const unsigned nblk = (unsigned)div_up((size_t)n, kSortTile);
  const unsigned nunit = (unsigned)div_up((size_t)n, (size_t)kHistItems * kSortThreads);
  if (blockIdx.x >= nunit) return;
  __shared__ uint32_t h[kMaxPasses][kRadix];
  for (int p = 0; p < passes; ++p) h[p][threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  for (unsigned tile = blockIdx.x; tile < nblk; tile += gridDim.x)  // look-back state of the sort tiles
    for (int p = 0; p < passes; ++p) status[(size_t)p * status_stride + (size_t)tile * kRadix + threadIdx.x] = 0;
  for (unsigned unit = blockIdx.x; unit < nunit; unit += gridDim.x) {
  const size_t base = (size_t)unit * kHistItems * kSortThreads;
#pragma unroll
  for (int r = 0; r < kHistItems; ++r) {
    const size_t i = base + (size_t)r * kSortThreads + threadIdx.x;
    const bool valid = i < n;
    const uint32_t k = valid ? keys[i] : 0u;
    for (int p = 0; p < passes; ++p) {
      const int shift = p * kRadixBits;
      const uint32_t mask = (1u << min(kRadixBits, key_bits - shift)) - 1u;
      const uint32_t dg = (k >> shift) & mask;
      // high digits are nearly constant across a warp (depth exponent, tile row): one add of 32 instead of 32 colliding adds
      const uint32_t d0 = __shfl_sync(0xFFFFFFFFu, dg, 0);
      if (__all_sync(0xFFFFFFFFu, valid && dg == d0)) {
        if (lane == 0) atomicAdd(&h[p][d0], 32u);
      } else if (valid) {
        atomicAdd(&h[p][dg], 1u);
      }
    }
  }
  }
  __syncthreads();
  for (int p = 0; p < passes; ++p) {
    const uint32_t c = h[p][threadIdx.x];
    if (c) atomicAdd(&ghist[p * kRadix + threadIdx.x], c);
  }
}

#ifndef OCGS_SORT_CTAS
#define OCGS_SORT_CTAS 3
#endif
constexpr int kSortCtas = OCGS_SORT_CTAS;  // resident blocks per SM the register budget is held to (80 registers; six passes at config 3: 200 us with 2, 178 with 3, 199 with 4;
                                           // with the 4-wide look-back: 161 us; 2048-key tiles (OCGS_SORT_ITEMS=8) 179 / 166 / 172 us with 3 / 4 / 6)
__global__ void __launch_bounds__(kSortThreads, kSortCtas) radix_onesweep_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                                                                      uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                                      const void* n_ptr, bool n_is_u64, size_t n_cap, int shift, uint32_t mask,
                                                                      const uint32_t* __restrict__ ghist, uint32_t* status,
                                                                      uint32_t* __restrict__ ticket) {
  const unsigned long long n = min(load_count(n_ptr, n_is_u64), (unsigned long long)n_cap);
  const unsigned nblk = (unsigned)div_up((size_t)n, kSortTile);
  constexpr int kWarps = kSortThreads / 32;
  __shared__ uint32_t cnt[kWarps][kRadix];
  __shared__ uint32_t s_gpos[kRadix];   // global position of smem slot 0 of each digit's run (may wrap below 0: used mod 2^32)
  __shared__ uint32_t s_keys[kSortTile];
  __shared__ uint32_t s_vals[kSortTile];
  __shared__ uint32_t s_warp[kWarps];
  __shared__ unsigned s_tile;
  __shared__ uint32_t s_wg[kWarps], s_wt[kWarps];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // persistent: the grid is a few blocks per SM, each takes tiles until the tickets run out (the key count lives on
  // the device, so a grid sized by the capacity would mostly launch blocks with nothing to do)
  while (true) {
  __syncthreads();  // previous tile fully written out before its shared state is reused
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
  for (int i = threadIdx.x; i < kWarps * kRadix; i += kSortThreads) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const unsigned tile = s_tile;
  if (tile >= nblk) return;
  // ---- rank: items are owned warp by warp in memory order (warp w: [w*512, w*512+512), round r, lane l) -----------
  const size_t base = (size_t)tile * kSortTile + (size_t)wid * (kSortItems * 32);
  uint32_t key[kSortItems], val[kSortItems];
  uint16_t rank[kSortItems];
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const size_t i = base + (size_t)r * 32 + lane;
    const bool valid = i < n;
    key[r] = valid ? keys_in[i] : 0xFFFFFFFFu;
    val[r] = valid ? vals_in[i] : 0u;
  }
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const bool valid = base + (size_t)r * 32 + lane < n;
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
  // ---- thread d: tile count of digit d, publish, exclusive prefixes over warps / digits / preceding tiles ---------
  const int d = threadIdx.x;  // kSortThreads == kRadix
  uint32_t total = 0;
#pragma unroll
  for (int w2 = 0; w2 < kWarps; ++w2) {
    const uint32_t t = cnt[w2][d];
    cnt[w2][d] = total;  // exclusive over warps
    total += t;
  }
  volatile uint32_t* st = status + (size_t)tile * kRadix + d;
  *st = (tile == 0 ? kFlagIncl : kFlagAgg) | total;
  // exclusive scan of ghist (global digit start) and of `total` (start of the digit's run inside the sorted tile)
  uint32_t gin = ghist[d], tin = total;
  uint32_t gsc = gin, tsc = tin;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t a = __shfl_up_sync(0xFFFFFFFFu, gsc, o), b2 = __shfl_up_sync(0xFFFFFFFFu, tsc, o);
    if (lane >= o) { gsc += a; tsc += b2; }
  }
  if (lane == 31) { s_wg[wid] = gsc; s_wt[wid] = tsc; }
  __syncthreads();
  uint32_t gpre = 0, tpre = 0;
#pragma unroll
  for (int w2 = 0; w2 < kWarps; ++w2)
    if (w2 < wid) { gpre += s_wg[w2]; tpre += s_wt[w2]; }
  const uint32_t gstart = gpre + gsc - gin, dstart = tpre + tsc - tin;
  // make cnt[w][d] the smem slot of warp w's first key of digit d
#pragma unroll
  for (int w2 = 0; w2 < kWarps; ++w2) cnt[w2][d] += dstart;
  __syncthreads();
  // ---- reorder the tile by digit in shared memory (local work, overlaps the predecessors' progress) ---------------
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    if (base + (size_t)r * 32 + lane < n) {
      const uint32_t dd = (key[r] >> shift) & mask;
      const uint32_t slot = cnt[wid][dd] + rank[r];
      s_keys[slot] = key[r];
      s_vals[slot] = val[r];
    }
  }
  // ---- decoupled look-back: keys of digit d in preceding tiles --------------------------------------------------
  uint32_t excl = 0;
  if (tile > 0) {
    int p = (int)tile - 1;  // the next predecessor to account for; tile 0 publishes inclusive, so the walk ends at or before it
    while (p >= 0) {
      uint32_t w[kLookbackWidth];
#pragma unroll
      for (int k = 0; k < kLookbackWidth; ++k)
        w[k] = p - k >= 0 ? *(volatile uint32_t*)(status + (size_t)(p - k) * kRadix + d) : (uint32_t)(2u << 30);  // before tile 0: kFlagIncl | 0
      bool stop = false;
#pragma unroll
      for (int k = 0; k < kLookbackWidth; ++k) {
        if (stop) continue;
        const uint32_t fl = w[k] & kFlagMask;
        if (fl == 0) { stop = true; continue; }  // not published yet (it is running: tickets are taken in order): load again from p
        excl += w[k] & kValMask;
        --p;
        if (fl == kFlagIncl) { p = -1; stop = true; }
      }
    }
    *st = kFlagIncl | (excl + total);
  }
  s_gpos[d] = gstart + excl - dstart;
  __syncthreads();
  // ---- coalesced write-out: slot i of the sorted tile goes to s_gpos[digit] + i ------------------------------------
  const unsigned in_tile = (unsigned)min((unsigned long long)kSortTile, n - (unsigned long long)tile * kSortTile);
#pragma unroll 4
  for (unsigned i = threadIdx.x; i < in_tile; i += kSortThreads) {
    const uint32_t k = s_keys[i];
    const uint32_t pos = s_gpos[(k >> shift) & mask] + i;
    keys_out[pos] = k;
    vals_out[pos] = s_vals[i];
  }
  }  // next ticket
}

// `prepared`: the producer of the keys has already built the digit histograms in `ghist` and cleared the look-back state
// (emit_keys_kernel does, for the tile sort); otherwise radix_hist_all_kernel reads the keys once to do both.
int radix_sort_pairs(uint32_t* keysA, uint32_t* valsA, uint32_t* keysB, uint32_t* valsB, const void* n_ptr, bool n_is_u64,
                     size_t n_max, int key_bits, uint32_t* status, uint32_t* ghist, bool* result_in_B, cudaStream_t st,
                     bool prepared) {
  static_assert(kSortThreads == kRadix, "one thread per digit");
  const int passes = (key_bits + kRadixBits - 1) / kRadixBits;
  const unsigned tiles_max = (unsigned)div_up(n_max, kSortTile);
  const unsigned grid = (unsigned)min(div_up(n_max, (size_t)kHistItems * kSortThreads), (size_t)sm_count() * 4);
  *result_in_B = (passes & 1) != 0;
  if (grid == 0 || passes == 0) { *result_in_B = false; return OCGS_OK; }
  if (passes > kMaxPasses || n_max > (size_t)kValMask) return OCGS_ERR_UNSUPPORTED;
  uint32_t* tickets = ghist + kMaxPasses * kRadix;
  const size_t stride = (size_t)tiles_max * kRadix;
  if (!prepared) {
    OCGS_CUDA_OK(cudaMemsetAsync(ghist, 0, (kMaxPasses * kRadix + kMaxPasses) * sizeof(uint32_t), st));
    radix_hist_all_kernel<<<grid, kSortThreads, 0, st>>>(keysA, n_ptr, n_is_u64, n_max, key_bits, passes, ghist, status, stride);
    OCGS_LAUNCHED(st, "radix_hist_all_kernel");
  }
  uint32_t *kin = keysA, *vin = valsA, *kout = keysB, *vout = valsB;
  for (int p = 0; p < passes; ++p) {
    const int shift = p * kRadixBits;
    const int bits = min(kRadixBits, key_bits - shift);
    const uint32_t mask = (1u << bits) - 1u;
    radix_onesweep_kernel<<<min(tiles_max, (unsigned)sm_count() * (unsigned)kSortCtas), kSortThreads, 0, st>>>(kin, vin, kout, vout, n_ptr, n_is_u64, n_max, shift, mask, ghist + p * kRadix,
                                                         status + (size_t)p * stride, tickets + p);
    OCGS_LAUNCHED(st, "radix_onesweep_kernel");
    uint32_t* t = kin; kin = kout; kout = t;
    t = vin; vin = vout; vout = t;
  }
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
  const int lane = threadIdx.x & 31;
  uint32_t t = 0, id = 0;
  if (r < n_vis) {
    id = rank_to_id[r];
    id_to_rank[id] = r;
    t = tiles[id];
    tcount[r] = t;
  }
  // the warp copies its 32 records (6 float4 each) together: lane l moves float4 l, l+32, ... of the 192, so the writes
  // are contiguous and each gathered record is read as one 96-byte run
  const unsigned r_warp = r - lane;
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const int f = i * 32 + lane, e = f / 6, part = f - 6 * e;
    const uint32_t src_id = __shfl_sync(0xFFFFFFFFu, id, e);
    if (r_warp + e < n_vis) {
      rec[(size_t)r_warp * 6 + f] = __ldg(rec_id + (size_t)src_id * 6 + part);
    }
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

// Offsets = exclusive scan of tiles-touched in rank order.  Every block sums the block sums in front of it itself (at most
// n_vis / 1024 values: one load per thread), so no separate scan of the block sums is launched; block 0 also totals all of
// them: K (64-bit), the capacity check and the closing entry offsets[n_vis].
__global__ void __launch_bounds__(kScanBlock) scan_apply_kernel(const uint32_t* __restrict__ tcount, const uint32_t* __restrict__ blocksum,
                                                                ocgs_header* __restrict__ header, size_t key_capacity,
                                                                uint32_t* __restrict__ offsets) {
  const unsigned n_vis = header->n_vis;
  const unsigned nb = (unsigned)div_up((size_t)n_vis, kScanBlock);
  if (blockIdx.x > 0 && blockIdx.x >= nb) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __shared__ unsigned long long wsum[32];
  __shared__ uint32_t ws[32];
  __shared__ unsigned long long s_pre;
  unsigned long long part = 0;
  const unsigned upto = blockIdx.x == 0 ? nb : blockIdx.x;  // block 0: the total; block b: the sums in front of it
  for (unsigned i = threadIdx.x; i < upto; i += kScanBlock) part += blocksum[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xFFFFFFFFu, part, o);
  if (lane == 0) wsum[wid] = part;
  __syncthreads();
  if (wid == 0) {
    unsigned long long w = wsum[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xFFFFFFFFu, w, o);
    if (lane == 0) s_pre = w;
  }
  __syncthreads();
  unsigned long long pre = s_pre;
  if (blockIdx.x == 0) {
    if (threadIdx.x == 0) {
      const unsigned long long K = pre;
      header->K = K;
      if (K > (unsigned long long)key_capacity || K > 0xFFFFFFF0ull) header->error |= 1u;
      offsets[n_vis] = (uint32_t)min(K, 0xFFFFFFFFull);
    }
    pre = 0;
    if (nb == 0) return;
  }
  const unsigned r = blockIdx.x * kScanBlock + threadIdx.x;
  const uint32_t v = r < n_vis ? tcount[r] : 0;
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
  if (r < n_vis) offsets[r] = (uint32_t)min(pre, 0xFFFFFFFFull) + (wid ? ws[wid - 1] : 0) + inc - v;
}

// ---- key emission: one thread per key, the owning surfel found by binary search in a shared slice of `offsets` -----
constexpr int kEmitThreads = 256;
constexpr int kEmitPerThread = 8;
constexpr int kEmitTile = kEmitThreads * kEmitPerThread;  // 2048 keys -> at most 2049 offsets entries

constexpr int kEmitBlocks = 6;  // resident blocks per SM = grid size / 148: one wave (1184 blocks of 40 registers ran as 1.33 waves: 42 us against 35)
__global__ void __launch_bounds__(kEmitThreads, kEmitBlocks) emit_keys_kernel(const ocgs_header* __restrict__ header, const uint32_t* __restrict__ offsets,
                                                                 const uint32_t* __restrict__ rank_to_id, const ushort4* __restrict__ rect,
                                                                 int tiles_x, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals,
                                                                 int passes, int key_bits, size_t key_capacity, uint32_t* __restrict__ ghist,
                                                                 uint32_t* __restrict__ status, size_t status_stride) {
  // look-back state of the sort tiles the tile sort will run over (also when the capacity overflowed: the passes still run)
  {
    const unsigned long long kc = min((unsigned long long)header->K, (unsigned long long)key_capacity);
    for (unsigned t = blockIdx.x; t < (unsigned)div_up((size_t)kc, kSortTile); t += gridDim.x)
      for (int p = 0; p < passes; ++p) status[(size_t)p * status_stride + (size_t)t * kRadix + threadIdx.x] = 0;
  }
  if (header->error) return;
  const unsigned K = (unsigned)header->K;
  const unsigned n_vis = header->n_vis;
  __shared__ uint32_t s_off[kEmitTile + 2];
  __shared__ unsigned s_r0, s_r1;
  // the tile sort's digit histograms (radix_sort_pairs, `prepared`) are built while the keys are still in registers
  __shared__ uint32_t s_h[2][kRadix];
  static_assert(kEmitThreads == kRadix, "one thread per digit");
  s_h[0][threadIdx.x] = 0; s_h[1][threadIdx.x] = 0;
  const uint32_t mask1 = passes > 1 ? (1u << min(kRadixBits, key_bits - kRadixBits)) - 1u : 0u;
  for (unsigned k0 = blockIdx.x * kEmitTile; k0 < K; k0 += gridDim.x * kEmitTile) {
  const unsigned k1 = min(k0 + kEmitTile, K);
  __syncthreads();  // previous tile's s_off fully consumed
  // r_lo = last rank with offsets[r] <= k0 (warp 0), r_hi = last rank with offsets[r] <= k1-1 (warp 1); offsets has
  // n_vis+1 strictly increasing entries with offsets[0] = 0 and offsets[n_vis] = K, searched 33-ary: 32 probes per round
  if (threadIdx.x < 64) {
    const int lane = threadIdx.x & 31;
    const unsigned key = (threadIdx.x < 32) ? k0 : k1 - 1;
    unsigned lo = 0, hi = n_vis;  // offsets[lo] <= key < offsets[hi]
    while (hi - lo > 1) {
      const unsigned step = (hi - lo + 32) / 33;
      const unsigned long long pos = (unsigned long long)lo + (unsigned long long)(lane + 1) * step;
      const bool le = pos < hi && offsets[pos] <= key;
      const int c = __popc(__ballot_sync(0xFFFFFFFFu, le));  // probes are increasing, so the true ones are lanes 0..c-1
      const unsigned nlo = lo + (unsigned)c * step;
      if (c < 32) hi = (unsigned)min((unsigned long long)hi, (unsigned long long)nlo + step);
      lo = nlo;
    }
    if (lane == 0) { if (threadIdx.x < 32) s_r0 = lo; else s_r1 = lo; }
  }
  __syncthreads();
  const unsigned r0 = s_r0, cnt = s_r1 - s_r0 + 1;  // surfels r0 .. r0+cnt-1 own the keys of this block (cnt <= kEmitTile)
  for (unsigned i = threadIdx.x; i <= cnt; i += kEmitThreads) s_off[i] = offsets[r0 + i];
  __syncthreads();
  // thread t emits the kEmitPerThread consecutive keys k0 + 8 t ..: one binary search for the first, then a walk along the
  // surfel's rect (x fastest) and on to the next surfels -- no search and no division for the other seven
  {
    const unsigned kk = k0 + threadIdx.x * kEmitPerThread;
    if (kk < k1) {
      unsigned lo = 0, hi = cnt;
      while (hi - lo > 1) { const unsigned mid = (lo + hi) >> 1; if (s_off[mid] <= kk) lo = mid; else hi = mid; }
      // (visible surfels touch >= 1 tile, so s_off is strictly increasing and every step below lands on a surfel with keys)
      unsigned r = r0 + lo, next_off = s_off[lo + 1];
      ushort4 rc = rect[rank_to_id[r]];
      unsigned tx0 = rc.x >> 4, wdt = (rc.z >> 4) + 1 - tx0;
      const unsigned local = kk - s_off[lo];
      unsigned ty = (rc.y >> 4) + local / wdt, tx = tx0 + local % wdt;
      uint32_t kbuf[kEmitPerThread], vbuf[kEmitPerThread];
      uint32_t run_digit = 0xFFFFFFFFu, run_len = 0;
      const int nk = (int)min((unsigned)kEmitPerThread, k1 - kk);
#pragma unroll
      for (int i = 0; i < kEmitPerThread; ++i) {
        if (i < nk) {
          if (kk + i >= next_off) {
            ++lo; r = r0 + lo; next_off = s_off[lo + 1];
            rc = rect[rank_to_id[r]];
            tx0 = rc.x >> 4; wdt = (rc.z >> 4) + 1 - tx0; tx = tx0; ty = rc.y >> 4;
          }
          const uint32_t key = ty * (unsigned)tiles_x + tx;
          kbuf[i] = key; vbuf[i] = r;
          if (++tx == tx0 + wdt) { tx = tx0; ++ty; }
          if (passes > 0) atomicAdd(&s_h[0][key & (kRadix - 1)], 1u);
          if (passes > 1) {  // the high digit (tile row) changes rarely along the walk: one add per run
            const uint32_t dg = (key >> kRadixBits) & mask1;
            if (dg != run_digit) {
              if (run_len) atomicAdd(&s_h[1][run_digit], run_len);
              run_digit = dg; run_len = 0;
            }
            ++run_len;
          }
        }
      }
      if (passes > 1 && run_len) atomicAdd(&s_h[1][run_digit], run_len);
      if (nk == kEmitPerThread) {  // k0 and 8 t are multiples of 8: 32-byte aligned
        uint4* kd = (uint4*)(keys + kk); uint4* vd = (uint4*)(vals + kk);
        kd[0] = make_uint4(kbuf[0], kbuf[1], kbuf[2], kbuf[3]); kd[1] = make_uint4(kbuf[4], kbuf[5], kbuf[6], kbuf[7]);
        vd[0] = make_uint4(vbuf[0], vbuf[1], vbuf[2], vbuf[3]); vd[1] = make_uint4(vbuf[4], vbuf[5], vbuf[6], vbuf[7]);
      } else {
#pragma unroll
        for (int i = 0; i < kEmitPerThread; ++i)
          if (i < nk) { keys[kk + i] = kbuf[i]; vals[kk + i] = vbuf[i]; }
      }
    }
  }
  }
  __syncthreads();
  for (int p = 0; p < min(passes, 2); ++p) {
    const uint32_t c = s_h[p][threadIdx.x];
    if (c) atomicAdd(&ghist[p * kRadix + threadIdx.x], c);
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
  // four consecutive keys per thread and iteration, one 16-byte load (+ the key before them): the kernel is a latency chain of
  // load -> compare, and a key per thread and iteration left it at 1.4 TB/s
  const size_t n4 = ((size_t)K + 3) / 4;
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < n4; i += stride) {
    const size_t k0 = 4 * i;
    uint32_t c[4];
    if (k0 + 3 < K) {
      const uint4 q = *reinterpret_cast<const uint4*>(keys + k0);
      c[0] = q.x; c[1] = q.y; c[2] = q.z; c[3] = q.w;
    } else {
#pragma unroll
      for (int e = 0; e < 4; ++e) c[e] = k0 + e < K ? keys[k0 + e] : 0u;
    }
    int prev = k0 == 0 ? -1 : (int)keys[k0 - 1];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const size_t k = k0 + e;
      if (k >= K) break;
      const int cur = (int)c[e];
      for (int t = prev + 1; t <= cur; ++t) {  // tiles in (prev, cur] start at k; the tile before each of them ends at k
        ranges[2 * t] = (uint32_t)k;
        if (t >= 1) ranges[2 * (t - 1) + 1] = (uint32_t)k;
      }
      if (k == K - 1) {
        for (int t = cur + 1; t < n_tiles; ++t) { ranges[2 * t] = K; ranges[2 * (t - 1) + 1] = K; }
        ranges[2 * (n_tiles - 1) + 1] = K;
      }
      prev = cur;
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
  scan_apply_kernel<<<nblk, kScanBlock, 0, st>>>(w.tcount, w.blocksum, w.header, w.key_capacity, w.offsets);
  OCGS_LAUNCHED(st, "scan_apply_kernel");
  const size_t cap = w.key_capacity;
  if (cap > 0 && n > 0) {
    int bits = 1;
    while ((1 << bits) < w.n_tiles) ++bits;
    const int passes = (bits + kRadixBits - 1) / kRadixBits;
    const bool fused_hist = passes <= 2;  // emit_keys_kernel keeps two histograms (n_tiles <= 65536)
    if (fused_hist) OCGS_CUDA_OK(cudaMemsetAsync(w.digit_total, 0, (kMaxPasses * kRadix + kMaxPasses) * sizeof(uint32_t), st));
    emit_keys_kernel<<<(unsigned)min(div_up(cap, kEmitTile), (size_t)sm_count() * kEmitBlocks), kEmitThreads, 0, st>>>(
        w.header, w.offsets, w.rank_to_id, w.rect, cam.tiles_x, w.tile_keys, w.tile_vals, fused_hist ? passes : 0, bits, cap, w.digit_total, w.hist,
        div_up(cap, kSortTile) * kRadix);
    OCGS_LAUNCHED(st, "emit_keys_kernel");
    bool inB = false;
    int rc = radix_sort_pairs(w.tile_keys, w.tile_vals, w.tkeyB, w.tvalB, &w.header->K, true, cap, bits, w.hist, w.digit_total, &inB, st, fused_hist);
    if (rc != OCGS_OK) return rc;
    if (inB) {  // odd number of passes: bring the result back to the documented sections
      const unsigned g = (unsigned)min(div_up(cap, 1024), (size_t)sm_count() * 8);
      copy_u32_kernel<<<g, 1024, 0, st>>>(w.tkeyB, w.tile_keys, w.header);
      copy_u32_kernel<<<g, 1024, 0, st>>>(w.tvalB, w.tile_vals, w.header);
      OCGS_LAUNCHED(st, "copy_u32_kernel");
    }
  }
  const unsigned rgrid = (unsigned)min(max(div_up(max(cap, (size_t)1), 1024), div_up((size_t)w.n_tiles, 256)), (size_t)sm_count() * 16);
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

// Blocks 1.. of the grid (backward pass only) clear the record-gradient accumulator, which is indexed by depth rank: only
// its first n_vis rows are ever touched.  One launch instead of two short dependent ones in front of render_bwd_kernel.
__global__ void __launch_bounds__(1024) order_tiles_kernel(const uint32_t* __restrict__ ranges, uint32_t* __restrict__ work, int n_tiles,
                                                           bool from_ranges, uint32_t* __restrict__ order,
                                                           const ocgs_header* __restrict__ header, float4* __restrict__ grad_rec) {
  if (blockIdx.x > 0) {
    const size_t n4 = (size_t)header->n_vis * (kRec / 4);
    for (size_t i = (size_t)(blockIdx.x - 1) * 1024 + threadIdx.x; i < n4; i += (size_t)(gridDim.x - 1) * 1024) grad_rec[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    return;
  }
  constexpr int kBuckets = 1024;
  __shared__ uint32_t s_cnt[kBuckets];
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_maxw;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  // the first kPer x 1024 tiles (all of them up to 1920x1080) stay in registers: their loads are issued together and the two later
  // passes do not read them again -- the kernel is ONE block on the step's critical path, twice per step, and a loop per pass was
  // 3 x 8 dependent L2 round trips
  constexpr int kPer = 8;
  uint32_t wreg[kPer];
  uint32_t mx = 0;
#pragma unroll
  for (int i = 0; i < kPer; ++i) {
    const int t = tid + i * 1024;
    wreg[i] = 0;
    if (t < n_tiles) wreg[i] = from_ranges ? ranges[2 * t + 1] - ranges[2 * t] : work[t];
  }
#pragma unroll
  for (int i = 0; i < kPer; ++i) {
    const int t = tid + i * 1024;
    if (from_ranges && t < n_tiles) work[t] = wreg[i];
    mx = max(mx, wreg[i]);
  }
  for (int t = tid + kPer * 1024; t < n_tiles; t += 1024) {
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
  // bucket 0 = heaviest; any monotone map of the work onto the buckets will do (a float scale instead of a 64-bit division)
  const float scale = (float)kBuckets / ((float)s_maxw + 1.0f);
#pragma unroll
  for (int i = 0; i < kPer; ++i) {
    if (tid + i * 1024 < n_tiles) {
      const uint32_t b = (kBuckets - 1) - min((uint32_t)(kBuckets - 1), (uint32_t)((float)wreg[i] * scale));
      atomicAdd(&s_cnt[b], 1u);
    }
  }
  for (int t = tid + kPer * 1024; t < n_tiles; t += 1024) {
    const uint32_t b = (kBuckets - 1) - min((uint32_t)(kBuckets - 1), (uint32_t)((float)work[t] * scale));
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
#pragma unroll
  for (int i = 0; i < kPer; ++i) {
    const int t = tid + i * 1024;
    if (t < n_tiles) {
      const uint32_t b = (kBuckets - 1) - min((uint32_t)(kBuckets - 1), (uint32_t)((float)wreg[i] * scale));
      order[atomicAdd(&s_cnt[b], 1u)] = (uint32_t)t;
    }
  }
  for (int t = tid + kPer * 1024; t < n_tiles; t += 1024) {
    const uint32_t b = (kBuckets - 1) - min((uint32_t)(kBuckets - 1), (uint32_t)((float)work[t] * scale));
    order[atomicAdd(&s_cnt[b], 1u)] = (uint32_t)t;
  }
}

int launch_order_tiles(const Workspace& w, bool from_ranges, cudaStream_t st, bool clear_grad_rec) {
  if (w.n_tiles == 0) return OCGS_OK;
  const unsigned clear_blocks = clear_grad_rec ? (unsigned)min(div_up((size_t)w.n * (kRec / 4), 1024), (size_t)sm_count() * 2) : 0u;
  order_tiles_kernel<<<1 + clear_blocks, 1024, 0, st>>>(w.ranges, w.tile_work, w.n_tiles, from_ranges, w.tile_order, w.header, (float4*)w.grad_rec);
  OCGS_LAUNCHED(st, "order_tiles_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
