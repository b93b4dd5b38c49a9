// prune.cu -- ocgs_prune_stats (O9): prune mask from the visibility statistics, exclusive scan, stable stream
// compaction of the five parameter arrays.  HBM-bound: 9 B read + 5 B written per surfel for mask/remap, then
// 232 B read and 232 B x kept-fraction written per surfel, element-parallel so reads and writes are coalesced.
#include "common.cuh"

namespace ocgs {

constexpr int kPruneBlock = 1024;

__global__ void __launch_bounds__(kPruneBlock) prune_flag_kernel(const uint32_t* __restrict__ vis_count, const float* __restrict__ contrib_sum,
                                                                 const float* __restrict__ opacity, int n, float tau, float min_opacity,
                                                                 uint8_t* __restrict__ prune_mask, uint32_t* __restrict__ blocksum) {
  const int j = blockIdx.x * kPruneBlock + threadIdx.x;
  uint32_t keep = 0;
  if (j < n) {
    // never blended in any render of the interval (occluded or out of frustum) -> removed
    const bool prune = (vis_count[j] == 0) || (contrib_sum[j] <= tau) || (opacity[j] < min_opacity);
    prune_mask[j] = prune ? 1 : 0;
    keep = prune ? 0u : 1u;
  }
  const unsigned bal = __ballot_sync(0xFFFFFFFFu, keep);
  __shared__ uint32_t ws[32];
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = (uint32_t)__popc(bal);
  __syncthreads();
  if (threadIdx.x < 32) {
    uint32_t s = ws[threadIdx.x];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(1024) prune_scan_kernel(uint32_t* __restrict__ blocksum, int nb, int* __restrict__ n_out) {
  __shared__ uint32_t warp_sums[32];
  __shared__ uint32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < nb ? blocksum[i] : 0;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
      uint32_t w = warp_sums[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, w, o);
        if (lane >= o) w += t;
      }
      warp_sums[lane] = w;
    }
    __syncthreads();
    const uint32_t c = carry;
    if (i < nb) blocksum[i] = c + (wid ? warp_sums[wid - 1] : 0) + inc - v;
    __syncthreads();
    if (threadIdx.x == 0) carry = c + warp_sums[31];
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_out = (int)carry;
}

__global__ void __launch_bounds__(kPruneBlock) prune_remap_kernel(const uint8_t* __restrict__ prune_mask, const uint32_t* __restrict__ blocksum,
                                                                  int n, int32_t* __restrict__ remap) {
  const int j = blockIdx.x * kPruneBlock + threadIdx.x;
  const bool keep = j < n && prune_mask[j] == 0;
  const unsigned bal = __ballot_sync(0xFFFFFFFFu, keep);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  __shared__ uint32_t ws[32];
  if (lane == 0) ws[wid] = (uint32_t)__popc(bal);
  __syncthreads();
  if (wid == 0) {
    const uint32_t v = ws[lane];
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
      if (lane >= o) inc += t;
    }
    ws[lane] = inc - v;
  }
  __syncthreads();
  if (j < n) remap[j] = keep ? (int32_t)(blocksum[blockIdx.x] + ws[wid] + (uint32_t)__popc(bal & ((1u << lane) - 1u))) : -1;
}

// element-parallel compaction: vector element i of surfel j = i / VPS is copied to out[remap[j] * VPS + i % VPS]
template <typename Vec, int VPS>
__global__ void __launch_bounds__(256) compact_kernel(const Vec* __restrict__ in, const int32_t* __restrict__ remap, size_t total,
                                                      Vec* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
    const size_t j = i / VPS;
    const int32_t r = __ldg(remap + j);
    if (r >= 0) out[(size_t)r * VPS + (i - j * VPS)] = in[i];
  }
}

template <typename Vec, int VPS>
static int launch_compact(const float* in, float* out, const int32_t* remap, int n, cudaStream_t st) {
  const size_t total = (size_t)n * VPS;
  if (total == 0) return OCGS_OK;
  const unsigned grid = (unsigned)min(div_up(total, 256), (size_t)sm_count() * 64);
  compact_kernel<Vec, VPS><<<grid, 256, 0, st>>>((const Vec*)in, remap, total, (Vec*)out);
  OCGS_LAUNCHED(st, "compact_kernel");
  return OCGS_OK;
}

// generic per-surfel rows (optimiser state, accumulated densification statistics, ...): row j of `row_floats` floats moves to row remap[j]
__global__ void __launch_bounds__(256) compact_rows_kernel(const float* __restrict__ in, const int32_t* __restrict__ remap, size_t total,
                                                           int row_floats, float* __restrict__ out) {
  for (size_t i = (size_t)blockIdx.x * 256 + threadIdx.x; i < total; i += (size_t)gridDim.x * 256) {
    const size_t j = i / (size_t)row_floats;
    const int32_t r = __ldg(remap + j);
    if (r >= 0) out[(size_t)r * row_floats + (i - j * row_floats)] = in[i];
  }
}

int launch_compact_rows(const float* in, const int32_t* remap, int n, int row_floats, float* out, cudaStream_t st) {
  const size_t total = (size_t)n * (size_t)row_floats;
  if (total == 0) return OCGS_OK;
  const unsigned grid = (unsigned)min(div_up(total, 256), (size_t)sm_count() * 64);
  compact_rows_kernel<<<grid, 256, 0, st>>>(in, remap, total, row_floats, out);
  OCGS_LAUNCHED(st, "compact_rows_kernel");
  return OCGS_OK;
}

int launch_prune(const ocgs_surfels& in, uint32_t* vis_count, float* contrib_sum, const ocgs_config& cfg, uint8_t* prune_mask,
                 int32_t* remap, const ocgs_surfels_mut* out, int* n_out, int reset_stats, void* ws, cudaStream_t st) {
  const int n = in.n;
  if (n == 0) {
    OCGS_CUDA_OK(cudaMemsetAsync(n_out, 0, sizeof(int), st));
    return OCGS_OK;
  }
  uint32_t* blocksum = (uint32_t*)ws;
  const int nb = (int)div_up((size_t)n, kPruneBlock);
  prune_flag_kernel<<<nb, kPruneBlock, 0, st>>>(vis_count, contrib_sum, in.opacity, n, cfg.tau_contrib, cfg.min_opacity, prune_mask, blocksum);
  OCGS_LAUNCHED(st, "prune_flag_kernel");
  prune_scan_kernel<<<1, 1024, 0, st>>>(blocksum, nb, n_out);
  OCGS_LAUNCHED(st, "prune_scan_kernel");
  prune_remap_kernel<<<nb, kPruneBlock, 0, st>>>(prune_mask, blocksum, n, remap);
  OCGS_LAUNCHED(st, "prune_remap_kernel");
  if (out) {
    int rc;
    if ((rc = launch_compact<float, 3>(in.pos, out->pos, remap, n, st)) != OCGS_OK) return rc;
    if ((rc = launch_compact<float2, 1>(in.scale, out->scale, remap, n, st)) != OCGS_OK) return rc;
    if ((rc = launch_compact<float4, 1>(in.quat, out->quat, remap, n, st)) != OCGS_OK) return rc;
    if ((rc = launch_compact<float, 1>(in.opacity, out->opacity, remap, n, st)) != OCGS_OK) return rc;
    if ((rc = launch_compact<float4, 12>(in.sh, out->sh, remap, n, st)) != OCGS_OK) return rc;
  }
  if (reset_stats) {
    OCGS_CUDA_OK(cudaMemsetAsync(vis_count, 0, (size_t)n * sizeof(uint32_t), st));
    OCGS_CUDA_OK(cudaMemsetAsync(contrib_sum, 0, (size_t)n * sizeof(float), st));
  }
  return OCGS_OK;
}

}  // namespace ocgs
