// densify.cu -- clone / split half of the adaptive density control (DESIGN.md
// reading R-densify).
//   ocgs_densify_accumulate: grad_accum[j] += |(W/2, H/2) * d_center2d_j| (the gradient w.r.t. the projected centre in NDC units,
//                            the unit the default threshold 2e-4 of the cited work is calibrated in), denom[j] += 1 for the
//                            surfels that passed this view's frustum test (id_to_rank of the workspace).
//   ocgs_densify:            class per surfel (keep / clone / split) from avg = grad_accum / denom in fp32, three exclusive
//                            scans, stable scatter: non-split surfels, then clones, then two children per split surfel
//                            (p + s_u xi0 t_u + s_v xi1 t_v, scales / 1.6); src[row] = source id; counts on the device.
// HBM-bound copies: 232 B read and ~232 B written per surfel.
#include "common.cuh"

namespace ocgs {

constexpr int kDenBlock = 256;

__global__ void __launch_bounds__(256) densify_accumulate_kernel(const uint32_t* __restrict__ id_to_rank, const float2* __restrict__ d_center2d,
                                                                 int n, float half_w, float half_h, float* __restrict__ grad_accum, uint32_t* __restrict__ denom) {
  const int j = blockIdx.x * 256 + threadIdx.x;
  if (j >= n || id_to_rank[j] == 0xFFFFFFFFu) return;
  const float2 g = d_center2d[j];
  const float gx = half_w * g.x, gy = half_h * g.y;  // pixel = ((ndc + 1) W - 1) / 2: d/d ndc = (W/2) d/d pixel
  grad_accum[j] += sqrtf(fmaf(gx, gx, gy * gy));
  denom[j] += 1u;
}

__device__ __forceinline__ int densify_class(float ga, uint32_t dn, float2 s, float grad_threshold, float scale_threshold) {
  const float avg = dn > 0 ? __fdiv_rn(ga, (float)dn) : 0.0f;
  if (!(avg >= grad_threshold)) return 0;
  return fmaxf(s.x, s.y) > scale_threshold ? 2 : 1;
}

// per block: number of non-split, cloned, split surfels
__global__ void __launch_bounds__(kDenBlock) densify_flag_kernel(const float* __restrict__ grad_accum, const uint32_t* __restrict__ denom,
                                                                 const float2* __restrict__ scale, int n, float grad_threshold,
                                                                 float scale_threshold, uint8_t* __restrict__ cls, uint32_t* __restrict__ blocksum) {
  const int j = blockIdx.x * kDenBlock + threadIdx.x;
  int c = -1;
  if (j < n) {
    c = densify_class(grad_accum[j], denom[j], scale[j], grad_threshold, scale_threshold);
    cls[j] = (uint8_t)c;
  }
  __shared__ uint32_t s_cnt[3];
  if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const unsigned b_keep = __ballot_sync(0xFFFFFFFFu, c == 0 || c == 1), b_clone = __ballot_sync(0xFFFFFFFFu, c == 1),
                 b_split = __ballot_sync(0xFFFFFFFFu, c == 2);
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&s_cnt[0], (uint32_t)__popc(b_keep)); atomicAdd(&s_cnt[1], (uint32_t)__popc(b_clone)); atomicAdd(&s_cnt[2], (uint32_t)__popc(b_split));
  }
  __syncthreads();
  if (threadIdx.x < 3) blocksum[3 * blockIdx.x + threadIdx.x] = s_cnt[threadIdx.x];
}

// one block: exclusive scans of the three block-count sequences; counts[0..3] = n_out, n_keep, n_clone, n_split
__global__ void __launch_bounds__(1024) densify_scan_kernel(uint32_t* __restrict__ blocksum, int nb, int* __restrict__ counts) {
  __shared__ uint32_t warp_sums[3][32];
  __shared__ uint32_t carry[3];
  if (threadIdx.x < 3) carry[threadIdx.x] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int i = base + threadIdx.x;
    uint32_t v[3], inc[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      v[c] = i < nb ? blocksum[3 * i + c] : 0;
      inc[c] = v[c];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc[c], o);
        if (lane >= o) inc[c] += t;
      }
      if (lane == 31) warp_sums[c][wid] = inc[c];
    }
    __syncthreads();
    if (wid < 3) {
      uint32_t w = warp_sums[wid][lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, w, o);
        if (lane >= o) w += t;
      }
      warp_sums[wid][lane] = w;
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 3; ++c)
      if (i < nb) blocksum[3 * i + c] = carry[c] + (wid ? warp_sums[c][wid - 1] : 0) + inc[c] - v[c];
    __syncthreads();
    if (threadIdx.x < 3) carry[threadIdx.x] += warp_sums[threadIdx.x][31];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    counts[1] = (int)carry[0]; counts[2] = (int)carry[1]; counts[3] = (int)carry[2];
    counts[0] = (int)(carry[0] + carry[1] + 2u * carry[2]);
  }
}

__device__ __forceinline__ void copy_row(const ocgs_surfels& in, const ocgs_surfels_mut& out, int j, size_t row, const float* pos3,
                                         float2 sc) {
  out.pos[3 * row] = pos3[0]; out.pos[3 * row + 1] = pos3[1]; out.pos[3 * row + 2] = pos3[2];
  ((float2*)out.scale)[row] = sc;
  ((float4*)out.quat)[row] = ((const float4*)in.quat)[j];
  out.opacity[row] = in.opacity[j];
  const float4* s = (const float4*)in.sh + (size_t)j * 12;
  float4* d = (float4*)out.sh + row * 12;
#pragma unroll
  for (int i = 0; i < 12; ++i) d[i] = __ldg(s + i);
}

__global__ void __launch_bounds__(kDenBlock) densify_scatter_kernel(ocgs_surfels in, const uint8_t* __restrict__ cls,
                                                                    const uint32_t* __restrict__ blocksum, const int* __restrict__ counts,
                                                                    const float* __restrict__ xi, ocgs_surfels_mut out,
                                                                    int32_t* __restrict__ src) {
  const int j = blockIdx.x * kDenBlock + threadIdx.x;
  const int n = in.n;
  const int c = j < n ? (int)cls[j] : -1;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  const unsigned b[3] = {__ballot_sync(0xFFFFFFFFu, c == 0 || c == 1), __ballot_sync(0xFFFFFFFFu, c == 1), __ballot_sync(0xFFFFFFFFu, c == 2)};
  __shared__ uint32_t ws[3][kDenBlock / 32];
  if (lane == 0) { ws[0][wid] = (uint32_t)__popc(b[0]); ws[1][wid] = (uint32_t)__popc(b[1]); ws[2][wid] = (uint32_t)__popc(b[2]); }
  __syncthreads();
  uint32_t pre[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    uint32_t s = blocksum[3 * blockIdx.x + k];
    for (int w2 = 0; w2 < wid; ++w2) s += ws[k][w2];
    pre[k] = s + (uint32_t)__popc(b[k] & lt);
  }
  if (c < 0) return;
  const size_t cap = (size_t)out.capacity;
  const size_t n_keep = (size_t)counts[1], n_clone = (size_t)counts[2];
  const float p[3] = {in.pos[3 * j], in.pos[3 * j + 1], in.pos[3 * j + 2]};
  const float2 sc = ((const float2*)in.scale)[j];
  if (c != 2) {  // survivors keep their relative order
    const size_t row = pre[0];
    if (row < cap) { copy_row(in, out, j, row, p, sc); if (src) src[row] = j; }
  }
  if (c == 1) {
    const size_t row = n_keep + pre[1];
    if (row < cap) { copy_row(in, out, j, row, p, sc); if (src) src[row] = j; }
  }
  if (c == 2) {
    const float4 q = ((const float4*)in.quat)[j];
    const float w = q.x, x = q.y, y = q.z, z = q.w;
    const float tu[3] = {1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y + w * z), 2.0f * (x * z - w * y)};
    const float tv[3] = {2.0f * (x * y - w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z + w * x)};
    const float2 cs = make_float2(sc.x / 1.6f, sc.y / 1.6f);
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const float a = sc.x * xi[4 * (size_t)j + 2 * k], bb = sc.y * xi[4 * (size_t)j + 2 * k + 1];
      const float pc[3] = {fmaf(a, tu[0], fmaf(bb, tv[0], p[0])), fmaf(a, tu[1], fmaf(bb, tv[1], p[1])), fmaf(a, tu[2], fmaf(bb, tv[2], p[2]))};
      const size_t row = n_keep + n_clone + 2 * (size_t)pre[2] + k;
      if (row < cap) { copy_row(in, out, j, row, pc, cs); if (src) src[row] = j; }
    }
  }
}

size_t densify_workspace_bytes(int n) {
  const size_t nb = div_up((size_t)(n > 0 ? n : 0), kDenBlock);
  return ((size_t)(n > 0 ? n : 0) + 255) / 256 * 256 + (3 * nb + 4) * sizeof(uint32_t);
}

int launch_densify_accumulate(const Workspace& w, const float* d_center2d, float* grad_accum, uint32_t* denom, cudaStream_t st) {
  if (w.n == 0) return OCGS_OK;
  densify_accumulate_kernel<<<(unsigned)div_up((size_t)w.n, 256), 256, 0, st>>>(w.id_to_rank, (const float2*)d_center2d, w.n, 0.5f * (float)w.width, 0.5f * (float)w.height, grad_accum, denom);
  OCGS_LAUNCHED(st, "densify_accumulate_kernel");
  return OCGS_OK;
}

int launch_densify(const ocgs_surfels& in, const float* grad_accum, const uint32_t* denom, float grad_threshold, float scale_threshold,
                   const float* xi, const ocgs_surfels_mut& out, int32_t* src, int* counts, void* ws, cudaStream_t st) {
  const int n = in.n;
  if (n == 0) {
    OCGS_CUDA_OK(cudaMemsetAsync(counts, 0, 4 * sizeof(int), st));
    return OCGS_OK;
  }
  uint8_t* cls = (uint8_t*)ws;
  uint32_t* blocksum = (uint32_t*)((char*)ws + ((size_t)n + 255) / 256 * 256);
  const int nb = (int)div_up((size_t)n, kDenBlock);
  densify_flag_kernel<<<nb, kDenBlock, 0, st>>>(grad_accum, denom, (const float2*)in.scale, n, grad_threshold, scale_threshold, cls, blocksum);
  OCGS_LAUNCHED(st, "densify_flag_kernel");
  densify_scan_kernel<<<1, 1024, 0, st>>>(blocksum, nb, counts);
  OCGS_LAUNCHED(st, "densify_scan_kernel");
  densify_scatter_kernel<<<nb, kDenBlock, 0, st>>>(in, cls, blocksum, counts, xi, out, src);
  OCGS_LAUNCHED(st, "densify_scatter_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
