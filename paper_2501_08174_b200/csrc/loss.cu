// loss.cu -- harness photometric term (S20): masked L1 between render and target and its gradient,
// L = 1/(3HW) sum_c sum_p |M (R - I)|, dL/dR = M sign(R - I) / (3HW)  (the L1 part of Eq. 2).
// Element-wise, HBM-bound: 25 B read + 12 B written per pixel.
#include "common.cuh"

namespace ocgs {

__global__ void __launch_bounds__(256) masked_l1_kernel(const float* __restrict__ color, const float* __restrict__ target,
                                                        const uint8_t* __restrict__ mask, size_t HW, float inv_norm,
                                                        float* __restrict__ dL_dcolor, float* __restrict__ partial) {
  float acc = 0.f;
  for (size_t p = (size_t)blockIdx.x * 256 + threadIdx.x; p < HW; p += (size_t)gridDim.x * 256) {
    const bool m = mask == nullptr || mask[p] != 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float d = m ? color[c * HW + p] - target[c * HW + p] : 0.f;
      acc += fabsf(d);
      dL_dcolor[c * HW + p] = d > 0.f ? inv_norm : (d < 0.f ? -inv_norm : 0.f);
    }
  }
  __shared__ float ws[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) s += ws[w];
    partial[blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(1024) sum_partials_kernel(const float* __restrict__ partial, int n, float scale, float* __restrict__ out) {
  __shared__ double s[1024];
  double acc = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) acc += (double)partial[i];
  s[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) s[threadIdx.x] += s[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = (float)(s[0] * (double)scale);
}

int launch_masked_l1(const float* color, const float* target, const uint8_t* mask, int W, int H, float* dL_dcolor, float* loss,
                     float* partial, int n_partial, cudaStream_t st) {
  const size_t HW = (size_t)W * H;
  const float inv_norm = (float)(1.0 / (3.0 * (double)HW));
  const int grid = (int)min((size_t)n_partial, div_up(HW, 256));
  if (grid == 0) return OCGS_OK;
  masked_l1_kernel<<<grid, 256, 0, st>>>(color, target, mask, HW, inv_norm, dL_dcolor, partial);
  OCGS_LAUNCHED(st, "masked_l1_kernel");
  if (loss) {
    sum_partials_kernel<<<1, 1024, 0, st>>>(partial, grid, inv_norm, loss);
    OCGS_LAUNCHED(st, "sum_partials_kernel");
  }
  return OCGS_OK;
}

}  // namespace ocgs
