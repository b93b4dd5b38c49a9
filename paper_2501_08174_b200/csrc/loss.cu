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

// ---- ocgs_masked_l1_static: the same term for callers that may not allocate -------------------------------------------------
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The per-block partial sums, the only
// scratch of this term, live in a file-scope device array instead of the caller's workspace: kStaticL1Partials floats = 32 KB,
// held by every GPU that loads the library until the process exits.  One block per 256 pixels, so the limit is
// OCGS_MASKED_L1_STATIC_MAX_PIXELS = 8192 * 256 = 2 097 152 pixels (every BASELINE.json config fits: 1920x1080 = 2 073 600),
// and the launch geometry -- hence the loss, bit for bit -- is that of ocgs_masked_l1.
// In HOST code the array's name is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.  All calls share the array: every slot a
// call reads it has written first (nothing has to start at zero, stale contents of the last call are never read), but two calls
// that overlap on the GPU (different streams, or concurrent graph branches) race on it.
namespace ocgs {
constexpr int kStaticL1Partials = 8192;
static __device__ __align__(256) float g_static_l1_partial[kStaticL1Partials];
static_assert((size_t)kStaticL1Partials * 256 == OCGS_MASKED_L1_STATIC_MAX_PIXELS, "limit stated in ocgs.h");
}  // namespace ocgs

#include <mutex>

extern "C" int ocgs_masked_l1_static(const float* color, const float* target, const uint8_t* mask, int width, int height, float* dL_dcolor,
                                     float* loss, void* stream) {
  using namespace ocgs;
  if (!color || !target || !dL_dcolor || width <= 0 || height <= 0) return OCGS_ERR_INVALID_ARG;
  if ((size_t)width * (size_t)height > (size_t)OCGS_MASKED_L1_STATIC_MAX_PIXELS) return OCGS_ERR_CAPACITY;  // beyond the static scratch
  // set-up, once per device: the device address of the scratch array on the CURRENT device
  constexpr int kMaxDevices = 64;
  static float* s_ptr[kMaxDevices] = {};
  static std::mutex s_mu;
  int dev = 0;
  OCGS_CUDA_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return OCGS_ERR_UNSUPPORTED;
  float* partial = nullptr;
  {
    std::lock_guard<std::mutex> lock(s_mu);
    if (!s_ptr[dev]) {
      void* p = nullptr;
      OCGS_CUDA_OK(cudaGetSymbolAddress(&p, g_static_l1_partial));
      if (!p) return OCGS_ERR_CUDA;
      s_ptr[dev] = (float*)p;
    }
    partial = s_ptr[dev];
  }
  return launch_masked_l1(color, target, mask, width, height, dL_dcolor, loss, partial, kStaticL1Partials, (cudaStream_t)stream);
}
