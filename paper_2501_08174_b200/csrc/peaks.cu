// peaks.cu -- ocgs_peak_probe: the two microbenchmarks SURVEY.md 8(d) asks the roofline of the raster kernels to be quoted
// against: sustained FP32 FMA rate (plain ALUs) and MUFU.EX2 rate of the device the bench runs on.  Diagnostic only: no
// step of the hot path calls it; bench.py times it with CUDA events and reports peaks.fp32_tflops_measured /
// peaks.ex2_tops_measured.
#include "common.cuh"

namespace ocgs {

constexpr int kPeakChains = 8;  // independent dependency chains per thread: enough to cover the 4-cycle FMA latency at any occupancy

// kind 0: a_k <- fma(a_k, b, c), 2 flop per chain step
__global__ void __launch_bounds__(256) fma_peak_kernel(float* __restrict__ out, int iters, float b, float c) {
  float a[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) a[k] = (float)(threadIdx.x + k) * 1e-3f;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) a[k] = fmaf(a[k], b, c);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += a[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 1: a_k <- ex2(a_k) (MUFU.EX2), one transcendental per chain step; the argument stays in [-1, 0]
__global__ void __launch_bounds__(256) ex2_peak_kernel(float* __restrict__ out, int iters) {
  float a[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) a[k] = -(float)((threadIdx.x + k) & 7) * 0.125f;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) a[k] = -ex2_approx(a[k]);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += a[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kind 2: the same chains with b and c in REGISTERS: the values arrive as kernel arguments and take a round trip through volatile
// shared memory, after which they are per-thread values to the compiler -- it can neither fold them into uniform / constant-bank
// operands nor share one register between the chains: the three-register form real kernels issue
__global__ void __launch_bounds__(256) fma3_peak_kernel(float* __restrict__ out, int iters, float b_in, float c_in) {
  __shared__ volatile float s_bc[2][256];
  s_bc[0][threadIdx.x] = b_in; s_bc[1][threadIdx.x] = c_in;
  __syncthreads();
  float a[kPeakChains], b[kPeakChains], c[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) {
    a[k] = (float)(threadIdx.x + k) * 1e-3f; b[k] = s_bc[0][(threadIdx.x + k) & 255]; c[k] = s_bc[1][(threadIdx.x + 2 * k) & 255];
  }
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) a[k] = fmaf(a[k], b[k], c[k]);
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) s += a[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// kinds 3, 4: packed fp32 (fma.rn.f32x2, sm_100; SASS FFMA2): kPeakChains chains of TWO fused multiply-adds per instruction, operands
// in registers.  kBroadcast (kind 3): b and c are pairs {x, x} -- ptxas turns them into FFMA2's scalar-broadcast operand form
// (`FFMA2 Rd, Ra.F32x2.HI_LO, Rb.F32, Rc.F32`: four registers read); kind 4: b and c are pairs of two different values (`...,
// Rb.F32x2.HI_LO, Rc.F32x2.HI_LO`: six registers read, register-file bound like the three-register scalar FFMA)
template <bool kBroadcast>
__global__ void __launch_bounds__(256) fma2_peak_kernel(float* __restrict__ out, int iters, float b_in, float c_in) {
  __shared__ volatile float s_bc[2][256];
  s_bc[0][threadIdx.x] = b_in; s_bc[1][threadIdx.x] = c_in;
  __syncthreads();
  unsigned long long a[kPeakChains], b[kPeakChains], c[kPeakChains];
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) {
    const float a0 = (float)(threadIdx.x + k) * 1e-3f, a1 = a0 + 0.5f;
    const float b0 = s_bc[0][(threadIdx.x + k) & 255], b1 = kBroadcast ? b0 : s_bc[0][(threadIdx.x + k + 8) & 255];
    const float c0 = s_bc[1][(threadIdx.x + 2 * k) & 255], c1 = kBroadcast ? c0 : s_bc[1][(threadIdx.x + 2 * k + 1) & 255];
    asm("mov.b64 %0, {%1, %2};" : "=l"(a[k]) : "f"(a0), "f"(a1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b[k]) : "f"(b0), "f"(b1));
    asm("mov.b64 %0, {%1, %2};" : "=l"(c[k]) : "f"(c0), "f"(c1));
  }
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int k = 0; k < kPeakChains; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[k]) : "l"(b[k]), "l"(c[k]));
  }
  float s = 0.f;
#pragma unroll
  for (int k = 0; k < kPeakChains; ++k) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a[k]));
    s += lo + hi;
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace ocgs

extern "C" int ocgs_peak_probe(int kind, int iters, float* d_out, size_t out_floats, double* ops_per_launch, void* stream) {
  using namespace ocgs;
  if (!d_out || !ops_per_launch || iters <= 0 || kind < 0 || kind > 4) return OCGS_ERR_INVALID_ARG;
  int dev = 0, sms = 0;
  OCGS_CUDA_OK(cudaGetDevice(&dev));
  OCGS_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8;  // 8 resident blocks of 256 threads per SM: full occupancy, one wave
  if (out_floats < (size_t)blocks * 256) return OCGS_ERR_CAPACITY;
  const double steps = (double)blocks * 256.0 * (double)iters * 8.0 * (double)kPeakChains;
  cudaStream_t st = (cudaStream_t)stream;
  if (kind == 2) {
    fma3_peak_kernel<<<blocks, 256, 0, st>>>(d_out, iters, 0.999f, 1e-3f);
    *ops_per_launch = 2.0 * steps;
  } else if (kind == 3 || kind == 4) {
    if (kind == 3) fma2_peak_kernel<true><<<blocks, 256, 0, st>>>(d_out, iters, 0.999f, 1e-3f);
    else fma2_peak_kernel<false><<<blocks, 256, 0, st>>>(d_out, iters, 0.999f, 1e-3f);
    *ops_per_launch = 4.0 * steps;
  } else if (kind == 0) {
    fma_peak_kernel<<<blocks, 256, 0, st>>>(d_out, iters, 0.999f, 1e-3f);
    *ops_per_launch = 2.0 * steps;  // flop
  } else {
    ex2_peak_kernel<<<blocks, 256, 0, st>>>(d_out, iters);
    *ops_per_launch = steps;        // EX2 evaluations
  }
  OCGS_LAUNCH_OK();
  return OCGS_OK;
}
