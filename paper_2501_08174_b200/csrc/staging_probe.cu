// staging_probe.cu -- ocgs_staging_probe: the staging step of the raster kernels in isolation, three ways (SURVEY.md section 7:
// "TMA where the layout allows ... cp.async.bulk.tensor.2d ... tile::gather4 ... probe it, fall back to LDG.128 / cp.async").
// Diagnostic only: no step of the hot path calls it.  Persistent CTAs of 256 threads (6 per SM, as the forward kernel) repeatedly
// gather a batch of 256 records of 96 bytes -- rows `ranks[...]` of the rank-ordered record table -- into shared memory and then
// read them the way the walk does (every thread reads one float4 of every 8th record: enough to make the data's arrival
// observable, little enough to leave the gather dominant):
//   kind 0  __ldg + st.shared + __syncthreads                       (what render_fwd_kernel / render_bwd_kernel do)
//   kind 1  cp.async 16 B (LDGSTS), double-buffered: batch b+1 is in flight while batch b is read
//   kind 2  TMA: cp.async.bulk.tensor.2d ... tile::gather4 over a [n_rec, 24] fp32 tensor map (box 24 x 1): one instruction gathers 4
//           rows (384 bytes), 32 instructions per batch issued by one warp, completion on an mbarrier (expect_tx = 12 288 bytes),
//           double-buffered
// Kinds 1 and 2 use batches of 128 records so that their two buffers take the shared memory of kind 0's one batch of 256.
#include <cuda.h>

#include "common.cuh"

namespace ocgs {

constexpr int kProbeBatch = 256;  // records per batch
constexpr int kProbeHalf = 128;   // records per batch of the double-buffered kinds (two buffers = the shared memory of one batch of 256)
constexpr int kProbeCtasPerSm = 6;

template <int B>
__device__ __forceinline__ float consume_batch(const float4* buf) {
  float acc = 0.f;
#pragma unroll
  for (int k = 0; k < B / 32; ++k) {  // record (tid + 32 k) mod B, float4 tid mod 6: B / 32 reads per thread, 1/6 of the batch in all
    const float4 x = buf[6 * ((threadIdx.x + 32 * k) & (B - 1)) + (threadIdx.x % 6)];
    acc += x.x + x.y + x.z + x.w;
  }
  return acc;
}

// kind 0
__global__ void __launch_bounds__(256, kProbeCtasPerSm) stage_ldg_kernel(const float4* __restrict__ rec, const uint32_t* __restrict__ ranks,
                                                                         uint32_t n_ranks, int iters, float* __restrict__ out) {
  __shared__ float4 s_rec[kProbeBatch * 6];
  __shared__ uint32_t s_rank[kProbeBatch];
  float acc = 0.f;
  for (int it = 0; it < iters; ++it) {
    const uint32_t base = (uint32_t)(((size_t)blockIdx.x * iters + it) * kProbeBatch % n_ranks);
    __syncthreads();
    s_rank[threadIdx.x] = ranks[(base + threadIdx.x) % n_ranks];
    __syncthreads();
    for (int i = threadIdx.x; i < kProbeBatch * 6; i += 256) {
      const int e = i / 6, part = i - 6 * e;
      s_rec[i] = __ldg(rec + (size_t)s_rank[e] * 6 + part);
    }
    __syncthreads();
    acc += consume_batch<kProbeBatch>(s_rec);
  }
  out[(size_t)blockIdx.x * 256 + threadIdx.x] = acc;
}

// kind 1
__global__ void __launch_bounds__(256, kProbeCtasPerSm) stage_cpasync_kernel(const float4* __restrict__ rec, const uint32_t* __restrict__ ranks,
                                                               uint32_t n_ranks, int iters, float* __restrict__ out) {
  __shared__ float4 s_rec[2][kProbeHalf * 6];
  float acc = 0.f;
  auto issue = [&](int buf, int it) {
    if (it < iters) {
      const uint32_t base = (uint32_t)(((size_t)blockIdx.x * iters + it) * kProbeHalf % n_ranks);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const int i = threadIdx.x + 256 * k, e = i / 6, part = i - 6 * e;
        const uint32_t r = __ldg(ranks + (base + e) % n_ranks);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(&s_rec[buf][i])),
                     "l"(rec + (size_t)r * 6 + part)
                     : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  issue(0, 0);
  for (int it = 0; it < iters; ++it) {
    issue((it + 1) & 1, it + 1);
    asm volatile("cp.async.wait_group 1;" ::: "memory");
    __syncthreads();
    acc += consume_batch<kProbeHalf>(s_rec[it & 1]);
    __syncthreads();  // the buffer is free for the batch after next
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  out[(size_t)blockIdx.x * 256 + threadIdx.x] = acc;
}

// kind 2
__global__ void __launch_bounds__(256, kProbeCtasPerSm) stage_tma_kernel(const __grid_constant__ CUtensorMap tmap, const uint32_t* __restrict__ ranks,
                                                                         uint32_t n_ranks, int iters, float* __restrict__ out) {
  __shared__ __align__(128) float4 s_rec[2][kProbeHalf * 6];
  __shared__ __align__(8) unsigned long long s_bar[2];
  const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(&s_bar[0]), bar1 = (uint32_t)__cvta_generic_to_shared(&s_bar[1]);
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar0) : "memory");
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar1) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  float acc = 0.f;
  // warp 0 issues the batch: lane l gathers records 4 l .. 4 l + 3 (384 bytes, contiguous in shared memory) with ONE instruction
  auto issue = [&](int buf, int it) {
    if (it < iters && threadIdx.x < 32) {
      const uint32_t bar = buf ? bar1 : bar0;
      if (threadIdx.x == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(kProbeHalf * 96) : "memory");
      const uint32_t base = (uint32_t)(((size_t)blockIdx.x * iters + it) * kProbeHalf % n_ranks);
      const uint32_t e = 4 * threadIdx.x;
      const int r0 = (int)__ldg(ranks + (base + e) % n_ranks), r1 = (int)__ldg(ranks + (base + e + 1) % n_ranks),
                r2 = (int)__ldg(ranks + (base + e + 2) % n_ranks), r3 = (int)__ldg(ranks + (base + e + 3) % n_ranks);
      const uint32_t dst = (uint32_t)__cvta_generic_to_shared(&s_rec[buf][6 * e]);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the generic-proxy reads of this buffer (two batches ago) precede the async-proxy writes
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                   ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(&tmap)), "r"(bar), "r"(0), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
                   : "memory");
    }
  };
  issue(0, 0);
  for (int it = 0; it < iters; ++it) {
    issue((it + 1) & 1, it + 1);
    const uint32_t bar = (it & 1) ? bar1 : bar0, parity = (uint32_t)(it >> 1) & 1u;
    uint32_t done = 0;
    while (!done) {
      asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    }
    acc += consume_batch<kProbeHalf>(s_rec[it & 1]);
    __syncthreads();  // every thread has read the buffer before the batch after next is gathered into it
  }
  out[(size_t)blockIdx.x * 256 + threadIdx.x] = acc;
}

}  // namespace ocgs

extern "C" int ocgs_staging_probe(int kind, const float* rec, const uint32_t* ranks, uint32_t n_rec, uint32_t n_ranks, int iters, float* d_out,
                                  size_t out_floats, double* bytes_per_launch, void* stream) {
  using namespace ocgs;
  if (!rec || !ranks || !d_out || !bytes_per_launch || n_rec == 0 || n_ranks < (uint32_t)kProbeBatch || iters <= 0 || kind < 0 || kind > 2)
    return OCGS_ERR_INVALID_ARG;
  const int blocks = sm_count() * kProbeCtasPerSm;
  if (out_floats < (size_t)blocks * 256) return OCGS_ERR_CAPACITY;
  cudaStream_t st = (cudaStream_t)stream;
  const int batch = kind == 0 ? kProbeBatch : kProbeHalf;
  *bytes_per_launch = (double)blocks * (double)iters * (double)batch * 96.0;  // record bytes gathered into shared memory
  if (kind == 0) {
    stage_ldg_kernel<<<blocks, 256, 0, st>>>((const float4*)rec, ranks, n_ranks, iters, d_out);
  } else if (kind == 1) {
    stage_cpasync_kernel<<<blocks, 256, 0, st>>>((const float4*)rec, ranks, n_ranks, iters, d_out);
  } else {
    // tensor map of the record table: [n_rec rows, 24 fp32 columns], row pitch 96 bytes, box = one row; the driver's encoder is
    // resolved through the runtime, so that the library does not link against libcuda
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres = cudaDriverEntryPointSymbolNotFound;
    OCGS_CUDA_OK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return OCGS_ERR_UNSUPPORTED;
    alignas(64) CUtensorMap tmap;
    const cuuint64_t gdim[2] = {24, n_rec};
    const cuuint64_t gstride[1] = {96};
    const cuuint32_t box[2] = {24, 1};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult cr = ((EncodeFn)fn)(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)rec, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                       CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (cr != CUDA_SUCCESS) { g_last_cuda_error = (int)cr; return OCGS_ERR_UNSUPPORTED; }
    stage_tma_kernel<<<blocks, 256, 0, st>>>(tmap, ranks, n_ranks, iters, d_out);
  }
  OCGS_LAUNCH_OK();
  return OCGS_OK;
}
