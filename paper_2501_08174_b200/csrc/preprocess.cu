// preprocess.cu -- ocgs_preprocess (O1): one thread per surfel.  HBM-bound: 40 B read per surfel, +192 B SH and ~116 B
// written per visible surfel.
#include "projection.cuh"

namespace ocgs {

// Two phases per block of 256 surfels.  (1) every thread projects and culls its surfel (Appendix A / R-bbox) and writes
// the per-id integers; the visible ones (29 % at config 3, scattered) are compacted into a block-local list.  (2) the
// list is processed densely, one visible surfel per thread: normal, SH colour (192 B read), the 96-byte raster record.
// Without the compaction every warp runs the long second part with a third of its lanes.
// kColour = false (the visibility pass): the facing normal and the SH colour are not needed -- the 192 B of SH per visible
// surfel are not read, the record's colour and normal slots stay zero.
template <bool kColour>
__global__ void __launch_bounds__(256) preprocess_kernel(const float* __restrict__ pos, const float2* __restrict__ scale,
                                                         const float4* __restrict__ quat, const float* __restrict__ opacity,
                                                         const float4* __restrict__ sh, int n, CamParams cam, ocgs_config cfg,
                                                         uint32_t* __restrict__ depth_bits, ushort4* __restrict__ rect,
                                                         uint32_t* __restrict__ tiles, uint8_t* __restrict__ clamp_bits,
                                                         float4* __restrict__ rec_id, uint32_t* __restrict__ id_to_rank,
                                                         uint32_t* __restrict__ sort_key, uint32_t* __restrict__ sort_val,
                                                         ocgs_header* __restrict__ header) {
  __shared__ uint32_t s_list[256];
  __shared__ uint32_t s_warp[8];
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  bool vis = false;
  if (j < n) {
    const float p[3] = {pos[3 * j], pos[3 * j + 1], pos[3 * j + 2]};
    Projected pr;
    project_surfel(p, scale[j].x, scale[j].y, quat[j], opacity[j], cam, cfg, pr);
    vis = pr.visible;
    const uint32_t zb = __float_as_uint(pr.pc[2]);
    depth_bits[j] = zb;
    sort_key[j] = vis ? zb : 0xFFFFFFFFu;  // culled surfels sort behind every positive depth
    sort_val[j] = (uint32_t)j;
    id_to_rank[j] = 0xFFFFFFFFu;
    uint32_t nt = 0;
    if (vis) {
      const int tx0 = pr.ix0 >> 4, tx1 = (pr.ix1 >> 4) + 1, ty0 = pr.iy0 >> 4, ty1 = (pr.iy1 >> 4) + 1;
      nt = (uint32_t)((tx1 - tx0) * (ty1 - ty0));
      rect[j] = make_ushort4((unsigned short)pr.ix0, (unsigned short)pr.iy0, (unsigned short)pr.ix1, (unsigned short)pr.iy1);
    } else {
      clamp_bits[j] = 0;
    }
    tiles[j] = nt;
  }
  // block-local compaction of the visible surfels (order inside the block is irrelevant: every output is indexed by id)
  const unsigned ball = __ballot_sync(0xFFFFFFFFu, vis);
  if (lane == 0) s_warp[wid] = (uint32_t)__popc(ball);
  __syncthreads();
  uint32_t before = 0, total = 0;
#pragma unroll
  for (int w2 = 0; w2 < 8; ++w2) {
    const uint32_t c = s_warp[w2];
    if (w2 < wid) before += c;
    total += c;
  }
  if (vis) s_list[before + (uint32_t)__popc(ball & ((1u << lane) - 1u))] = (uint32_t)j;
  if (threadIdx.x == 0 && total) atomicAdd(&header->n_vis, total);
  __syncthreads();
  if (threadIdx.x >= total) return;
  {
    const int id = (int)s_list[threadIdx.x];
    const float p[3] = {pos[3 * id], pos[3 * id + 1], pos[3 * id + 2]};
    const float4 q = quat[id];
    const float o = opacity[id];
    Projected pr;
    project_surfel(p, scale[id].x, scale[id].y, q, o, cam, cfg, pr);  // same inputs, same fp32 sequence: same result as phase 1
    uint8_t cl = 0;
    float nx = 0.f, ny = 0.f, nz = 0.f;
    float col[3] = {0.f, 0.f, 0.f};
    if (kColour) {
      // facing normal (view space): n = R_wc t_w, flipped when n . p_c > 0
      const float w = q.x, x = q.y, y = q.z, z = q.w;
      const float tw0 = 2.0f * (x * z + w * y), tw1 = 2.0f * (y * z - w * x), tw2 = 1.0f - 2.0f * (x * x + y * y);
      nx = cam.V[0] * tw0 + cam.V[1] * tw1 + cam.V[2] * tw2;
      ny = cam.V[4] * tw0 + cam.V[5] * tw1 + cam.V[6] * tw2;
      nz = cam.V[8] * tw0 + cam.V[9] * tw1 + cam.V[10] * tw2;
      if (nx * pr.pc[0] + ny * pr.pc[1] + nz * pr.pc[2] > 0.0f) { nx = -nx; ny = -ny; nz = -nz; }
      // SH colour (S14); the clamp decision follows the fixed fp32 sequence of reading R-clamp
      cl = sh_colour_rn(p, sh + (size_t)id * 12, cam, cfg.sh_degree, col);
    }
    {
      // centred record (common.cuh): P, Q, R, D0 in fp64 from the fp32 M, rounded once
      const float* M = pr.M;
      const double cxd = pr.cx, cyd = pr.cy;
      const double m2[3] = {M[6], M[7], M[8]};
      const double a0[3] = {M[0] - cxd * m2[0], M[1] - cxd * m2[1], M[2] - cxd * m2[2]};
      const double a1[3] = {M[3] - cyd * m2[0], M[4] - cyd * m2[1], M[5] - cyd * m2[2]};
      const double P[3] = {m2[1] * a1[2] - m2[2] * a1[1], m2[2] * a1[0] - m2[0] * a1[2], m2[0] * a1[1] - m2[1] * a1[0]};
      const double Q[3] = {a0[1] * m2[2] - a0[2] * m2[1], a0[2] * m2[0] - a0[0] * m2[2], a0[0] * m2[1] - a0[1] * m2[0]};
      const double R[3] = {a0[1] * a1[2] - a0[2] * a1[1], a0[2] * a1[0] - a0[0] * a1[2], a0[0] * a1[1] - a0[1] * a1[0]};
      const double D0 = m2[0] * R[0] + m2[1] * R[1] + m2[2] * R[2];
      float4* out = rec_id + (size_t)id * 6;
      out[0] = make_float4((float)P[0], (float)P[1], (float)P[2], (float)Q[0]);
      out[1] = make_float4((float)Q[1], (float)Q[2], (float)R[0], (float)R[1]);
      out[2] = make_float4((float)R[2], (float)D0, pr.cx, pr.cy);
      out[3] = make_float4(pr.rho_cut, M[8], __uint_as_float((uint32_t)pr.ix0 | ((uint32_t)pr.iy0 << 16)),
                           __uint_as_float((uint32_t)pr.ix1 | ((uint32_t)pr.iy1 << 16)));
      out[4] = make_float4(o, col[0], col[1], col[2]);
      out[5] = make_float4(nx, ny, nz, 0.0f);
    }
    clamp_bits[id] = cl;
  }
}

int launch_preprocess(const ocgs_surfels& s, const CamParams& cam, const ocgs_config& cfg, Workspace& w, cudaStream_t st, bool colour) {
  OCGS_CUDA_OK(cudaMemsetAsync(w.header, 0, sizeof(ocgs_header), st));
  if (g_prof_on) prof_mark(st, "memset_header");
  if (s.n == 0) return OCGS_OK;
  const int blocks = (int)div_up((size_t)s.n, 256);
  if (colour)
    preprocess_kernel<true><<<blocks, 256, 0, st>>>(s.pos, (const float2*)s.scale, (const float4*)s.quat, s.opacity, (const float4*)s.sh,
                                                    s.n, cam, cfg, w.depth_bits, w.rect, w.tiles, w.clamp, (float4*)w.rec_id,
                                                    w.id_to_rank, w.dkeyA, w.rank_to_id, w.header);
  else
    preprocess_kernel<false><<<blocks, 256, 0, st>>>(s.pos, (const float2*)s.scale, (const float4*)s.quat, s.opacity, (const float4*)s.sh,
                                                     s.n, cam, cfg, w.depth_bits, w.rect, w.tiles, w.clamp, (float4*)w.rec_id,
                                                     w.id_to_rank, w.dkeyA, w.rank_to_id, w.header);
  OCGS_LAUNCHED(st, "preprocess_kernel");
  return OCGS_OK;
}

}  // namespace ocgs
