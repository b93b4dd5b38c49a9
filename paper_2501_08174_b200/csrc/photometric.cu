// photometric.cu -- ocgs_photometric_loss: the masked photometric loss L_c^M = L_c(I M, R M) of Eq. 2
// and its gradient w.r.t. the rendered colour.  L_c = (1 - lam) mean|x - y| + lam (1 - mean SSIM(x, y)) (reading S20b,
// DESIGN.md): SSIM per channel over an 11x11 Gaussian window (sigma 1.5, normalised), zero padding, C1 = 1e-4, C2 = 9e-4.
//
// Two stencil kernels, each a separable 11-tap blur staged through shared memory (block = 32x32 output pixels of one
// channel, 42x42 input region, 256 threads x 4 pixels):
//   ssim_terms_kernel: x = R M, y = I M; blurs x, y, x^2, y^2, x y; SSIM per pixel; writes the three per-pixel factors
//                      gS dS/dmu_x, gS dS/d(G*x^2), gS dS/d(G*xy) (gS = -lam/(3HW)) and block partials of sum|x-y|, sum SSIM
//   ssim_grad_kernel:  blurs the three factor maps (the adjoint of a windowed sum with a symmetric window is the same
//                      windowed sum) and combines dL/dx = G*d_mu + 2 x G*d_xx + y G*d_xy + (1-lam) sign(x-y)/(3HW), dL/dR = M dL/dx
// HBM-bound by design: 25 B read + 36 B written per pixel (terms), 61 B read + 12 B written (grad).
#include "common.cuh"

namespace ocgs {

constexpr int kPT = 32;            // output tile edge
constexpr int kPH = 5;             // window half width
constexpr int kPR = kPT + 2 * kPH;  // 42: staged region edge

struct GaussTaps { float g[11]; };

// resident blocks per SM the register budgets are held to (terms: 92 us with 5, 101 with 4; grad: 82 us with 6, 84 with 5)
constexpr int kSsimTermsBlocks = 5, kSsimGradBlocks = 6;
__global__ void __launch_bounds__(256, kSsimTermsBlocks) ssim_terms_kernel(const float* __restrict__ color, const float* __restrict__ target,
                                                         const uint8_t* __restrict__ mask, int W, int H, GaussTaps taps, float gS,
                                                         float* __restrict__ d_mu, float* __restrict__ d_xx, float* __restrict__ d_xy,
                                                         double* __restrict__ partial /*[blocks][2]*/) {
  __shared__ float s_x[kPR][kPR + 1], s_y[kPR][kPR + 1];
  __shared__ float s_h[5][kPR][kPT + 1];  // horizontally blurred x, y, xx, yy, xy
  __shared__ double s_red[2][8];
  const int c = blockIdx.z;
  const size_t HW = (size_t)W * H;
  const float* R = color + (size_t)c * HW;
  const float* I = target + (size_t)c * HW;
  const int x0 = blockIdx.x * kPT, y0 = blockIdx.y * kPT;
  // staging: warp w takes rows w, w + 8, ..., lane l columns l and l + 32; the loads of a thread are independent of one
  // another (the mask selects afterwards), so all of them are in flight together
  {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < (kPR + 7) / 8; ++k) {
      const int ry = warp + 8 * k, y = y0 + ry - kPH;
      if (ry >= kPR) break;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int rx = lane + 32 * h, x = x0 + rx - kPH;
        if (rx >= kPR) continue;
        float xv = 0.f, yv = 0.f;
        if (x >= 0 && y >= 0 && x < W && y < H) {  // zero padding outside the image
          const size_t p = (size_t)y * W + x;
          const bool m = mask == nullptr || mask[p] != 0;
          xv = R[p]; yv = I[p];
          if (!m) { xv = 0.f; yv = 0.f; }
        }
        s_x[ry][rx] = xv; s_y[ry][rx] = yv;
      }
    }
  }
  __syncthreads();
  // horizontal pass, 8 adjacent outputs per thread: 18 staged values feed 8 x 11 taps (one map at a time)
  for (int i = threadIdx.x; i < kPR * (kPT / 8); i += 256) {
    const int ry = i / (kPT / 8), ox0 = (i - ry * (kPT / 8)) * 8;
    float xs[18], ys[18];
#pragma unroll
    for (int t = 0; t < 18; ++t) { xs[t] = s_x[ry][ox0 + t]; ys[t] = s_y[ry][ox0 + t]; }
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      float v[18];
#pragma unroll
      for (int t = 0; t < 18; ++t) v[t] = m == 0 ? xs[t] : m == 1 ? ys[t] : m == 2 ? xs[t] * xs[t] : m == 3 ? ys[t] * ys[t] : xs[t] * ys[t];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        float a = 0.f;
#pragma unroll
        for (int t = 0; t < 11; ++t) a = fmaf(taps.g[t], v[k + t], a);
        s_h[m][ry][ox0 + k] = a;
      }
    }
  }
  __syncthreads();
  double l1 = 0.0, ss = 0.0;
  // vertical pass, 4 vertically adjacent outputs per thread: 14 values per map feed 4 x 11 taps
  for (int i = threadIdx.x; i < kPT * (kPT / 4); i += 256) {
    const int ox = i % kPT, oy0 = (i / kPT) * 4;
    float bl[5][4];
#pragma unroll
    for (int m = 0; m < 5; ++m) {
      float v[14];
#pragma unroll
      for (int t = 0; t < 14; ++t) v[t] = s_h[m][oy0 + t][ox];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        float a = 0.f;
#pragma unroll
        for (int t = 0; t < 11; ++t) a = fmaf(taps.g[t], v[k + t], a);
        bl[m][k] = a;
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int oy = oy0 + k, ix = x0 + ox, iy = y0 + oy;
      if (ix >= W || iy >= H) continue;
      const float mx = bl[0][k], my = bl[1][k], exx = bl[2][k], eyy = bl[3][k], exy = bl[4][k];
      const float sxx = exx - mx * mx, syy = eyy - my * my, sxy = exy - mx * my;
      const float A1 = fmaf(2.0f * mx, my, 1e-4f), A2 = fmaf(2.0f, sxy, 9e-4f);
      const float B1 = fmaf(mx, mx, fmaf(my, my, 1e-4f)), B2 = sxx + syy + 9e-4f;
      const float iB1 = 1.0f / B1, iB2 = 1.0f / B2, iB = iB1 * iB2;
      const float S = A1 * A2 * iB;
      const size_t p = (size_t)c * HW + (size_t)iy * W + ix;
      d_mu[p] = gS * (2.0f * my * (A2 - A1) * iB - 2.0f * mx * S * (iB1 - iB2));
      d_xx[p] = gS * (-S * iB2);
      d_xy[p] = gS * (2.0f * A1 * iB);
      l1 += (double)fabsf(s_x[oy + kPH][ox + kPH] - s_y[oy + kPH][ox + kPH]);
      ss += (double)S;
    }
  }
  // block partials (fixed order -> deterministic totals)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { l1 += __shfl_xor_sync(0xFFFFFFFFu, l1, o); ss += __shfl_xor_sync(0xFFFFFFFFu, ss, o); }
  if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = l1; s_red[1][threadIdx.x >> 5] = ss; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) { a += s_red[0][w]; b += s_red[1][w]; }
    const size_t blk = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    partial[2 * blk] = a; partial[2 * blk + 1] = b;
  }
}

__global__ void __launch_bounds__(256, kSsimGradBlocks) ssim_grad_kernel(const float* __restrict__ color, const float* __restrict__ target,
                                                        const uint8_t* __restrict__ mask, int W, int H, GaussTaps taps, float l1_scale,
                                                        const float* __restrict__ d_mu, const float* __restrict__ d_xx,
                                                        const float* __restrict__ d_xy, float* __restrict__ dL_dcolor) {
  __shared__ float s_in[3][kPR][kPR + 1];
  __shared__ float s_h[3][kPR][kPT + 1];
  const int c = blockIdx.z;
  const size_t HW = (size_t)W * H;
  const int x0 = blockIdx.x * kPT, y0 = blockIdx.y * kPT;
  const float* src[3] = {d_mu + (size_t)c * HW, d_xx + (size_t)c * HW, d_xy + (size_t)c * HW};
  {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < (kPR + 7) / 8; ++k) {
      const int ry = warp + 8 * k, y = y0 + ry - kPH;
      if (ry >= kPR) break;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int rx = lane + 32 * h, x = x0 + rx - kPH;
        if (rx >= kPR) continue;
        const bool in = x >= 0 && y >= 0 && x < W && y < H;
        const size_t p = in ? (size_t)y * W + x : 0;
#pragma unroll
        for (int m = 0; m < 3; ++m) s_in[m][ry][rx] = in ? src[m][p] : 0.f;
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kPR * (kPT / 8); i += 256) {
    const int ry = i / (kPT / 8), ox0 = (i - ry * (kPT / 8)) * 8;
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      float v[18];
#pragma unroll
      for (int t = 0; t < 18; ++t) v[t] = s_in[m][ry][ox0 + t];
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        float a = 0.f;
#pragma unroll
        for (int t = 0; t < 11; ++t) a = fmaf(taps.g[t], v[k + t], a);
        s_h[m][ry][ox0 + k] = a;
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < kPT * (kPT / 4); i += 256) {
    const int ox = i % kPT, oy0 = (i / kPT) * 4;
    float bl[3][4];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      float v[14];
#pragma unroll
      for (int t = 0; t < 14; ++t) v[t] = s_h[m][oy0 + t][ox];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        float a = 0.f;
#pragma unroll
        for (int t = 0; t < 11; ++t) a = fmaf(taps.g[t], v[k + t], a);
        bl[m][k] = a;
      }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int ix = x0 + ox, iy = y0 + oy0 + k;
      if (ix >= W || iy >= H) continue;
      const size_t pp = (size_t)iy * W + ix;
      const bool m = mask == nullptr || mask[pp] != 0;
      float out = 0.f;
      if (m) {  // x = R M: no gradient reaches the render outside the mask
        const float x = color[(size_t)c * HW + pp], y = target[(size_t)c * HW + pp];
        const float d = x - y;
        out = bl[0][k] + 2.0f * x * bl[1][k] + y * bl[2][k] + (d > 0.f ? l1_scale : (d < 0.f ? -l1_scale : 0.f));
      }
      dL_dcolor[(size_t)c * HW + pp] = out;
    }
  }
}

__global__ void __launch_bounds__(1024) photometric_final_kernel(const double* __restrict__ partial, int n_blocks, double inv_n, float lam,
                                                                 float* __restrict__ loss /*[3]: total, l1, dssim*/) {
  __shared__ double s[2][1024];
  double a = 0.0, b = 0.0;
  for (int i = threadIdx.x; i < n_blocks; i += 1024) { a += partial[2 * i]; b += partial[2 * i + 1]; }
  s[0][threadIdx.x] = a; s[1][threadIdx.x] = b;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) { s[0][threadIdx.x] += s[0][threadIdx.x + o]; s[1][threadIdx.x] += s[1][threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const double l1 = s[0][0] * inv_n, dssim = 1.0 - s[1][0] * inv_n;
    loss[0] = (float)((1.0 - (double)lam) * l1 + (double)lam * dssim);
    loss[1] = (float)l1;
    loss[2] = (float)dssim;
  }
}

static size_t photo_align(size_t x) { return (x + 255) & ~(size_t)255; }

size_t photometric_workspace_bytes(int W, int H) {
  if (W <= 0 || H <= 0) return 0;
  const size_t HW = (size_t)W * H;
  const size_t blocks = div_up((size_t)W, kPT) * div_up((size_t)H, kPT) * 3;
  return 3 * photo_align(3 * HW * sizeof(float)) + photo_align(blocks * 2 * sizeof(double));
}

int launch_photometric(const float* color, const float* target, const uint8_t* mask, int W, int H, float lam, float* dL_dcolor,
                       float* loss, void* scratch, cudaStream_t st) {
  const size_t HW = (size_t)W * H;
  char* b = (char*)scratch;
  const size_t map_bytes = photo_align(3 * HW * sizeof(float));
  float* d_mu = (float*)b;
  float* d_xx = (float*)(b + map_bytes);
  float* d_xy = (float*)(b + 2 * map_bytes);
  double* partial = (double*)(b + 3 * map_bytes);
  GaussTaps taps;
  double g[11], sum = 0.0;
  for (int i = 0; i < 11; ++i) { g[i] = exp(-(double)((i - 5) * (i - 5)) / (2.0 * 1.5 * 1.5)); sum += g[i]; }
  for (int i = 0; i < 11; ++i) taps.g[i] = (float)(g[i] / sum);
  const double n = 3.0 * (double)HW;
  const dim3 grid((unsigned)div_up((size_t)W, kPT), (unsigned)div_up((size_t)H, kPT), 3);
  ssim_terms_kernel<<<grid, 256, 0, st>>>(color, target, mask, W, H, taps, (float)(-(double)lam / n), d_mu, d_xx, d_xy, partial);
  OCGS_LAUNCHED(st, "ssim_terms_kernel");
  ssim_grad_kernel<<<grid, 256, 0, st>>>(color, target, mask, W, H, taps, (float)((1.0 - (double)lam) / n), d_mu, d_xx, d_xy, dL_dcolor);
  OCGS_LAUNCHED(st, "ssim_grad_kernel");
  if (loss) {
    photometric_final_kernel<<<1, 1024, 0, st>>>(partial, (int)(grid.x * grid.y * grid.z), 1.0 / n, lam, loss);
    OCGS_LAUNCHED(st, "photometric_final_kernel");
  }
  return OCGS_OK;
}

}  // namespace ocgs
