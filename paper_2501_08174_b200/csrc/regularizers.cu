// regularizers.cu -- ocgs_regularizers: the depth-distortion and normal-consistency terms L_d, L_n of Eq. 3
// (the 2DGS regularisers, "unchanged", unmasked) as image-space functions of the maps the renderer
// returns for a view, and the upstream gradients ocgs_render_bwd_reg consumes (readings R-moments, R-Ld, R-Ln):
//   L_d = 1/(hw) sum_p (A m2 - m1^2)                (= sum_{i<j} w_i w_j (z_i - z_j)^2 per pixel; m1, m2 the depth moments about
//                                                    the first blended pair's depth, which keeps this difference well conditioned)
//   L_n = 1/(hw) sum_p (A - Nrm . Nhat),  Nhat = unit normal of the expected-depth surface zbar = D/A by central differences
// Two element-wise / 5-point-stencil kernels, HBM-bound: reg_terms_kernel reads 28 B and writes 48 B per pixel (dL/dNrm,
// dL/dm1, dL/dm2 and the gradients g_a, g_b of the two difference vectors), reg_gather_kernel reads ~44 B and writes 8 B.
// The surface-normal arithmetic runs in fp64: zbar differences of neighbouring pixels cancel to 1e-3 of zbar at f = 2800,
// which in fp32 would leave 1e-4 in Nhat; it is ~60 fp64 operations per pixel, far below the kernel's memory time.
#include "common.cuh"

namespace ocgs {

constexpr float kRegEpsA = 1e-4f;  // pixels with A <= this carry no surface (R-Ln)

struct RegCam { double inv_fx, inv_fy, ox, oy; int W, H; };

__device__ __forceinline__ bool reg_surface(const float* __restrict__ alpha, const float* __restrict__ depth, int x, int y, int W,
                                            double* zbar) {
  const size_t p = (size_t)y * W + x;
  const float a = alpha[p];
  if (!(a > kRegEpsA)) { *zbar = 0.0; return false; }
  *zbar = (double)depth[p] / (double)a;
  return true;
}

__global__ void __launch_bounds__(256) reg_terms_kernel(const float* __restrict__ alpha, const float* __restrict__ depth,
                                                        const float* __restrict__ mom /*[3,H,W]: origin, m1, m2*/, const float* __restrict__ normal, RegCam cam,
                                                        float wd_hw, float wn_hw, float* __restrict__ gM /*[2,H,W]*/, float* __restrict__ gN,
                                                        float* __restrict__ g_ab /*[6,H,W]*/, double* __restrict__ partial /*[blocks][2]*/) {
  const int W = cam.W, H = cam.H;
  const size_t HW = (size_t)W * H;
  const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
  double ld = 0.0, ln = 0.0;
  if (x < W && y < H) {
    const size_t p = (size_t)y * W + x;
    const float A = alpha[p], m1 = mom[HW + p], m2 = mom[2 * HW + p];
    const float n0 = normal[p], n1 = normal[HW + p], n2 = normal[2 * HW + p];
    ld = (double)A * (double)m2 - (double)m1 * (double)m1;
    gM[p] = -2.0f * wd_hw * m1;
    gM[HW + p] = wd_hw * A;
    double Nh[3] = {0.0, 0.0, 0.0}, ga[3] = {0.0, 0.0, 0.0}, gb[3] = {0.0, 0.0, 0.0};
    double z0, zxm, zxp, zym, zyp;
    bool valid = x > 0 && y > 0 && x < W - 1 && y < H - 1;
    if (valid) {
      valid = reg_surface(alpha, depth, x, y, W, &z0) & reg_surface(alpha, depth, x - 1, y, W, &zxm) & reg_surface(alpha, depth, x + 1, y, W, &zxp) &
              reg_surface(alpha, depth, x, y - 1, W, &zym) & reg_surface(alpha, depth, x, y + 1, W, &zyp);
    }
    if (valid) {
      // P = zbar r, r = ((x - ox)/fx, (y - oy)/fy, 1); a = (P(x+1) - P(x-1))/2 = (dz r + sz e_x/fx)/2 with dz, sz the
      // difference and sum of the two zbar (r(x+-1) = r -+ e_x/fx): no subtraction of nearly equal points
      const double rx = ((double)x - cam.ox) * cam.inv_fx, ry = ((double)y - cam.oy) * cam.inv_fy;
      const double dzx = zxp - zxm, szx = zxp + zxm, dzy = zyp - zym, szy = zyp + zym;
      const double a[3] = {0.5 * (dzx * rx + szx * cam.inv_fx), 0.5 * dzx * ry, 0.5 * dzx};
      const double b[3] = {0.5 * dzy * rx, 0.5 * (dzy * ry + szy * cam.inv_fy), 0.5 * dzy};
      const double c[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
      const double nc = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
      if (nc > 0.0) {
        const double inc = 1.0 / nc;
        Nh[0] = -c[0] * inc; Nh[1] = -c[1] * inc; Nh[2] = -c[2] * inc;
        // l = A - Nrm . Nhat: g_Nhat = -w_n Nrm / hw;  Nhat = -c/|c|  =>  g_c = -(g - Nhat (Nhat . g)) / |c|
        const double g[3] = {-(double)wn_hw * n0, -(double)wn_hw * n1, -(double)wn_hw * n2};
        const double dt = Nh[0] * g[0] + Nh[1] * g[1] + Nh[2] * g[2];
        const double gc[3] = {-(g[0] - Nh[0] * dt) * inc, -(g[1] - Nh[1] * dt) * inc, -(g[2] - Nh[2] * dt) * inc};
        // c = a x b  =>  g_a = b x g_c, g_b = g_c x a
        ga[0] = b[1] * gc[2] - b[2] * gc[1]; ga[1] = b[2] * gc[0] - b[0] * gc[2]; ga[2] = b[0] * gc[1] - b[1] * gc[0];
        gb[0] = gc[1] * a[2] - gc[2] * a[1]; gb[1] = gc[2] * a[0] - gc[0] * a[2]; gb[2] = gc[0] * a[1] - gc[1] * a[0];
      }
    }
    ln = (double)A - ((double)n0 * Nh[0] + (double)n1 * Nh[1] + (double)n2 * Nh[2]);
    gN[p] = (float)(-(double)wn_hw * Nh[0]); gN[HW + p] = (float)(-(double)wn_hw * Nh[1]); gN[2 * HW + p] = (float)(-(double)wn_hw * Nh[2]);
#pragma unroll
    for (int k = 0; k < 3; ++k) { g_ab[(size_t)k * HW + p] = (float)ga[k]; g_ab[(size_t)(3 + k) * HW + p] = (float)gb[k]; }
  }
  __shared__ double s_red[2][8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { ld += __shfl_xor_sync(0xFFFFFFFFu, ld, o); ln += __shfl_xor_sync(0xFFFFFFFFu, ln, o); }
  if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = ld; s_red[1][threadIdx.x >> 5] = ln; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) { a += s_red[0][w]; b += s_red[1][w]; }
    const size_t blk = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
    partial[2 * blk] = a; partial[2 * blk + 1] = b;
  }
}

__global__ void __launch_bounds__(256) reg_gather_kernel(const float* __restrict__ alpha, const float* __restrict__ depth,
                                                         const float* __restrict__ mom, RegCam cam, float wd_hw, float wn_hw,
                                                         const float* __restrict__ g_ab, float* __restrict__ gA, float* __restrict__ gD) {
  const int W = cam.W, H = cam.H;
  const size_t HW = (size_t)W * H;
  const int x = blockIdx.x * 32 + (threadIdx.x & 31), y = blockIdx.y * 8 + (threadIdx.x >> 5);
  if (x >= W || y >= H) return;
  const size_t p = (size_t)y * W + x;
  // g_P(q) = ( g_a(q - e_x) - g_a(q + e_x) + g_b(q - e_y) - g_b(q + e_y) ) / 2
  double gP[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    double v = 0.0;
    if (x > 0) v += (double)g_ab[(size_t)k * HW + p - 1];
    if (x < W - 1) v -= (double)g_ab[(size_t)k * HW + p + 1];
    if (y > 0) v += (double)g_ab[(size_t)(3 + k) * HW + p - W];
    if (y < H - 1) v -= (double)g_ab[(size_t)(3 + k) * HW + p + W];
    gP[k] = 0.5 * v;
  }
  const double rx = ((double)x - cam.ox) * cam.inv_fx, ry = ((double)y - cam.oy) * cam.inv_fy;
  const double gz = gP[0] * rx + gP[1] * ry + gP[2];  // P = zbar r
  const float A = alpha[p], D = depth[p];
  double ga = (double)wd_hw * (double)mom[2 * HW + p] + (double)wn_hw;  // d(A m2 - m1^2)/dA + d(A - Nrm.Nhat)/dA
  double gd = 0.0;
  if (A > kRegEpsA) {  // zbar = D / A
    const double ia = 1.0 / (double)A;
    gd += gz * ia;
    ga -= gz * (double)D * ia * ia;
  }
  gA[p] = (float)ga;
  gD[p] = (float)gd;
}

__global__ void __launch_bounds__(1024) reg_final_kernel(const double* __restrict__ partial, int n_blocks, double inv_hw, float* __restrict__ loss) {
  __shared__ double s[2][1024];
  double a = 0.0, b = 0.0;
  for (int i = threadIdx.x; i < n_blocks; i += 1024) { a += partial[2 * i]; b += partial[2 * i + 1]; }
  s[0][threadIdx.x] = a; s[1][threadIdx.x] = b;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) { s[0][threadIdx.x] += s[0][threadIdx.x + o]; s[1][threadIdx.x] += s[1][threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { loss[0] = (float)(s[0][0] * inv_hw); loss[1] = (float)(s[1][0] * inv_hw); }
}

static size_t reg_align(size_t x) { return (x + 255) & ~(size_t)255; }

size_t regularizers_workspace_bytes(int W, int H) {
  if (W <= 0 || H <= 0) return 0;
  const size_t HW = (size_t)W * H;
  const size_t blocks = div_up((size_t)W, 32) * div_up((size_t)H, 8);
  return reg_align(6 * HW * sizeof(float)) + reg_align(blocks * 2 * sizeof(double));
}

int launch_regularizers(const float* alpha, const float* depth, const float* mom, const float* normal, const ocgs_camera& c, float w_d,
                        float w_n, float* gA, float* gD, float* gM, float* gN, float* loss, void* scratch, cudaStream_t st) {
  RegCam cam;
  cam.inv_fx = 1.0 / (double)c.fx; cam.inv_fy = 1.0 / (double)c.fy;
  cam.ox = (double)(c.cx - 0.5f); cam.oy = (double)(c.cy - 0.5f);
  cam.W = c.width; cam.H = c.height;
  const size_t HW = (size_t)c.width * c.height;
  float* g_ab = (float*)scratch;
  double* partial = (double*)((char*)scratch + reg_align(6 * HW * sizeof(float)));
  const double inv_hw = 1.0 / (double)HW;
  const dim3 grid((unsigned)div_up((size_t)c.width, 32), (unsigned)div_up((size_t)c.height, 8));
  reg_terms_kernel<<<grid, 256, 0, st>>>(alpha, depth, mom, normal, cam, (float)((double)w_d * inv_hw), (float)((double)w_n * inv_hw), gM, gN,
                                         g_ab, partial);
  OCGS_LAUNCHED(st, "reg_terms_kernel");
  reg_gather_kernel<<<grid, 256, 0, st>>>(alpha, depth, mom, cam, (float)((double)w_d * inv_hw), (float)((double)w_n * inv_hw), g_ab, gA, gD);
  OCGS_LAUNCHED(st, "reg_gather_kernel");
  if (loss) {
    reg_final_kernel<<<1, 1024, 0, st>>>(partial, (int)(grid.x * grid.y), inv_hw, loss);
    OCGS_LAUNCHED(st, "reg_final_kernel");
  }
  return OCGS_OK;
}

}  // namespace ocgs
