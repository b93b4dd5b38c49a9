// api.cu -- extern "C" entry points of libocgs (include/ocgs.h): argument checks, workspace carving, stage launches.
#include <string.h>

#include <vector>

#include "common.cuh"

namespace ocgs {

thread_local int g_last_cuda_error = 0;

// ---- diagnostic per-launch timing -------------------------------------------------------------------------------
thread_local bool g_prof_on = false;
namespace {
struct Prof { std::vector<cudaEvent_t> ev; std::vector<const char*> names; size_t used = 0; };
thread_local Prof g_prof;
}
void prof_mark(cudaStream_t st, const char* name) {
  if (g_prof.used >= g_prof.ev.size()) return;
  cudaEventRecord(g_prof.ev[g_prof.used], st);
  g_prof.names[g_prof.used] = name;
  ++g_prof.used;
}

int sm_count() {
  thread_local int n = 0;
  if (n == 0) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;  // B200
  }
  return n;
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

bool carve_workspace(void* ws, int n, int width, int height, size_t key_capacity, Workspace* out, ocgs_ws_layout* layout) {
  if (n < 0 || width <= 0 || height <= 0 || width > OCGS_MAX_DIM || height > OCGS_MAX_DIM) return false;
  if (key_capacity >= (1ull << 30) || (size_t)n >= (1ull << 30)) return false;  // 30-bit counts in the radix status words
  const int tiles_x = (width + kTile - 1) / kTile, tiles_y = (height + kTile - 1) / kTile;
  const size_t n_tiles = (size_t)tiles_x * tiles_y;
  const size_t N = (size_t)n, K = key_capacity;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off = align256(off + bytes); return o; };
  ocgs_ws_layout L;
  memset(&L, 0, sizeof(L));
  L.header = take(256);
  L.depth_bits = take(N * 4);
  L.rect = take(N * 8);
  L.tiles = take(N * 4);
  L.clamp = take(N);
  L.rec_id = take(N * kRec * 4);
  L.id_to_rank = take(N * 4);
  L.rank_to_id = take(N * 4);
  L.rec = take(N * kRec * 4);
  L.offsets = take((N + 1) * 4);
  L.tile_keys = take(K * 4);
  L.tile_vals = take(K * 4);
  L.ranges = take(n_tiles * 8);
  L.grad_rec = take(N * kRec * 4);
  L.loss_partial = take(n_tiles * 8);  // two per-tile partial sums (L_b, fused L1)
  L.final_T = take((size_t)width * height * 4);
  L.scratch = off;
  const size_t o_dkeyA = take(N * 4), o_dkeyB = take(N * 4), o_dvalB = take(N * 4);
  const size_t o_tkeyB = take(K * 4), o_tvalB = take(K * 4);
  const size_t o_hit = take(K * 8);
  const size_t max_items = N > K ? N : K;
  const size_t o_hist = take((div_up(max_items, kSortTile) + 1) * kRadix * 4 * 4);  // look-back status words, 4 passes
  const size_t o_dtot = take((4 * kRadix + 4) * 4);  // global digit histograms of 4 passes + 4 tile tickets
  const size_t o_tcount = take(N * 4);
  const size_t o_bsum = take((div_up(N, 1024) + 2) * 4);
  const size_t o_twork = take(n_tiles * 4), o_torder = take(n_tiles * 4);
  L.total_bytes = off;
  if (layout) *layout = L;
  if (out) {
    char* b = (char*)ws;
    out->header = (ocgs_header*)(b + L.header);
    out->depth_bits = (uint32_t*)(b + L.depth_bits);
    out->rect = (ushort4*)(b + L.rect);
    out->tiles = (uint32_t*)(b + L.tiles);
    out->clamp = (uint8_t*)(b + L.clamp);
    out->rec_id = (float*)(b + L.rec_id);
    out->id_to_rank = (uint32_t*)(b + L.id_to_rank);
    out->rank_to_id = (uint32_t*)(b + L.rank_to_id);
    out->rec = (float*)(b + L.rec);
    out->offsets = (uint32_t*)(b + L.offsets);
    out->tile_keys = (uint32_t*)(b + L.tile_keys);
    out->tile_vals = (uint32_t*)(b + L.tile_vals);
    out->ranges = (uint32_t*)(b + L.ranges);
    out->grad_rec = (float*)(b + L.grad_rec);
    out->loss_partial = (float*)(b + L.loss_partial);
    out->final_T = (float*)(b + L.final_T);
    out->dkeyA = (uint32_t*)(b + o_dkeyA);
    out->dkeyB = (uint32_t*)(b + o_dkeyB);
    out->dvalB = (uint32_t*)(b + o_dvalB);
    out->tkeyB = (uint32_t*)(b + o_tkeyB);
    out->tvalB = (uint32_t*)(b + o_tvalB);
    out->blist = (uint2*)(b + o_hit);
    out->hist = (uint32_t*)(b + o_hist);
    out->digit_total = (uint32_t*)(b + o_dtot);
    out->tcount = (uint32_t*)(b + o_tcount);
    out->blocksum = (uint32_t*)(b + o_bsum);
    out->tile_work = (uint32_t*)(b + o_twork);
    out->tile_order = (uint32_t*)(b + o_torder);
    out->n = n; out->width = width; out->height = height;
    out->tiles_x = tiles_x; out->tiles_y = tiles_y; out->n_tiles = (int)n_tiles;
    out->key_capacity = key_capacity;
  }
  return true;
}

CamParams make_cam(const ocgs_camera& c) {
  CamParams p;
  for (int i = 0; i < 12; ++i) p.V[i] = c.view[i];
  p.fx = c.fx; p.fy = c.fy;
  p.ox = c.cx - 0.5f; p.oy = c.cy - 0.5f;
  // camera position -R^T t (double, rounded once)
  for (int k = 0; k < 3; ++k)
    p.campos[k] = (float)(-((double)c.view[k] * c.view[3] + (double)c.view[4 + k] * c.view[7] + (double)c.view[8 + k] * c.view[11]));
  p.W = c.width; p.H = c.height;
  p.tiles_x = (c.width + kTile - 1) / kTile;
  p.tiles_y = (c.height + kTile - 1) / kTile;
  return p;
}

static int check_cfg(const ocgs_config* cfg) {
  if (!cfg) return OCGS_ERR_INVALID_ARG;
  if (cfg->tile != kTile || cfg->sh_degree < 0 || cfg->sh_degree > 3) return OCGS_ERR_UNSUPPORTED;
  if (!(cfg->filter_sigma2 > 0.f) || !(cfg->alpha_min > 0.f)) return OCGS_ERR_INVALID_ARG;
  return OCGS_OK;
}

}  // namespace ocgs

using namespace ocgs;

extern "C" {

void ocgs_default_config(ocgs_config* c) {
  c->tile = 16; c->near_z = 0.2f; c->alpha_min = (float)(1.0 / 255.0); c->alpha_max = 0.99f; c->t_min = 1e-4f;
  c->rho_max = 9.0f; c->filter_sigma2 = 0.5f; c->bg[0] = c->bg[1] = c->bg[2] = 0.f; c->gamma_bg = 0.5f;
  c->tau_contrib = 0.f; c->min_opacity = 0.f; c->sh_degree = 3;
}

int ocgs_workspace_layout(int n, int width, int height, size_t key_capacity, ocgs_ws_layout* out) {
  if (!out) return OCGS_ERR_INVALID_ARG;
  return carve_workspace(nullptr, n, width, height, key_capacity, nullptr, out) ? OCGS_OK : OCGS_ERR_UNSUPPORTED;
}

size_t ocgs_workspace_bytes(int n, int width, int height, size_t key_capacity) {
  ocgs_ws_layout L;
  return carve_workspace(nullptr, n, width, height, key_capacity, nullptr, &L) ? L.total_bytes : 0;
}

int ocgs_last_cuda_error(void) { return g_last_cuda_error; }

int ocgs_check(const void* ws, void* stream, ocgs_header* header_out) {
  if (!ws) return OCGS_ERR_INVALID_ARG;
  ocgs_header h;
  OCGS_CUDA_OK(cudaMemcpyAsync(&h, ws, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  OCGS_CUDA_OK(cudaStreamSynchronize((cudaStream_t)stream));
  if (header_out) *header_out = h;
  return (h.error & 1u) ? OCGS_ERR_CAPACITY : (h.error & 2u) ? OCGS_ERR_UNSUPPORTED : OCGS_OK;
}

int ocgs_preprocess(const ocgs_surfels* s, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, void* stream) {
  if (!s || !cam || !ws) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if (s->n > 0 && (!s->pos || !s->scale || !s->quat || !s->opacity || !s->sh)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, s->n, cam->width, cam->height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  return launch_preprocess(*s, make_cam(*cam), *cfg, w, (cudaStream_t)stream);
}

int ocgs_bin_sort(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, uint32_t* sorted_ids, void* stream) {
  if (!cam || !ws) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  Workspace w;
  if (!carve_workspace(ws, n, cam->width, cam->height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  return launch_bin_sort(make_cam(*cam), w, sorted_ids, (cudaStream_t)stream);
}

static int carve_for_render(void* ws, int n, const ocgs_camera* cam, size_t key_capacity, Workspace* w) {
  return carve_workspace(ws, n, cam->width, cam->height, key_capacity, w, nullptr) ? OCGS_OK : OCGS_ERR_UNSUPPORTED;
}

int ocgs_render_fwd_reg(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                        float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg,
                        uint32_t* vis_count, float* contrib_sum, float* moments, void* stream) {
  if (!cam || !ws || !color || !alpha || !depth || !normal || !n_contrib) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if ((vis_count == nullptr) != (contrib_sum == nullptr)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if ((rc = carve_for_render(ws, n, cam, key_capacity, &w)) != OCGS_OK) return rc;
  return launch_render_fwd(make_cam(*cam), *cfg, w, mask, color, alpha, depth, normal, n_contrib, loss_bg, vis_count, contrib_sum,
                           moments, /*prim=*/0, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int ocgs3d_preprocess(const ocgs_gaussians3d* g, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, void* stream) {
  if (!g || !cam || !ws) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if (g->n > 0 && (!g->pos || !g->scale || !g->quat || !g->opacity || !g->sh)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, g->n, cam->width, cam->height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  return launch_preprocess3d(*g, make_cam(*cam), *cfg, w, (cudaStream_t)stream);
}

int ocgs3d_render_fwd(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                      float* color, float* alpha, float* depth, uint32_t* n_contrib, float* loss_bg, uint32_t* vis_count,
                      float* contrib_sum, void* stream) {
  if (!cam || !ws || !color || !alpha || !depth || !n_contrib) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if ((vis_count == nullptr) != (contrib_sum == nullptr)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if ((rc = carve_for_render(ws, n, cam, key_capacity, &w)) != OCGS_OK) return rc;
  return launch_render_fwd(make_cam(*cam), *cfg, w, mask, color, alpha, depth, /*normal=*/nullptr, n_contrib, loss_bg, vis_count, contrib_sum,
                           nullptr, /*prim=*/1, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int ocgs_visibility_pass(const ocgs_surfels* s, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                         uint32_t* vis_count, float* contrib_sum, void* stream) {
  if (!s || !cam || !ws || !vis_count || !contrib_sum) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if (s->n > 0 && (!s->pos || !s->scale || !s->quat || !s->opacity)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, s->n, cam->width, cam->height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  const CamParams cp = make_cam(*cam);
  if ((rc = launch_preprocess(*s, cp, *cfg, w, (cudaStream_t)stream, /*colour=*/false)) != OCGS_OK) return rc;
  if ((rc = launch_bin_sort(cp, w, nullptr, (cudaStream_t)stream)) != OCGS_OK) return rc;
  return launch_render_stats(cp, *cfg, w, vis_count, contrib_sum, /*prim=*/0, (cudaStream_t)stream);
}

int ocgs3d_visibility_pass(const ocgs_gaussians3d* g, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                           uint32_t* vis_count, float* contrib_sum, void* stream) {
  if (!g || !cam || !ws || !vis_count || !contrib_sum) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if (g->n > 0 && (!g->pos || !g->scale || !g->quat || !g->opacity || !g->sh)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, g->n, cam->width, cam->height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  const CamParams cp = make_cam(*cam);
  if ((rc = launch_preprocess3d(*g, cp, *cfg, w, (cudaStream_t)stream)) != OCGS_OK) return rc;
  if ((rc = launch_bin_sort(cp, w, nullptr, (cudaStream_t)stream)) != OCGS_OK) return rc;
  return launch_render_stats(cp, *cfg, w, vis_count, contrib_sum, /*prim=*/1, (cudaStream_t)stream);
}

int ocgs_render_fwd_l1(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                       const float* target, float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg,
                       float* loss_l1, float* dL_dcolor, uint32_t* vis_count, float* contrib_sum, void* stream) {
  if (!cam || !ws || !color || !alpha || !depth || !normal || !n_contrib || !target || !dL_dcolor) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if ((vis_count == nullptr) != (contrib_sum == nullptr)) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if ((rc = carve_for_render(ws, n, cam, key_capacity, &w)) != OCGS_OK) return rc;
  if (w.n_tiles == 0 || n == 0) {  // nothing to rasterise: the plain calls define the outputs
    if ((rc = ocgs_render_fwd(n, cam, cfg, ws, key_capacity, mask, color, alpha, depth, normal, n_contrib, loss_bg, vis_count, contrib_sum, stream)) != OCGS_OK) return rc;
    return ocgs_masked_l1(color, target, mask, cam->width, cam->height, dL_dcolor, loss_l1, ws, n, key_capacity, stream);
  }
  return launch_render_fwd(make_cam(*cam), *cfg, w, mask, color, alpha, depth, normal, n_contrib, loss_bg, vis_count, contrib_sum, nullptr,
                           /*prim=*/0, target, dL_dcolor, loss_l1, (cudaStream_t)stream);
}

int ocgs_render_fwd(int n, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity, const uint8_t* mask,
                        float* color, float* alpha, float* depth, float* normal, uint32_t* n_contrib, float* loss_bg,
                        uint32_t* vis_count, float* contrib_sum, void* stream) {
  return ocgs_render_fwd_reg(n, cam, cfg, ws, key_capacity, mask, color, alpha, depth, normal, n_contrib, loss_bg, vis_count,
                             contrib_sum, nullptr, stream);
}

int ocgs_render_bwd_reg(const ocgs_surfels* s, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                        const uint8_t* mask, const uint32_t* n_contrib, const float* gC, const float* gA, const float* gD,
                        const float* gN, const float* moments, const float* gM, float* d_pos, float* d_scale, float* d_quat,
                        float* d_opacity, float* d_sh, float* d_center2d, void* stream) {
  if (!s || !cam || !ws || !n_contrib) return OCGS_ERR_INVALID_ARG;
  int rc = check_cfg(cfg);
  if (rc != OCGS_OK) return rc;
  if (s->n > 0 && (!d_pos || !d_scale || !d_quat || !d_opacity || !d_sh)) return OCGS_ERR_INVALID_ARG;
  if ((gM != nullptr) != (moments != nullptr)) return OCGS_ERR_INVALID_ARG;
  const float* gM1 = gM;
  const float* gM2 = gM ? gM + (size_t)cam->width * cam->height : nullptr;
  Workspace w;
  if ((rc = carve_for_render(ws, s->n, cam, key_capacity, &w)) != OCGS_OK) return rc;
  return launch_render_bwd(*s, make_cam(*cam), *cfg, w, mask, w.final_T, n_contrib, gC, gA, gD, gN, moments, gM1, gM2, d_pos, d_scale, d_quat,
                           d_opacity, d_sh, d_center2d, (cudaStream_t)stream);
}

int ocgs_render_bwd(const ocgs_surfels* s, const ocgs_camera* cam, const ocgs_config* cfg, void* ws, size_t key_capacity,
                        const uint8_t* mask, const uint32_t* n_contrib, const float* gC, const float* gA, const float* gD,
                        const float* gN, float* d_pos, float* d_scale, float* d_quat, float* d_opacity, float* d_sh,
                        float* d_center2d, void* stream) {
  return ocgs_render_bwd_reg(s, cam, cfg, ws, key_capacity, mask, n_contrib, gC, gA, gD, gN, nullptr, nullptr, d_pos, d_scale, d_quat, d_opacity,
                             d_sh, d_center2d, stream);
}

int ocgs_masked_l1(const float* color, const float* target, const uint8_t* mask, int width, int height, float* dL_dcolor, float* loss,
                   void* ws, int n, size_t key_capacity, void* stream) {
  if (!color || !target || !dL_dcolor || !ws) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, n, width, height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  return launch_masked_l1(color, target, mask, width, height, dL_dcolor, loss, w.loss_partial, w.n_tiles, (cudaStream_t)stream);
}

size_t ocgs_regularizers_workspace_bytes(int width, int height) { return regularizers_workspace_bytes(width, height); }

int ocgs_regularizers(const float* alpha, const float* depth, const float* moments, const float* normal, const ocgs_camera* cam, float w_d,
                      float w_n, float* dL_dalpha, float* dL_ddepth, float* dL_dmoments, float* dL_dnormal, float* loss, void* scratch,
                      void* stream) {
  if (!alpha || !depth || !moments || !normal || !cam || !dL_dalpha || !dL_ddepth || !dL_dmoments || !dL_dnormal || !scratch)
    return OCGS_ERR_INVALID_ARG;
  if (cam->width <= 0 || cam->height <= 0 || !(cam->fx > 0.f) || !(cam->fy > 0.f)) return OCGS_ERR_INVALID_ARG;
  if (cam->width > OCGS_MAX_DIM || cam->height > OCGS_MAX_DIM) return OCGS_ERR_UNSUPPORTED;
  return launch_regularizers(alpha, depth, moments, normal, *cam, w_d, w_n, dL_dalpha, dL_ddepth, dL_dmoments, dL_dnormal, loss, scratch,
                             (cudaStream_t)stream);
}

size_t ocgs_photometric_workspace_bytes(int width, int height) { return photometric_workspace_bytes(width, height); }

int ocgs_photometric_loss(const float* color, const float* target, const uint8_t* mask, int width, int height, float lambda_dssim,
                          float* dL_dcolor, float* loss, void* scratch, void* stream) {
  if (!color || !target || !dL_dcolor || !scratch || width <= 0 || height <= 0) return OCGS_ERR_INVALID_ARG;
  if (!(lambda_dssim >= 0.f && lambda_dssim <= 1.f)) return OCGS_ERR_INVALID_ARG;
  if (width > OCGS_MAX_DIM || height > OCGS_MAX_DIM) return OCGS_ERR_UNSUPPORTED;
  return launch_photometric(color, target, mask, width, height, lambda_dssim, dL_dcolor, loss, scratch, (cudaStream_t)stream);
}

int ocgs_profile_begin(int capacity, void* stream) {
  if (capacity <= 0) return OCGS_ERR_INVALID_ARG;
  while ((int)g_prof.ev.size() < capacity + 1) {
    cudaEvent_t e;
    OCGS_CUDA_OK(cudaEventCreate(&e));
    g_prof.ev.push_back(e);
    g_prof.names.push_back("");
  }
  g_prof.used = 0;
  g_prof_on = true;
  prof_mark((cudaStream_t)stream, "begin");
  return OCGS_OK;
}

int ocgs_profile_end(void* stream, int max_out, float* ms_out, char* names_out, int* count) {
  g_prof_on = false;
  OCGS_CUDA_OK(cudaStreamSynchronize((cudaStream_t)stream));
  int c = 0;
  for (size_t i = 1; i < g_prof.used && c < max_out; ++i, ++c) {
    float ms = 0.f;
    OCGS_CUDA_OK(cudaEventElapsedTime(&ms, g_prof.ev[i - 1], g_prof.ev[i]));
    ms_out[c] = ms;
    strncpy(names_out + (size_t)c * 32, g_prof.names[i], 31);
    names_out[(size_t)c * 32 + 31] = 0;
  }
  if (count) *count = c;
  return OCGS_OK;
}

size_t ocgs_prune_workspace_bytes(int n) { return (div_up((size_t)(n > 0 ? n : 0), 1024) + 2) * sizeof(uint32_t); }

int ocgs_prune_stats(const ocgs_surfels* in, uint32_t* vis_count, float* contrib_sum, const ocgs_config* cfg, uint8_t* prune_mask,
                     int32_t* remap, const ocgs_surfels_mut* out, int* n_out, int reset_stats, void* ws, void* stream) {
  if (!in || !vis_count || !contrib_sum || !cfg || !prune_mask || !remap || !n_out || !ws) return OCGS_ERR_INVALID_ARG;
  if (out && out->capacity < in->n) return OCGS_ERR_CAPACITY;
  return launch_prune(*in, vis_count, contrib_sum, *cfg, prune_mask, remap, out, n_out, reset_stats, ws, (cudaStream_t)stream);
}

size_t ocgs_densify_workspace_bytes(int n) { return densify_workspace_bytes(n); }

int ocgs_densify_accumulate(void* ws, int n, int width, int height, size_t key_capacity, const float* d_center2d, float* grad_accum,
                            uint32_t* denom, void* stream) {
  if (!ws || (n > 0 && (!d_center2d || !grad_accum || !denom))) return OCGS_ERR_INVALID_ARG;
  Workspace w;
  if (!carve_workspace(ws, n, width, height, key_capacity, &w, nullptr)) return OCGS_ERR_UNSUPPORTED;
  return launch_densify_accumulate(w, d_center2d, grad_accum, denom, (cudaStream_t)stream);
}

int ocgs_densify(const ocgs_surfels* in, const float* grad_accum, const uint32_t* denom, float grad_threshold, float scale_threshold,
                 const float* xi, const ocgs_surfels_mut* out, int32_t* src, int* counts, void* ws, void* stream) {
  if (!in || !out || !counts || !ws) return OCGS_ERR_INVALID_ARG;
  if (in->n > 0 && (!grad_accum || !denom || !xi || !in->pos || !in->scale || !in->quat || !in->opacity || !in->sh || !out->pos ||
                    !out->scale || !out->quat || !out->opacity || !out->sh)) return OCGS_ERR_INVALID_ARG;
  if (out->capacity < in->n) return OCGS_ERR_CAPACITY;
  return launch_densify(*in, grad_accum, denom, grad_threshold, scale_threshold, xi, *out, src, counts, ws, (cudaStream_t)stream);
}

int ocgs_compact_rows(const float* in, const int32_t* remap, int n, int row_floats, float* out, void* stream) {
  if (n < 0 || row_floats <= 0) return OCGS_ERR_INVALID_ARG;
  if (n > 0 && (!in || !remap || !out || in == out)) return OCGS_ERR_INVALID_ARG;
  return launch_compact_rows(in, remap, n, row_floats, out, (cudaStream_t)stream);
}

int ocgs_step_view_host(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask,
                        const float* h_target, float* h_losses, uint8_t* d_mask, float* d_images, uint32_t* d_ncontrib,
                        float* d_grad_pos, float* d_grad_scale, float* d_grad_quat, float* d_grad_opacity, float* d_grad_sh,
                        uint32_t* d_vis_count, float* d_contrib_sum, float* d_losses, void* ws, size_t key_capacity, void* stream,
                        void* copy_stream) {
  int rc = ocgs_step_view_host_enqueue(surfels, cam, cfg, h_mask, h_target, h_losses, nullptr, d_mask, d_images, d_ncontrib, d_grad_pos,
                                       d_grad_scale, d_grad_quat, d_grad_opacity, d_grad_sh, d_vis_count, d_contrib_sum, d_losses, ws,
                                       key_capacity, stream, copy_stream);
  if (rc != OCGS_OK) { cudaStreamSynchronize((cudaStream_t)stream); return rc; }
  return ocgs_check(ws, stream, nullptr);
}

int ocgs_step_view_host_enqueue(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask,
                                const float* h_target, float* h_losses, ocgs_header* h_header, uint8_t* d_mask, float* d_images,
                                uint32_t* d_ncontrib, float* d_grad_pos, float* d_grad_scale, float* d_grad_quat, float* d_grad_opacity,
                                float* d_grad_sh, uint32_t* d_vis_count, float* d_contrib_sum, float* d_losses, void* ws,
                                size_t key_capacity, void* stream, void* copy_stream) {
  if (!surfels || !cam || !cfg || !h_mask || !h_target || !h_losses || !d_mask || !d_images || !d_ncontrib || !d_losses || !ws)
    return OCGS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  cudaStream_t cs = copy_stream ? (cudaStream_t)copy_stream : st;
  const size_t HW = (size_t)cam->width * cam->height;
  float* color = d_images; float* alpha = color + 3 * HW; float* depth = alpha + HW; float* normal = depth + HW;
  float* target = normal + 3 * HW;
  float* gC = target + 3 * HW;
  // the view's inputs travel on the copy stream while preprocess / sort / forward run: the mask is needed by the forward
  // pass, the target only by the photometric term
  cudaEvent_t ev_begin = nullptr, ev_mask = nullptr, ev_target = nullptr;
  const bool overlap = cs != st;
  bool forked = false;  // the copy stream has been made to depend on `st` (inside a capture: it has joined the capture)
  const int n = surfels->n;
  int rc = OCGS_OK;
#define OCGS_STEP_OK(expr) { const cudaError_t _e = (expr); if (_e != cudaSuccess) { rc = cuda_fail(_e); break; } }
  do {
    if (overlap) {
      OCGS_STEP_OK(cudaEventCreateWithFlags(&ev_begin, cudaEventDisableTiming));
      OCGS_STEP_OK(cudaEventCreateWithFlags(&ev_mask, cudaEventDisableTiming));
      OCGS_STEP_OK(cudaEventCreateWithFlags(&ev_target, cudaEventDisableTiming));
      OCGS_STEP_OK(cudaEventRecord(ev_begin, st));  // the previous step's readers of d_mask / target are done
      OCGS_STEP_OK(cudaStreamWaitEvent(cs, ev_begin, 0));
      forked = true;
    }
    OCGS_STEP_OK(cudaMemcpyAsync(d_mask, h_mask, HW, cudaMemcpyHostToDevice, cs));
    if (overlap) OCGS_STEP_OK(cudaEventRecord(ev_mask, cs));
    OCGS_STEP_OK(cudaMemcpyAsync(target, h_target, 3 * HW * sizeof(float), cudaMemcpyHostToDevice, cs));
    if (overlap) OCGS_STEP_OK(cudaEventRecord(ev_target, cs));
    if ((rc = ocgs_preprocess(surfels, cam, cfg, ws, key_capacity, stream)) != OCGS_OK) break;
    if ((rc = ocgs_bin_sort(n, cam, cfg, ws, key_capacity, nullptr, stream)) != OCGS_OK) break;
    if (overlap && cudaStreamWaitEvent(st, ev_mask, 0) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
    // (the fused ocgs_render_fwd_l1 would need the target before the forward pass: here the 23 MB upload is still in
    // flight then, so the forward runs unfused and only the L1 kernel waits for it -- measured 2.46 vs 2.63 ms)
    if ((rc = ocgs_render_fwd(n, cam, cfg, ws, key_capacity, d_mask, color, alpha, depth, normal, d_ncontrib, d_losses, d_vis_count,
                              d_contrib_sum, stream)) != OCGS_OK) break;
    if (overlap && cudaStreamWaitEvent(st, ev_target, 0) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
    if ((rc = ocgs_masked_l1(color, target, d_mask, cam->width, cam->height, gC, d_losses + 1, ws, n, key_capacity, stream)) != OCGS_OK) break;
    if ((rc = ocgs_render_bwd(surfels, cam, cfg, ws, key_capacity, d_mask, d_ncontrib, gC, nullptr, nullptr, nullptr, d_grad_pos, d_grad_scale,
                              d_grad_quat, d_grad_opacity, d_grad_sh, nullptr, stream)) != OCGS_OK) break;
    if (cudaMemcpyAsync(h_losses, d_losses, 2 * sizeof(float), cudaMemcpyDeviceToHost, st) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
    if (h_header && cudaMemcpyAsync(h_header, ws, sizeof(ocgs_header), cudaMemcpyDeviceToHost, st) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
  } while (false);
  // every exit goes through here: a failed call must not leave the copy stream dangling off a capture or racing the caller's
  // buffers (join it back into `st` with a fresh record), and the events are always destroyed
  if (forked && rc != OCGS_OK && ev_target && cudaEventRecord(ev_target, cs) == cudaSuccess) cudaStreamWaitEvent(st, ev_target, 0);
  if (ev_begin) cudaEventDestroy(ev_begin);
  if (ev_mask) cudaEventDestroy(ev_mask);
  if (ev_target) cudaEventDestroy(ev_target);
  return rc;
}

int ocgs_step_view_prefetch_enqueue(const ocgs_surfels* surfels, const ocgs_camera* cam, const ocgs_config* cfg,
                                    const uint8_t* h_next_mask, const float* h_next_target, float* h_losses, ocgs_header* h_header,
                                    const uint8_t* d_mask_cur, const float* d_target_cur, uint8_t* d_mask_next, float* d_target_next,
                                    float* d_images, uint32_t* d_ncontrib, float* d_grad_pos, float* d_grad_scale, float* d_grad_quat,
                                    float* d_grad_opacity, float* d_grad_sh, uint32_t* d_vis_count, float* d_contrib_sum,
                                    float* d_losses, void* ws, size_t key_capacity, void* stream, void* copy_stream) {
  if (!surfels || !cam || !cfg || !h_losses || !d_mask_cur || !d_target_cur || !d_images || !d_ncontrib || !d_losses || !ws)
    return OCGS_ERR_INVALID_ARG;
  const bool prefetch = h_next_mask != nullptr || h_next_target != nullptr;
  if (prefetch && (!h_next_mask || !h_next_target || !d_mask_next || !d_target_next)) return OCGS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  cudaStream_t cs = copy_stream ? (cudaStream_t)copy_stream : st;
  const size_t HW = (size_t)cam->width * cam->height;
  float* color = d_images; float* alpha = color + 3 * HW; float* depth = alpha + HW; float* normal = depth + HW;
  float* gC = normal + 3 * HW;
  cudaEvent_t ev_begin = nullptr, ev_done = nullptr;
  const bool fork = prefetch && cs != st;
  bool forked = false, done_recorded = false;
  const int n = surfels->n;
  int rc = OCGS_OK;
  do {
    if (prefetch) {
      if (fork) {
        OCGS_STEP_OK(cudaEventCreateWithFlags(&ev_begin, cudaEventDisableTiming));
        OCGS_STEP_OK(cudaEventCreateWithFlags(&ev_done, cudaEventDisableTiming));
        OCGS_STEP_OK(cudaEventRecord(ev_begin, st));  // the step that last read d_*_next has finished
        OCGS_STEP_OK(cudaStreamWaitEvent(cs, ev_begin, 0));
        forked = true;
      }
      OCGS_STEP_OK(cudaMemcpyAsync(d_mask_next, h_next_mask, HW, cudaMemcpyHostToDevice, cs));
      OCGS_STEP_OK(cudaMemcpyAsync(d_target_next, h_next_target, 3 * HW * sizeof(float), cudaMemcpyHostToDevice, cs));
      if (fork) { OCGS_STEP_OK(cudaEventRecord(ev_done, cs)); done_recorded = true; }
    }
    if ((rc = ocgs_preprocess(surfels, cam, cfg, ws, key_capacity, stream)) != OCGS_OK) break;
    if ((rc = ocgs_bin_sort(n, cam, cfg, ws, key_capacity, nullptr, stream)) != OCGS_OK) break;
    if ((rc = ocgs_render_fwd_l1(n, cam, cfg, ws, key_capacity, d_mask_cur, d_target_cur, color, alpha, depth, normal, d_ncontrib, d_losses,
                                 d_losses + 1, gC, d_vis_count, d_contrib_sum, stream)) != OCGS_OK) break;
    if ((rc = ocgs_render_bwd(surfels, cam, cfg, ws, key_capacity, d_mask_cur, d_ncontrib, gC, nullptr, nullptr, nullptr, d_grad_pos, d_grad_scale,
                              d_grad_quat, d_grad_opacity, d_grad_sh, nullptr, stream)) != OCGS_OK) break;
    if (cudaMemcpyAsync(h_losses, d_losses, 2 * sizeof(float), cudaMemcpyDeviceToHost, st) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
    if (h_header && cudaMemcpyAsync(h_header, ws, sizeof(ocgs_header), cudaMemcpyDeviceToHost, st) != cudaSuccess) { rc = OCGS_ERR_CUDA; break; }
  } while (false);
  // every exit goes through here.  join: the next call (and the end of a capture) sees the prefetch finished; after a failure
  // in between, whatever the copy stream got is joined with a fresh record
  if (forked && ev_done && (done_recorded || cudaEventRecord(ev_done, cs) == cudaSuccess)) cudaStreamWaitEvent(st, ev_done, 0);
  if (ev_begin) cudaEventDestroy(ev_begin);
  if (ev_done) cudaEventDestroy(ev_done);
  return rc;
}
#undef OCGS_STEP_OK

int ocgs_step_host(const float* h_pos, const float* h_scale, const float* h_quat, const float* h_opacity, const float* h_sh, int n,
                   const ocgs_camera* cam, const ocgs_config* cfg, const uint8_t* h_mask, const float* h_target, float* h_grads,
                   float* h_alpha, float* h_loss_bg, float* d_params, uint8_t* d_mask, float* d_images, uint32_t* d_ncontrib,
                   float* d_grads, uint32_t* d_vis_count, float* d_contrib_sum, float* d_loss_bg, void* ws, size_t key_capacity,
                   void* stream) {
  if (!cam || !cfg || !ws || !d_params || !d_mask || !d_images || !d_ncontrib || !d_grads || !d_loss_bg) return OCGS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t N = (size_t)n, HW = (size_t)cam->width * cam->height;
  float* p_pos = d_params;               // 3N
  float* p_scale = p_pos + 3 * N;         // 2N   (3N*4 bytes is 8-aligned only when N is even: keep sections 16-B aligned)
  // section starts rounded up to 4 floats so float2/float4 loads stay aligned
  auto up4 = [](size_t x) { return (x + 3) & ~(size_t)3; };
  p_scale = d_params + up4(3 * N);
  float* p_quat = p_scale + up4(2 * N);
  float* p_opa = p_quat + 4 * N;
  float* p_sh = p_opa + up4(N);
  OCGS_CUDA_OK(cudaMemcpyAsync(p_pos, h_pos, 3 * N * 4, cudaMemcpyHostToDevice, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(p_scale, h_scale, 2 * N * 4, cudaMemcpyHostToDevice, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(p_quat, h_quat, 4 * N * 4, cudaMemcpyHostToDevice, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(p_opa, h_opacity, N * 4, cudaMemcpyHostToDevice, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(p_sh, h_sh, 48 * N * 4, cudaMemcpyHostToDevice, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(d_mask, h_mask, HW, cudaMemcpyHostToDevice, st));
  float* color = d_images; float* alpha = color + 3 * HW; float* depth = alpha + HW; float* normal = depth + HW;
  float* target = normal + 3 * HW;
  float* gC = target + 3 * HW;
  OCGS_CUDA_OK(cudaMemcpyAsync(target, h_target, 3 * HW * 4, cudaMemcpyHostToDevice, st));
  ocgs_surfels s = {p_pos, p_scale, p_quat, p_opa, p_sh, n};
  int rc;
  if ((rc = ocgs_preprocess(&s, cam, cfg, ws, key_capacity, stream)) != OCGS_OK) return rc;
  if ((rc = ocgs_bin_sort(n, cam, cfg, ws, key_capacity, nullptr, stream)) != OCGS_OK) return rc;
  if ((rc = ocgs_render_fwd(n, cam, cfg, ws, key_capacity, d_mask, color, alpha, depth, normal, d_ncontrib, d_loss_bg, d_vis_count,
                            d_contrib_sum, stream)) != OCGS_OK) return rc;
  if ((rc = ocgs_masked_l1(color, target, d_mask, cam->width, cam->height, gC, nullptr, ws, n, key_capacity, stream)) != OCGS_OK) return rc;
  float* g_pos = d_grads; float* g_scale = d_grads + up4(3 * N); float* g_quat = g_scale + up4(2 * N); float* g_opa = g_quat + 4 * N;
  float* g_sh = g_opa + up4(N);
  if ((rc = ocgs_render_bwd(&s, cam, cfg, ws, key_capacity, d_mask, d_ncontrib, gC, nullptr, nullptr, nullptr, g_pos, g_scale, g_quat,
                            g_opa, g_sh, nullptr, stream)) != OCGS_OK) return rc;
  OCGS_CUDA_OK(cudaMemcpyAsync(h_grads, g_pos, 3 * N * 4, cudaMemcpyDeviceToHost, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(h_grads + 3 * N, g_scale, 2 * N * 4, cudaMemcpyDeviceToHost, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(h_grads + 5 * N, g_quat, 4 * N * 4, cudaMemcpyDeviceToHost, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(h_grads + 9 * N, g_opa, N * 4, cudaMemcpyDeviceToHost, st));
  OCGS_CUDA_OK(cudaMemcpyAsync(h_grads + 10 * N, g_sh, 48 * N * 4, cudaMemcpyDeviceToHost, st));
  if (h_alpha) OCGS_CUDA_OK(cudaMemcpyAsync(h_alpha, alpha, HW * 4, cudaMemcpyDeviceToHost, st));
  if (h_loss_bg) OCGS_CUDA_OK(cudaMemcpyAsync(h_loss_bg, d_loss_bg, 4, cudaMemcpyDeviceToHost, st));
  return ocgs_check(ws, stream, nullptr);
}

}  // extern "C"
