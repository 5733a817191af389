// api.cu -- the C ABI of include/splx.h: argument validation and stage sequencing only; every
// step of the path runs in the kernels of project.cu / sort.cu / render.cu / compose.cu / adam.cu.
#include "common.cuh"

static char g_create_err[512] = "";

// near_z must be positive: with z <= 0 admitted 1/z blows up in J and float_bits(depth) no longer sorts as an unsigned key
static bool cam_ok(const splx_camera* c) {
  if (!c || c->width <= 0 || c->height <= 0) return false;
  const float f[5] = {c->fx, c->fy, c->cx, c->cy, c->near_z};
  for (float x : f) if (!(x == x) || x - x != 0.f) return false;      // NaN or infinity
  for (int i = 0; i < 9; ++i) if (!(c->R[i] - c->R[i] == 0.f)) return false;
  for (int i = 0; i < 3; ++i) if (!(c->t[i] - c->t[i] == 0.f)) return false;
  return c->fx > 0.f && c->fy > 0.f && c->near_z > 0.f;
}
static bool proj_ok(const splx_projected* p) {
  return p && p->means2d && p->depth && p->conic_opacity && p->rgb && p->radius && p->tiles_touched &&
         p->clamp && p->blend && aligned16(p->means2d) && aligned16(p->conic_opacity) && aligned16(p->blend);
}
static bool gauss_ok(const splx_gaussians* g) {
  return g && g->n >= 0 && (g->n == 0 || (g->mean && g->log_scale && g->quat && g->opacity_logit && g->sh &&
                                          aligned16(g->quat) && aligned16(g->sh)));
}
static bool partial_ok(const splx_partial* p) {
  return p && p->ct && p->d && p->n_contrib && aligned16(p->ct);
}
static bool bins_ok(const splx_binning* b) {
  return b && b->keys && b->vals && b->tile_ranges && b->num_intersections && aligned16(b->keys);
}

// ---- launch plans ---------------------------------------------------------------------------
// Validates a splx_plan against K and builds the device-side copy.  All views must share one image size.
int make_plan_dev(splx_ctx* ctx, const char* who, int K, const splx_plan* plan, PlanDev* out) {
  if (!plan || !plan->cams || !plan->view_of_part) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: plan, cams or view_of_part is NULL", who);
  if (K < 1 || K > SPLX_MAX_K) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: K=%d not in [1,%d]", who, K, SPLX_MAX_K);
  if (plan->n_views < 1 || plan->n_views > SPLX_MAX_VIEWS)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: n_views=%d not in [1,%d]", who, plan->n_views, SPLX_MAX_VIEWS);
  if (plan->flags & ~SPLX_PLAN_SPARSE) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: unknown plan flags %d", who, plan->flags);
  memset(out, 0, sizeof *out);
  for (int b = 0; b < plan->n_views; ++b) {
    if (!cam_ok(&plan->cams[b])) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: camera %d invalid", who, b);
    if (plan->cams[b].width != plan->cams[0].width || plan->cams[b].height != plan->cams[0].height)
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: all views of a plan must have the same size", who);
    out->cam[b] = make_camdev(&plan->cams[b], ctx->cfg);
  }
  for (int k = 0; k < K; ++k) {
    const int v = plan->view_of_part[k];
    if (v < -1 || v >= plan->n_views) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: view_of_part[%d]=%d out of range", who, k, v);
    out->pv.v[k] = (signed char)v;
  }
  for (int k = K; k < SPLX_MAX_K; ++k) out->pv.v[k] = -1;
  for (int k = 0; k < SPLX_MAX_K; ++k) {
    out->max_scale[k] = (plan->max_scale && k < K) ? plan->max_scale[k] : -1.0f;
    if (plan->max_scale && k < K && !(plan->max_scale[k] >= 0.f)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: max_scale[%d] must be >= 0", who, k);
  }
  out->B = plan->n_views; out->K = K;
  out->W = out->cam[0].W; out->H = out->cam[0].H; out->TX = out->cam[0].TX; out->TY = out->cam[0].TY;
  out->ntiles = out->TX * out->TY;
  out->flags = plan->flags;
  out->tile_state = plan->tile_state;
  if (plan->open_slots != 0 && !plan->tile_state) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: open_slots without tile_state", who);
  if (plan->slot_map && (plan->open_slots == 0 || !aligned16(plan->slot_map)))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "%s: slot_map without open_slots, or misaligned", who);
  out->slot_map = plan->slot_map;
  out->open_slots = (uint32_t)(plan->open_slots < 0 ? -(int64_t)plan->open_slots : (int64_t)plan->open_slots);
  out->open_forced = plan->open_slots < 0;
  return SPLX_OK;
}

static bool offsets_ok(const int64_t* po, int K, int64_t n) {
  if (!po || po[0] != 0 || po[K] != n) return false;
  for (int k = 0; k < K; ++k) if (po[k + 1] < po[k]) return false;
  return true;
}

// One view, every partition renders it: the plan behind the single-view calls.
struct SinglePlan {
  int32_t views[SPLX_MAX_K];
  splx_plan plan;
  explicit SinglePlan(const splx_camera* cam) {
    for (int k = 0; k < SPLX_MAX_K; ++k) views[k] = 0;
    plan.n_views = 1; plan.cams = cam; plan.view_of_part = views; plan.tile_state = nullptr; plan.flags = 0;
    plan.max_scale = nullptr; plan.open_slots = 0; plan.slot_map = nullptr;
  }
};

extern "C" {

int splx_create(splx_ctx** out, int device, void* cuda_stream, const splx_config* cfg) {
  if (!out) { snprintf(g_create_err, sizeof g_create_err, "splx_create: out is NULL"); return SPLX_ERR_INVALID_ARG; }
  *out = nullptr;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= 0) {
    snprintf(g_create_err, sizeof g_create_err, "splx_create: no CUDA device (%s); there is no CPU fallback",
             e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    return SPLX_ERR_CUDA;
  }
  if (device < 0 || device >= ndev) {
    snprintf(g_create_err, sizeof g_create_err, "splx_create: device %d out of range [0,%d)", device, ndev);
    return SPLX_ERR_INVALID_ARG;
  }
  if ((e = cudaSetDevice(device)) != cudaSuccess) {
    snprintf(g_create_err, sizeof g_create_err, "cudaSetDevice: %s", cudaGetErrorString(e));
    return SPLX_ERR_CUDA;
  }
  splx_ctx* c = new splx_ctx();
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  c->launches = 0;
  c->err[0] = 0;
  c->iter_ready = false;
  if (cfg) c->cfg = *cfg;
  else c->cfg = splx_config{1.0f / 255.0f, 0.99f, 1e-4f, 0.3f, 1.3f, 0.1f};
  if (!(c->cfg.alpha_max > 0.f) || c->cfg.alpha_min < 0.f || c->cfg.T_eps < 0.f) {
    delete c;
    snprintf(g_create_err, sizeof g_create_err, "splx_create: bad config");
    return SPLX_ERR_INVALID_ARG;
  }
  *out = c;
  return SPLX_OK;
}

int splx_destroy(splx_ctx* ctx) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  iteration_release(ctx);
  delete ctx;
  return SPLX_OK;
}

const char* splx_last_error(const splx_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

int splx_set_stream(splx_ctx* ctx, void* cuda_stream) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  ctx->stream = (cudaStream_t)cuda_stream;
  return SPLX_OK;
}

int64_t splx_launch_count(const splx_ctx* ctx) { return ctx ? ctx->launches : -1; }

size_t splx_slot_map_words(int K, const splx_camera* cam) {
  if (!cam || cam->width <= 0 || cam->height <= 0 || K < 1 || K > SPLX_MAX_K) return 0;
  const size_t tiles = (size_t)((cam->width + SPLX_TILE - 1) / SPLX_TILE) * (size_t)((cam->height + SPLX_TILE - 1) / SPLX_TILE);
  return 2 * (size_t)K * tiles + 2;
}

int splx_slot_map(splx_ctx* ctx, int K, const splx_plan* plan, uint32_t* slot_map_out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!slot_map_out || !aligned16(slot_map_out)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_slot_map: slot_map_out null or misaligned");
  splx_plan p;
  if (plan) { p = *plan; p.slot_map = nullptr; }
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_slot_map", K, plan ? &p : nullptr, &pd))) return rc;
  if (!pd.tile_state || pd.open_slots == 0 || !aligned16(pd.tile_state))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_slot_map: the plan needs tile_state (16-byte aligned) and open_slots");
  return launch_slot_map(ctx, pd, slot_map_out);
}

int splx_project_plan(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets, const splx_plan* plan,
                      int sh_degree, const splx_projected* out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && g->n == 0) return SPLX_OK;   // empty scene: nothing to write
  if (!gauss_ok(g) || !proj_ok(out)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project: null/misaligned argument");
  if (sh_degree < 0 || sh_degree > 3) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project: sh_degree %d not in [0,3]", sh_degree);
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_project", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project: part_offsets must run monotonically from 0 to n");
  return launch_project_fwd(ctx, g, pd, part_offsets, sh_degree, out);
}

int splx_project_geometry_plan(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets, const splx_plan* plan,
                               const splx_projected* out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && g->n == 0) return SPLX_OK;
  if (!gauss_ok(g) || !proj_ok(out)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_geometry: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_project_geometry", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_geometry: part_offsets must run monotonically from 0 to n");
  return launch_project_fwd(ctx, g, pd, part_offsets, 0, out, false);
}

int splx_project_colour_list_plan(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets, const splx_plan* plan,
                                  int sh_degree, const splx_projected* out, const uint32_t* visible, const uint64_t* num_visible) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && g->n == 0) return SPLX_OK;
  if (!gauss_ok(g) || !proj_ok(out) || !visible || !num_visible)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_colour_list: null/misaligned argument");
  if (sh_degree < 0 || sh_degree > 3) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_colour_list: sh_degree %d not in [0,3]", sh_degree);
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_project_colour_list", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_colour_list: part_offsets must run monotonically from 0 to n");
  return launch_project_colour_list(ctx, g, pd, part_offsets, sh_degree, out, visible, num_visible);
}

int splx_project(splx_ctx* ctx, const splx_gaussians* g, const splx_camera* cam, int sh_degree,
                 const splx_projected* out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && g->n == 0) return SPLX_OK;
  if (!gauss_ok(g) || !cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project: null/misaligned argument");
  const SinglePlan sp(cam);
  const int64_t po[2] = {0, g->n};
  return splx_project_plan(ctx, g, 1, po, &sp.plan, sh_degree, out);
}

size_t splx_bin_sort_ws_bytes(int64_t n, uint64_t capacity, int K, const splx_camera* cam) {
  if (n < 0 || !cam_ok(cam) || K < 1) return 0;
  const int TX = (cam->width + SPLX_TILE - 1) / SPLX_TILE, TY = (cam->height + SPLX_TILE - 1) / SPLX_TILE;
  return bin_sort_ws_bytes(n, capacity, K, TX, TY);
}

int splx_bin_sort_plan(splx_ctx* ctx, const splx_projected* proj, int64_t n, int K, const int64_t* part_offsets,
                       const splx_plan* plan, const splx_binning* out, void* ws, size_t ws_bytes) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!proj_ok(proj) || !bins_ok(out) || n < 0 || (!ws && ws_bytes))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_bin_sort", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: part_offsets must run monotonically from 0 to n");
  if (n >= ((int64_t)1 << 32) || out->capacity >= ((uint64_t)1 << 32))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: n and capacity must be < 2^32");
  if ((uint64_t)K * pd.ntiles >= ((uint64_t)1 << 31)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: K*tiles too large");
  if (!aligned16(ws)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: workspace not 16-byte aligned");
  return launch_bin_sort(ctx, proj, n, pd, part_offsets, out, ws, ws_bytes);
}

int splx_bin_sort_filtered_plan(splx_ctx* ctx, const splx_projected* proj, int64_t n, int K, const int64_t* part_offsets,
                                const splx_plan* plan, const uint64_t* cross_mask, const float* part_depth_range,
                                const splx_binning* out, void* ws, size_t ws_bytes) {
  if (!cross_mask) return splx_bin_sort_plan(ctx, proj, n, K, part_offsets, plan, out, ws, ws_bytes);
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!proj_ok(proj) || !bins_ok(out) || n < 0 || (!ws && ws_bytes) || !part_depth_range)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_filtered: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_bin_sort_filtered", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_filtered: part_offsets must run monotonically from 0 to n");
  if (n >= ((int64_t)1 << 32) || out->capacity >= ((uint64_t)1 << 32))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_filtered: n and capacity must be < 2^32");
  if ((uint64_t)K * pd.ntiles >= ((uint64_t)1 << 31)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_filtered: K*tiles too large");
  if (!aligned16(ws)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_filtered: workspace not 16-byte aligned");
  CrossDev cd;
  memset(&cd, 0, sizeof cd);
  cd.mask = cross_mask;
  for (int k = 0; k < K; ++k) { cd.zlo[k] = part_depth_range[2 * k]; cd.zhi[k] = part_depth_range[2 * k + 1]; }
  return launch_bin_sort(ctx, proj, n, pd, part_offsets, out, ws, ws_bytes, &cd);
}

int splx_cross_sets(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets, const float* cell_lo,
                    const float* cell_hi, float support_sigma, uint64_t* cross_mask) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!g || g->n < 0 || !cell_lo || !cell_hi || (g->n > 0 && (!g->mean || !g->log_scale || !g->quat || !cross_mask)))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: null argument");
  if (K < 1 || K > SPLX_MAX_K) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: K=%d not in [1,%d]", K, SPLX_MAX_K);
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: part_offsets must run monotonically from 0 to n");
  if (!(support_sigma >= 0.f)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: support_sigma must be >= 0");
  if (((uintptr_t)g->quat & 15) || ((uintptr_t)cross_mask & 7)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: quat must be 16-byte, cross_mask 8-byte aligned");
  for (int k = 0; k < K; ++k)
    for (int a = 0; a < 3; ++a)
      if (!(cell_lo[3 * k + a] <= cell_hi[3 * k + a])) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_cross_sets: box %d has lo > hi", k);
  return launch_cross_sets(ctx, g, K, part_offsets, cell_lo, cell_hi, support_sigma, cross_mask);
}

int splx_bin_sort(splx_ctx* ctx, const splx_projected* proj, int64_t n, int K, const int64_t* part_offsets,
                  const splx_camera* cam, const splx_binning* out, void* ws, size_t ws_bytes) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: null/misaligned argument");
  const SinglePlan sp(cam);
  return splx_bin_sort_plan(ctx, proj, n, K, part_offsets, &sp.plan, out, ws, ws_bytes);
}

int splx_check_capacity(splx_ctx* ctx, const splx_binning* bins, uint64_t* m_host) {
  if (!ctx || !bins || !bins->num_intersections) return SPLX_ERR_INVALID_ARG;
  uint64_t m = 0;
  SPLX_CUDA_OK(ctx, cudaMemcpyAsync(&m, bins->num_intersections, sizeof m, cudaMemcpyDeviceToHost, ctx->stream));
  SPLX_CUDA_OK(ctx, cudaStreamSynchronize(ctx->stream));
  if (m_host) *m_host = m;
  if (m > bins->capacity)
    SPLX_FAIL(ctx, SPLX_ERR_CAPACITY, "splx_bin_sort: %llu intersections exceed capacity %llu",
              (unsigned long long)m, (unsigned long long)bins->capacity);
  return SPLX_OK;
}

int splx_render_partial_plan(splx_ctx* ctx, const splx_projected* proj, const splx_binning* bins, int K,
                             const splx_plan* plan, const splx_partial* out, uint64_t* pairs) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!proj_ok(proj) || !bins_ok(bins) || !partial_ok(out))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_render_partial: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_render_partial", K, plan, &pd))) return rc;
  return launch_render_fwd(ctx, proj, bins, pd, out, pairs);
}

int splx_render_partial(splx_ctx* ctx, const splx_projected* proj, const splx_binning* bins, int K,
                        const splx_camera* cam, const splx_partial* out, uint64_t* pairs) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_render_partial: null/misaligned argument");
  const SinglePlan sp(cam);
  return splx_render_partial_plan(ctx, proj, bins, K, &sp.plan, out, pairs);
}

int splx_compose_plan(splx_ctx* ctx, int K, const splx_partial* partials, const splx_binning* bins, const splx_plan* plan,
                      const float bg[3], float* image, float* T_total, float sat_eps, uint8_t* tile_state_out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!partial_ok(partials) || !bg || !image) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_compose", K, plan, &pd))) return rc;
  if ((pd.flags & SPLX_PLAN_SPARSE) && !bins_ok(bins))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose: SPLX_PLAN_SPARSE needs the binning");
  if (tile_state_out && !(sat_eps >= 0.f)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose: sat_eps must be >= 0");
  const ViewBufs vb = contiguous_views(pd.B, (size_t)pd.W * pd.H, nullptr, image, T_total, nullptr, nullptr);
  return launch_compose_fwd(ctx, partials, bins, pd, bg, vb, sat_eps, tile_state_out);
}

int splx_compose_l1_backward_plan(splx_ctx* ctx, int K, const splx_partial* partials, const splx_binning* bins,
                                  const splx_plan* plan, const float bg[3], const float* targets, float scale,
                                  float* image, float* T_total, double* loss_sum, float* g_ct, float sat_eps,
                                  uint8_t* tile_state_out) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!partial_ok(partials) || !bg || !image || !targets || !g_ct || !aligned16(g_ct))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_l1_backward: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_compose_l1_backward", K, plan, &pd))) return rc;
  if ((pd.flags & SPLX_PLAN_SPARSE) && !bins_ok(bins))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_l1_backward: SPLX_PLAN_SPARSE needs the binning");
  if (tile_state_out && !(sat_eps >= 0.f)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_l1_backward: sat_eps must be >= 0");
  const ViewBufs vb = contiguous_views(pd.B, (size_t)pd.W * pd.H, targets, image, T_total, nullptr, nullptr);
  return launch_compose_fused(ctx, partials, bins, pd, bg, vb, scale, loss_sum, g_ct, sat_eps, tile_state_out);
}

int splx_compose(splx_ctx* ctx, int K, const splx_partial* partials, const splx_camera* cam, const float bg[3],
                 float* image, float* T_total) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose: null/misaligned argument");
  const SinglePlan sp(cam);
  return splx_compose_plan(ctx, K, partials, nullptr, &sp.plan, bg, image, T_total, 0.f, nullptr);
}

int splx_l1_loss_grad(splx_ctx* ctx, const float* image, const float* target, int64_t count, float scale,
                      float* dL_dimage, double* loss_sum) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!image || !target || !dL_dimage || count < 0 || !aligned16(image) || !aligned16(target) || !aligned16(dL_dimage))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_l1_loss_grad: null/misaligned argument");
  return launch_l1(ctx, image, target, count, scale, dL_dimage, loss_sum);
}

int splx_compose_backward_plan(splx_ctx* ctx, int K, const splx_partial* partials, const splx_binning* bins,
                               const splx_plan* plan, const float bg[3], const float* dL_dimage,
                               const float* dL_dT_total, float* g_ct) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!partial_ok(partials) || !bg || !dL_dimage || !g_ct || !aligned16(g_ct))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_backward: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_compose_backward", K, plan, &pd))) return rc;
  if ((pd.flags & SPLX_PLAN_SPARSE) && !bins_ok(bins))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_backward: SPLX_PLAN_SPARSE needs the binning");
  const ViewBufs vb = contiguous_views(pd.B, (size_t)pd.W * pd.H, nullptr, nullptr, nullptr, const_cast<float*>(dL_dimage), dL_dT_total);
  return launch_compose_bwd(ctx, partials, bins, pd, bg, vb, g_ct);
}

int splx_compose_backward(splx_ctx* ctx, int K, const splx_partial* partials, const splx_camera* cam,
                          const float bg[3], const float* dL_dimage, const float* dL_dT_total, float* g_ct) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_compose_backward: null/misaligned argument");
  const SinglePlan sp(cam);
  return splx_compose_backward_plan(ctx, K, partials, nullptr, &sp.plan, bg, dL_dimage, dL_dT_total, g_ct);
}

int splx_raster_backward_plan(splx_ctx* ctx, const splx_projected* proj, const splx_binning* bins, int K,
                              const splx_plan* plan, const splx_partial* partials, const float* g_ct, float* g2d) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!proj_ok(proj) || !bins_ok(bins) || !partial_ok(partials) || !g_ct || !g2d || !aligned16(g_ct) || !aligned16(g2d))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_raster_backward: null/misaligned argument");
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_raster_backward", K, plan, &pd))) return rc;
  return launch_raster_bwd(ctx, proj, bins, pd, partials, g_ct, g2d);
}

int splx_raster_backward(splx_ctx* ctx, const splx_projected* proj, const splx_binning* bins, int K,
                         const splx_camera* cam, const splx_partial* partials, const float* g_ct, float* g2d) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_raster_backward: null/misaligned argument");
  const SinglePlan sp(cam);
  return splx_raster_backward_plan(ctx, proj, bins, K, &sp.plan, partials, g_ct, g2d);
}

int splx_project_backward_plan(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets,
                               const splx_plan* plan, int sh_degree, const splx_projected* proj, float* g2d, int flags,
                               const splx_gaussian_grads* grads) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && grads && g->n == 0 && grads->n == 0) return SPLX_OK;   // empty scene: nothing to write
  if (!gauss_ok(g) || !proj_ok(proj) || !g2d || !aligned16(g2d) || !grads || !grads->mean ||
      !grads->log_scale || !grads->quat || !grads->opacity_logit || !grads->sh || !aligned16(grads->quat) ||
      !aligned16(grads->mean) || !aligned16(grads->log_scale) || !aligned16(grads->sh) || !aligned16(grads->opacity_logit) ||
      grads->n != g->n)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward: null/misaligned argument");
  if (sh_degree < 0 || sh_degree > 3) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward: sh_degree %d not in [0,3]", sh_degree);
  if (flags & ~(SPLX_PB_CLEAR_G2D | SPLX_PB_OVERWRITE)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward: unknown flags %d", flags);
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_project_backward", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward: part_offsets must run monotonically from 0 to n");
  return launch_project_bwd(ctx, g, pd, part_offsets, sh_degree, proj, g2d, flags, grads, nullptr, nullptr, nullptr);
}

int splx_bin_sort_visible(const void* ws, int64_t n, uint64_t capacity, int K, const splx_camera* cam,
                          const uint32_t** visible, const uint64_t** num_visible) {
  if (!ws || n < 0 || K < 1 || K > SPLX_MAX_K || !cam_ok(cam) || !visible || !num_visible) return SPLX_ERR_INVALID_ARG;
  const int TX = (cam->width + SPLX_TILE - 1) / SPLX_TILE, TY = (cam->height + SPLX_TILE - 1) / SPLX_TILE;
  return bin_sort_visible(ws, n, capacity, K, TX, TY, visible, num_visible);
}

int splx_bin_sort_gradient_rows(splx_ctx* ctx, void* ws, int64_t n, uint64_t capacity, int K, const splx_camera* cam,
                                const float* g2d, const uint32_t** rows, const uint64_t** num_rows) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!ws || n < 0 || K < 1 || K > SPLX_MAX_K || !cam_ok(cam) || !g2d || !aligned16(g2d) || !rows || !num_rows)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort_gradient_rows: null/misaligned argument");
  *rows = nullptr; *num_rows = nullptr;
  if (n == 0) return SPLX_OK;
  const int TX = (cam->width + SPLX_TILE - 1) / SPLX_TILE, TY = (cam->height + SPLX_TILE - 1) / SPLX_TILE;
  return launch_gradient_rows(ctx, ws, n, capacity, K, TX, TY, g2d, rows, num_rows);
}

int splx_project_backward_list_plan(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets,
                                    const splx_plan* plan, int sh_degree, const splx_projected* proj, float* g2d, int flags,
                                    const splx_gaussian_grads* grads, const uint32_t* visible, const uint64_t* num_visible,
                                    uint8_t* touched) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!visible || !num_visible) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: visible list is NULL");
  if (flags & SPLX_PB_OVERWRITE) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: accumulates only (no SPLX_PB_OVERWRITE)");
  if (g && grads && g->n == 0 && grads->n == 0) return SPLX_OK;
  if (!gauss_ok(g) || !proj_ok(proj) || !g2d || !aligned16(g2d) || !grads || !grads->mean ||
      !grads->log_scale || !grads->quat || !grads->opacity_logit || !grads->sh || !aligned16(grads->quat) ||
      !aligned16(grads->mean) || !aligned16(grads->log_scale) || !aligned16(grads->sh) || !aligned16(grads->opacity_logit) ||
      grads->n != g->n)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: null/misaligned argument");
  if (sh_degree < 0 || sh_degree > 3) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: sh_degree %d not in [0,3]", sh_degree);
  if (flags & ~SPLX_PB_CLEAR_G2D) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: unknown flags %d", flags);
  PlanDev pd;
  int rc;
  if ((rc = make_plan_dev(ctx, "splx_project_backward_list", K, plan, &pd))) return rc;
  if (!offsets_ok(part_offsets, K, g->n)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward_list: part_offsets must run monotonically from 0 to n");
  return launch_project_bwd(ctx, g, pd, part_offsets, sh_degree, proj, g2d, flags, grads, visible, num_visible, touched);
}

int splx_project_backward(splx_ctx* ctx, const splx_gaussians* g, const splx_camera* cam, int sh_degree,
                          const splx_projected* proj, float* g2d, int flags, const splx_gaussian_grads* grads) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (g && grads && g->n == 0 && grads->n == 0) return SPLX_OK;
  if (!gauss_ok(g) || !cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_project_backward: null/misaligned argument");
  const SinglePlan sp(cam);
  const int64_t po[2] = {0, g->n};
  return splx_project_backward_plan(ctx, g, 1, po, &sp.plan, sh_degree, proj, g2d, flags, grads);
}

size_t splx_backward_ws_bytes(int64_t n, int K, const splx_camera* cam) {
  if (n < 0 || K < 1 || !cam_ok(cam)) return 0;
  const size_t g_ct = align_up((size_t)K * cam->width * cam->height * 4 * sizeof(float), 256);
  const size_t g2d = align_up((size_t)n * SPLX_G2D_STRIDE * sizeof(float), 256);
  return g_ct + g2d;
}

int splx_backward_plan(splx_ctx* ctx, int K, const int64_t* part_offsets, const splx_plan* plan,
                       const splx_partial* partials, const float bg[3], const float* dL_dimage,
                       const float* dL_dT_total, const splx_gaussians* g, const splx_projected* proj,
                       const splx_binning* bins, int sh_degree, const splx_gaussian_grads* grads, void* ws,
                       size_t ws_bytes, int flags) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (flags & ~SPLX_PB_OVERWRITE) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_backward: unknown flags %d", flags);
  if (!gauss_ok(g) || !plan || !plan->cams || plan->n_views < 1 || !cam_ok(&plan->cams[0]))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_backward: null/misaligned argument");
  const splx_camera* cam = &plan->cams[0];
  const size_t need = splx_backward_ws_bytes(g->n, K, cam);
  if (!ws || !aligned16(ws) || ws_bytes < need)
    SPLX_FAIL(ctx, SPLX_ERR_WORKSPACE, "splx_backward: workspace %zu B < required %zu B", ws_bytes, need);
  float* g_ct = (float*)ws;
  float* g2d = (float*)((char*)ws + align_up((size_t)K * cam->width * cam->height * 4 * sizeof(float), 256));
  int rc;
  // a8: Eq.6-7 hand dL/dC^k, dL/dT^k to every partition's rasteriser backward
  if ((rc = splx_compose_backward_plan(ctx, K, partials, bins, plan, bg, dL_dimage, dL_dT_total, g_ct))) return rc;
  SPLX_CUDA_OK(ctx, cudaMemsetAsync(g2d, 0, (size_t)g->n * SPLX_G2D_STRIDE * sizeof(float), ctx->stream));
  // a9: reverse-order blend gradients into means2D, conic, opacity, colour
  if ((rc = splx_raster_backward_plan(ctx, proj, bins, K, plan, partials, g_ct, g2d))) return rc;
  // a10: projection backward to the 3-D parameters
  return splx_project_backward_plan(ctx, g, K, part_offsets, plan, sh_degree, proj, g2d, flags, grads);
}

int splx_backward(splx_ctx* ctx, int K, const splx_partial* partials, const splx_camera* cam, const float bg[3],
                  const float* dL_dimage, const float* dL_dT_total, const splx_gaussians* g,
                  const splx_projected* proj, const splx_binning* bins, int sh_degree,
                  const splx_gaussian_grads* grads, void* ws, size_t ws_bytes, int flags) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!gauss_ok(g) || !cam_ok(cam)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_backward: null/misaligned argument");
  if (K < 1 || K > SPLX_MAX_K) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_backward: K=%d not in [1,%d]", K, SPLX_MAX_K);
  const SinglePlan sp(cam);
  // the projection backward needs no partition structure for a single view: one run over all Gaussians
  int64_t po[SPLX_MAX_K + 1];
  po[0] = 0;
  for (int k = 1; k <= K; ++k) po[k] = g->n;
  return splx_backward_plan(ctx, K, po, &sp.plan, partials, bg, dL_dimage, dL_dT_total, g, proj, bins, sh_degree, grads,
                            ws, ws_bytes, flags);
}

int splx_adam_sparse(splx_ctx* ctx, const splx_gaussian_grads* params, const splx_gaussian_grads* grads,
                     const splx_gaussian_grads* m, const splx_gaussian_grads* v, uint8_t* touched, const float lr[5],
                     float beta1, float beta2, float eps, int step, float grad_scale) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!params || !grads || !m || !v || !touched || !lr || step < 1)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_sparse: null argument or step < 1");
  const splx_gaussian_grads* sets[4] = {params, grads, m, v};
  for (const splx_gaussian_grads* s : sets)
    if (s->n != params->n || (s->n > 0 && (!s->mean || !s->log_scale || !s->quat || !s->opacity_logit || !s->sh ||
                                           !aligned16(s->quat) || !aligned16(s->sh))))
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_sparse: params, grads, m, v must be four sets of n rows (quat, sh 16-byte aligned)");
  return launch_adam_sparse(ctx, params, grads, m, v, touched, lr, beta1, beta2, eps, step, grad_scale);
}

int splx_adam(splx_ctx* ctx, float* param, float* grad, float* m, float* v, int64_t count, float lr, float beta1,
              float beta2, float eps, int step, float grad_scale, int zero_grad) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!param || !grad || !m || !v || count < 0 || step < 1 || !aligned16(param) || !aligned16(grad) ||
      !aligned16(m) || !aligned16(v))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam: null/misaligned argument or step < 1");
  return launch_adam(ctx, param, grad, m, v, count, lr, beta1, beta2, eps, step, grad_scale, zero_grad);
}

int splx_adam_groups(splx_ctx* ctx, float* param, float* grad, float* m, float* v, int n_groups,
                     const int64_t* group_offsets, const float* lr, float beta1, float beta2, float eps, int step,
                     float grad_scale, int zero_grad) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!param || !grad || !m || !v || !group_offsets || !lr || step < 1 || !aligned16(param) || !aligned16(grad) ||
      !aligned16(m) || !aligned16(v))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups: null/misaligned argument or step < 1");
  if (n_groups < 1 || n_groups > SPLX_ADAM_MAX_GROUPS)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups: n_groups=%d not in [1,%d]", n_groups, SPLX_ADAM_MAX_GROUPS);
  if (group_offsets[0] != 0) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups: group_offsets[0] must be 0");
  for (int j = 0; j < n_groups; ++j)
    if (group_offsets[j + 1] < group_offsets[j] || (group_offsets[j + 1] & 3))
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups: offsets must be monotone multiples of 4");
  return launch_adam_groups(ctx, param, grad, m, v, n_groups, group_offsets, lr, beta1, beta2, eps, step, grad_scale,
                            zero_grad);
}

int splx_adam_groups_flagged(splx_ctx* ctx, float* param, const float* grad, float* m, float* v, int n_groups,
                             const int64_t* group_offsets, const int32_t* widths, int64_t rows, const uint8_t* touched,
                             const float* lr, float beta1, float beta2, float eps, int step, float grad_scale) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!param || !grad || !m || !v || !group_offsets || !widths || !touched || !lr || step < 1 || rows < 0 || !aligned16(param) ||
      !aligned16(grad) || !aligned16(m) || !aligned16(v))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: null/misaligned argument or step < 1");
  if (n_groups < 1 || n_groups > SPLX_ADAM_MAX_GROUPS)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: n_groups=%d not in [1,%d]", n_groups, SPLX_ADAM_MAX_GROUPS);
  if (group_offsets[0] != 0) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: group_offsets[0] must be 0");
  for (int j = 0; j < n_groups; ++j) {
    if (group_offsets[j + 1] < group_offsets[j] || (group_offsets[j + 1] & 3))
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: offsets must be monotone multiples of 4");
    if (widths[j] < 1 || group_offsets[j + 1] - group_offsets[j] < rows * widths[j])
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: group %d does not hold rows x width floats", j);
  }
  return launch_adam_groups(ctx, param, const_cast<float*>(grad), m, v, n_groups, group_offsets, lr, beta1, beta2, eps, step,
                            grad_scale, 0, widths, rows, touched);
}

}  // extern "C"
