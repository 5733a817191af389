// common.cuh -- shared declarations of the CUDA path (sm_100a).  Nothing here is shared
// with oracle/: the oracle restates every formula on its own.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <math.h>
#include <string.h>

#include "../../include/splx.h"

#define SPLX_SM_COUNT 148  // B200: 2 dies x 74 SMs; grids of persistent kernels are multiples of it

struct splx_ctx {
  int device;
  cudaStream_t stream;
  splx_config cfg;
  int64_t launches;
  char err[512];
  // splx_iteration's own streams and events, created at its first call (iteration.cu), destroyed by splx_destroy
  bool iter_ready;
  cudaStream_t s_front, s_up, s_down;     // a1-a4 of the next bucket; host -> device targets; device -> host results
  cudaEvent_t ev_start, ev_up, ev_front[2], ev_back[2], ev_img, ev_down;
};
void iteration_release(splx_ctx*);

// Device-side copy of the camera plus derived quantities, passed by value to kernels.
struct CamDev {
  float R[9], t[3];
  float fx, fy, cx, cy;
  int W, H, TX, TY;
  float near_z;
  float o[3];  // camera centre -R^T t
  float limx, limy;
  // reach test of a mean (reading s21): a Gaussian of scale <= s can touch the image only if
  //   -(reach_l z + 3 reach_c s) <= fx x <= reach_r z + 3 reach_c s   and the same with (reach_t, reach_b) for fy y
  float reach_l, reach_r, reach_t, reach_b, reach_c;
};

static inline CamDev make_camdev(const splx_camera* c, const splx_config& cfg) {
  CamDev d;
  for (int i = 0; i < 9; ++i) d.R[i] = c->R[i];
  for (int i = 0; i < 3; ++i) d.t[i] = c->t[i];
  d.fx = c->fx; d.fy = c->fy; d.cx = c->cx; d.cy = c->cy;
  d.W = c->width; d.H = c->height;
  d.TX = (c->width + SPLX_TILE - 1) / SPLX_TILE;
  d.TY = (c->height + SPLX_TILE - 1) / SPLX_TILE;
  d.near_z = c->near_z;
  for (int j = 0; j < 3; ++j)
    d.o[j] = -(c->R[0 * 3 + j] * c->t[0] + c->R[1 * 3 + j] * c->t[1] + c->R[2 * 3 + j] * c->t[2]);
  d.limx = cfg.lim_factor * (float)c->width / (2.0f * c->fx);
  d.limy = cfg.lim_factor * (float)c->height / (2.0f * c->fy);
  {   // g = 2.5 + 3 sqrt(dilation + sqrt(radius_floor)) pixels, +0.5 and 1e-4 relative for the fp32 evaluation of the test
    const double e = (double)cfg.dilation + sqrt((double)cfg.radius_floor), g = 3.0 + 3.0 * sqrt(e);
    const double fm = c->fx > c->fy ? c->fx : c->fy;
    d.reach_l = (float)((c->cx + g) * 1.0001); d.reach_r = (float)(((double)c->width - c->cx + g) * 1.0001);
    d.reach_t = (float)((c->cy + g) * 1.0001); d.reach_b = (float)(((double)c->height - c->cy + g) * 1.0001);
    d.reach_c = (float)(fm * sqrt(1.0 + (double)d.limx * d.limx + (double)d.limy * d.limy) * 1.0001);
  }
  return d;
}

// Launch plan on the device side (splx_plan): B views of identical size, the view each partition
// renders in this launch (-1 = the partition does not participate), the optional per-(partition,
// tile) visibility state and the flags.  Passed to kernels as a __grid_constant__ parameter so that
// the per-partition camera is an indexed constant-bank load.
struct PartView { signed char v[SPLX_MAX_K]; };

struct PlanDev {
  int B, K, W, H, TX, TY, ntiles, flags;
  const uint8_t* tile_state;
  PartView pv;
  CamDev cam[SPLX_MAX_VIEWS];
  float max_scale[SPLX_MAX_K];   // splx_plan.max_scale, or < 0: no reach test
  uint32_t open_slots;           // |splx_plan.open_slots|
  bool open_forced;              // splx_plan.open_slots < 0: renumber even where no radix pass is saved
  const uint32_t* slot_map;      // splx_plan.slot_map
};

// Per-view buffers of the composition kernels (view b of the launch -> its own pointers), so that the views of a
// launch need not be contiguous in one allocation (a bucket takes views 0 and 3 of an iteration, say).
struct ViewBufs {
  const float* target[SPLX_MAX_VIEWS];     // [H,W,3]
  float* image[SPLX_MAX_VIEWS];            // [H,W,3]
  float* T_total[SPLX_MAX_VIEWS];          // [H,W] or nullptr
  float* g_image[SPLX_MAX_VIEWS];          // [H,W,3]: written by the loss kernels, read by the composition backward
  const float* g_T_total[SPLX_MAX_VIEWS];  // [H,W] or nullptr
};
// views 0..B-1 of contiguous [B,H,W,*] arrays (any of them may be nullptr)
static inline ViewBufs contiguous_views(int B, size_t HW, const float* target, float* image, float* T_total,
                                        float* g_image, const float* g_T_total) {
  ViewBufs vb;
  memset(&vb, 0, sizeof vb);
  for (int b = 0; b < B; ++b) {
    vb.target[b] = target ? target + 3 * HW * b : nullptr;
    vb.image[b] = image ? image + 3 * HW * b : nullptr;
    vb.T_total[b] = T_total ? T_total + HW * b : nullptr;
    vb.g_image[b] = g_image ? g_image + 3 * HW * b : nullptr;
    vb.g_T_total[b] = g_T_total ? g_T_total + HW * b : nullptr;
  }
  return vb;
}

// Cross-boundary per-ray filtering (L474-L476): the per-Gaussian Q_cross masks and the depth interval D^k of every
// partition under the view it renders.  mask == nullptr = no filtering.
struct CrossDev {
  const uint64_t* mask;
  float zlo[SPLX_MAX_K], zhi[SPLX_MAX_K];
};

// splx_binning.slot_order is built and used only where it pays: measured +1 % to +6 % at 1080p (8160 tiles, K = 4..32:
// few waves of blend CTAs, the tail matters) and -0.5 % at 4K (32400 tiles, K = 16: many waves, and the order costs
// locality in L2).  One rule for the producer (bin_sort) and the consumers (blend kernels).
static inline bool slot_order_pays(const PlanDev& p) { return p.ntiles <= 16384; }

// Contiguous runs of Gaussians (one per participating partition) covered by ONE launch of a
// per-Gaussian kernel: block b works on run r with block_prefix[r] <= b < block_prefix[r+1].
// view[r] < 0 marks a run of a non-participating partition (only present when its outputs must
// be cleared).  jprefix = running count of Gaussians, for kernels indexed by element.
struct RunTable {
  int n, blocks_total;
  int64_t begin[SPLX_MAX_K], end[SPLX_MAX_K], jprefix[SPLX_MAX_K + 1];
  int block_prefix[SPLX_MAX_K + 1];
  signed char view[SPLX_MAX_K];
  signed char part[SPLX_MAX_K];     // the partition of run r
};

static inline RunTable make_runs(const PlanDev& plan, const int64_t* part_offsets, int block, bool with_inactive) {
  RunTable rt;
  memset(&rt, 0, sizeof rt);
  for (int k = 0; k < plan.K; ++k) {
    const int v = plan.pv.v[k];
    const int64_t b = part_offsets[k], e = part_offsets[k + 1];
    if (e <= b || (v < 0 && !with_inactive)) continue;
    const int r = rt.n++;
    rt.begin[r] = b; rt.end[r] = e; rt.view[r] = (signed char)v; rt.part[r] = (signed char)k;
    rt.jprefix[r + 1] = rt.jprefix[r] + (e - b);
    rt.block_prefix[r + 1] = rt.block_prefix[r] + (int)((e - b + block - 1) / block);
  }
  rt.blocks_total = rt.block_prefix[rt.n];
  return rt;
}

#define SPLX_FAIL(ctx, code, ...)                                  \
  do {                                                             \
    snprintf((ctx)->err, sizeof((ctx)->err), __VA_ARGS__);         \
    return (code);                                                 \
  } while (0)

#define SPLX_CUDA_OK(ctx, expr)                                                          \
  do {                                                                                   \
    cudaError_t e_ = (expr);                                                             \
    if (e_ != cudaSuccess)                                                               \
      SPLX_FAIL(ctx, SPLX_ERR_CUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));     \
  } while (0)

#define SPLX_LAUNCH_CHECK(ctx, name)                                                     \
  do {                                                                                   \
    cudaError_t e_ = cudaGetLastError();                                                 \
    if (e_ != cudaSuccess)                                                               \
      SPLX_FAIL(ctx, SPLX_ERR_CUDA, "launch of %s failed: %s", name, cudaGetErrorString(e_)); \
    (ctx)->launches++;                                                                   \
  } while (0)

static inline bool aligned16(const void* p) { return (((uintptr_t)p) & 15u) == 0; }
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Tile rectangle of a projected footprint (reading s11): pixel i samples i+0.5,
// so [u-r, u+r] covers pixel columns i with u-0.5-r <= i <= u-0.5+r.  Written with explicit
// round-to-nearest intrinsics so that no fused multiply-add can change the integer result.
__device__ __forceinline__ void tile_rect(float u, float v, int radius, int TX, int TY, int& x0,
                                          int& y0, int& x1, int& y1) {
  const float rf = (float)radius;
  const float ux = __fsub_rn(u, 0.5f), vy = __fsub_rn(v, 0.5f);
  const float x0f = floorf(__fmul_rn(__fsub_rn(ux, rf), 0.0625f));
  const float x1f = floorf(__fmul_rn(__fadd_rn(__fadd_rn(ux, rf), 15.0f), 0.0625f));
  const float y0f = floorf(__fmul_rn(__fsub_rn(vy, rf), 0.0625f));
  const float y1f = floorf(__fmul_rn(__fadd_rn(__fadd_rn(vy, rf), 15.0f), 0.0625f));
  x0 = !(x0f > 0.0f) ? 0 : (x0f >= (float)TX ? TX : (int)x0f);
  x1 = !(x1f > 0.0f) ? 0 : (x1f >= (float)TX ? TX : (int)x1f);
  y0 = !(y0f > 0.0f) ? 0 : (y0f >= (float)TY ? TY : (int)y0f);
  y1 = !(y1f > 0.0f) ? 0 : (y1f >= (float)TY ? TY : (int)y1f);
}

// validates a splx_plan against K and builds the device-side copy (api.cu)
int make_plan_dev(splx_ctx*, const char* who, int K, const splx_plan*, PlanDev* out);

// ---- stage launchers (defined one per .cu file, called from api.cu) ----------------------
int launch_project_fwd(splx_ctx*, const splx_gaussians*, const PlanDev&, const int64_t* part_offsets, int sh_degree,
                       const splx_projected*, bool with_colour = true);
int launch_project_colour_list(splx_ctx*, const splx_gaussians*, const PlanDev&, const int64_t* part_offsets, int sh_degree,
                               const splx_projected*, const uint32_t* visible_list, const uint64_t* num_visible);
int launch_project_bwd(splx_ctx*, const splx_gaussians*, const PlanDev&, const int64_t* part_offsets, int sh_degree,
                       const splx_projected*, float* g2d, int flags, const splx_gaussian_grads*,
                       const uint32_t* visible_list, const uint64_t* num_visible, uint8_t* touched);
int launch_adam_sparse(splx_ctx*, const splx_gaussian_grads* params, const splx_gaussian_grads* grads,
                       const splx_gaussian_grads* m, const splx_gaussian_grads* v, uint8_t* touched, const float* lr,
                       float beta1, float beta2, float eps, int step, float grad_scale);
// the depth-sorted list of visible Gaussians a bin_sort leaves in its workspace, and its device-side count
int bin_sort_visible(const void* ws, int64_t n, uint64_t capacity, int K, int TX, int TY, const uint32_t** list,
                     const uint64_t** count);
size_t bin_sort_ws_bytes(int64_t n, uint64_t capacity, int K, int TX, int TY);
int launch_slot_map(splx_ctx*, const PlanDev&, uint32_t* slot_map_out);
int launch_gradient_rows(splx_ctx*, void* ws, int64_t n, uint64_t capacity, int K, int TX, int TY, const float* g2d,
                         const uint32_t** rows, const uint64_t** num_rows);
int launch_bin_sort(splx_ctx*, const splx_projected*, int64_t n, const PlanDev&, const int64_t* part_offsets,
                    const splx_binning*, void* ws, size_t ws_bytes, const CrossDev* cross = nullptr);
int launch_cross_sets(splx_ctx*, const splx_gaussians*, int K, const int64_t* part_offsets, const float* cell_lo,
                      const float* cell_hi, float support_sigma, uint64_t* cross_mask);
int launch_render_fwd(splx_ctx*, const splx_projected*, const splx_binning*, const PlanDev&,
                      const splx_partial*, uint64_t* pairs);
int launch_raster_bwd(splx_ctx*, const splx_projected*, const splx_binning*, const PlanDev&,
                      const splx_partial*, const float* g_ct, float* g2d);
int launch_compose_fwd(splx_ctx*, const splx_partial*, const splx_binning* bins, const PlanDev&, const float* bg,
                       const ViewBufs&, float sat_eps, uint8_t* tile_state_out);
int launch_compose_bwd(splx_ctx*, const splx_partial*, const splx_binning* bins, const PlanDev&, const float* bg,
                       const ViewBufs&, float* g_ct);
int launch_compose_fused(splx_ctx*, const splx_partial*, const splx_binning* bins, const PlanDev&, const float* bg,
                         const ViewBufs&, float scale, double* loss_sum, float* g_ct, float sat_eps,
                         uint8_t* tile_state_out);
size_t dssim_ws_floats(int W, int H);
int launch_dssim(splx_ctx*, int B, int W, int H, const ViewBufs&, float lambda, float scale, double* loss_sum, float* ws);
int launch_l1(splx_ctx*, const float* image, const float* target, int64_t count, float scale,
              float* g_image, double* loss_sum);
int launch_adam_groups(splx_ctx*, float* param, float* grad, float* m, float* v, int n_groups,
                       const int64_t* group_offsets, const float* lr, float beta1, float beta2, float eps, int step,
                       float grad_scale, int zero_grad, const int32_t* widths = nullptr, int64_t rows = 0,
                       const uint8_t* touched = nullptr);
int launch_adam(splx_ctx*, float* param, float* grad, float* m, float* v, int64_t count, float lr,
                float beta1, float beta2, float eps, int step, float grad_scale, int zero_grad);
