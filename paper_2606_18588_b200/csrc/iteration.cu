// iteration.cu -- splx_iteration: one whole training iteration (a1-a10, optionally a11) over the buckets of views of
// PAPER.md L249 behind ONE C-ABI call, with the host <-> device copies of the end-to-end path inside the library.
// Sequencing only (Fig. 9: local render -> pixel exchange -> global composition -> loss -> backward,
// per view; L249: views of a conflict-free bucket together): every step runs in the kernels of the other files.
//
// Streams: the context's stream carries the blending half (a5-a10) of every bucket; s_front carries projection +
// binning (a1-a4) of the NEXT bucket when the caller gave a second splx_frontset (small latency-bound kernels that
// leave most SMs idle beside the blend kernels); s_up / s_down carry the pinned-host copies (SPLX_ITER_HOST).  All
// of them are forked from and joined back into the context's stream with events, so the call is asynchronous, never
// synchronises, and can be captured into a CUDA graph by the caller.
#include "common.cuh"

static int iteration_streams(splx_ctx* ctx) {
  if (ctx->iter_ready) return SPLX_OK;
  SPLX_CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->s_front, cudaStreamNonBlocking));
  SPLX_CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->s_up, cudaStreamNonBlocking));
  SPLX_CUDA_OK(ctx, cudaStreamCreateWithFlags(&ctx->s_down, cudaStreamNonBlocking));
  cudaEvent_t* evs[] = {&ctx->ev_start, &ctx->ev_up, &ctx->ev_front[0], &ctx->ev_front[1], &ctx->ev_back[0],
                        &ctx->ev_back[1], &ctx->ev_img, &ctx->ev_down};
  for (cudaEvent_t* e : evs) SPLX_CUDA_OK(ctx, cudaEventCreateWithFlags(e, cudaEventDisableTiming));
  ctx->iter_ready = true;
  return SPLX_OK;
}

void iteration_release(splx_ctx* ctx) {
  if (!ctx->iter_ready) return;
  cudaStreamDestroy(ctx->s_front); cudaStreamDestroy(ctx->s_up); cudaStreamDestroy(ctx->s_down);
  cudaEvent_t evs[] = {ctx->ev_start, ctx->ev_up, ctx->ev_front[0], ctx->ev_front[1], ctx->ev_back[0], ctx->ev_back[1],
                       ctx->ev_img, ctx->ev_down};
  for (cudaEvent_t e : evs) cudaEventDestroy(e);
  ctx->iter_ready = false;
}

namespace {

// runs `body` with the context's stream temporarily set to `st`
struct StreamScope {
  splx_ctx* ctx; cudaStream_t saved;
  StreamScope(splx_ctx* c, cudaStream_t st) : ctx(c), saved(c->stream) { c->stream = st; }
  ~StreamScope() { ctx->stream = saved; }
};

bool grads_ok(const splx_gaussian_grads& s, int64_t n) {
  return s.n == n && (n == 0 || (s.mean && s.log_scale && s.quat && s.opacity_logit && s.sh));
}

}  // namespace

extern "C" {

size_t splx_dssim_ws_floats(const splx_camera* cam) {
  if (!cam || cam->width <= 0 || cam->height <= 0) return 0;
  return dssim_ws_floats(cam->width, cam->height);
}

int splx_dssim_loss_grad(splx_ctx* ctx, int n_views, const splx_camera* cam, const float* image, const float* target,
                         float lambda, float scale, float* dL_dimage, double* loss_sum, float* ws) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam || cam->width <= 0 || cam->height <= 0 || n_views < 1 || n_views > SPLX_MAX_VIEWS || !image || !target ||
      !dL_dimage || !ws || !(lambda >= 0.f))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_dssim_loss_grad: null argument, bad size, n_views not in [1,%d] or lambda < 0",
              SPLX_MAX_VIEWS);
  const ViewBufs vb = contiguous_views(n_views, (size_t)cam->width * cam->height, target, const_cast<float*>(image), nullptr,
                                       dL_dimage, nullptr);
  return launch_dssim(ctx, n_views, cam->width, cam->height, vb, lambda, scale, loss_sum, ws);
}

int splx_iteration(splx_ctx* ctx, const splx_trainset* ts, int n_buckets, const splx_bucket* buckets, int n_views,
                   const float* const* targets, float* const* images_out, double* loss_out, uint64_t* m_out,
                   const splx_iter_opts* opts, const splx_adam_cfg* adam) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!ts || !buckets || !targets || !opts || n_buckets < 1 || n_views < 1)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: null argument or empty iteration");
  if (opts->flags & ~(SPLX_ITER_HOST | SPLX_ITER_FUSED_PROJECTION | SPLX_ITER_KEEP_ZERO_ROWS)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: unknown flags %d", opts->flags);
  const bool host = (opts->flags & SPLX_ITER_HOST) != 0;
  if (!host && (images_out || loss_out)) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: images_out / loss_out need SPLX_ITER_HOST");
  const int64_t n = ts->params.n;
  const int K = ts->K;
  if (K < 1 || K > SPLX_MAX_K || !ts->part_offsets || !grads_ok(ts->params, n) || !grads_ok(ts->grads, n))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: K, part_offsets, params or grads invalid");
  if (n_views > ts->max_views || !ts->images || !ts->g_ct || !ts->g2d || !ts->loss_sum || (host && !ts->targets) ||
      !ts->front[0].ws)
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: trainset buffers missing or n_views > max_views");
  const bool dssim = opts->lambda_dssim > 0.f;
  if (!(opts->lambda_dssim >= 0.f) || (dssim && (!ts->g_images || !ts->dssim_ws)))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: lambda_dssim < 0, or > 0 without g_images / dssim_ws");
  // every view in exactly one bucket, all views of one size
  int seen[SPLX_MAX_VIEWS * SPLX_MAX_K];
  if (n_views > SPLX_MAX_VIEWS * SPLX_MAX_K) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: too many views");
  for (int v = 0; v < n_views; ++v) { seen[v] = 0; if (!targets[v]) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: targets[%d] is NULL", v); }
  int W = 0, H = 0;
  for (int g = 0; g < n_buckets; ++g) {
    const splx_plan& p = buckets[g].plan;
    if (!p.cams || !p.view_of_part || !buckets[g].view_index || p.n_views < 1 || p.n_views > SPLX_MAX_VIEWS)
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: bucket %d: plan or view_index invalid", g);
    if (ts->cross_mask && !buckets[g].part_depth_range)
      SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: bucket %d: cross_mask needs part_depth_range", g);
    for (int b = 0; b < p.n_views; ++b) {
      const int v = buckets[g].view_index[b];
      if (v < 0 || v >= n_views || seen[v]++) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: bucket %d: view index %d out of range or used twice", g, v);
      if (g == 0 && b == 0) { W = p.cams[0].width; H = p.cams[0].height; }
      if (p.cams[b].width != W || p.cams[b].height != H) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: all views must have one size");
    }
  }
  for (int v = 0; v < n_views; ++v) if (!seen[v]) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_iteration: view %d is in no bucket", v);
  int rc;
  if ((rc = iteration_streams(ctx))) return rc;

  const size_t HW = (size_t)W * H;
  cudaStream_t main = ctx->stream;
  const bool pipelined = n_buckets > 1 && ts->front[1].ws != nullptr;
  const bool down = host && (images_out || loss_out);
  const splx_gaussians g{ts->params.mean, ts->params.log_scale, ts->params.quat, ts->params.opacity_logit, ts->params.sh, n};

  SPLX_CUDA_OK(ctx, cudaMemsetAsync(ts->loss_sum, 0, 2 * sizeof(double), main));
  if (ts->touched && n > 0) SPLX_CUDA_OK(ctx, cudaMemsetAsync(ts->touched, 0, (size_t)n, main));
  SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_start, main));
  if (host) {   // the targets travel while the first bucket is projected, binned and rendered: first needed by the loss
    SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(ctx->s_up, ctx->ev_start, 0));
    for (int v = 0; v < n_views; ++v)
      SPLX_CUDA_OK(ctx, cudaMemcpyAsync(ts->targets + 3 * HW * v, targets[v], 3 * HW * sizeof(float), cudaMemcpyHostToDevice, ctx->s_up));
    SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_up, ctx->s_up));
  }
  bool down_used = false;

  // a1-a4 of bucket gi into front set `set`, on stream st
  auto front = [&](int gi, int set, cudaStream_t st) -> int {
    StreamScope scope(ctx, st);
    const splx_bucket& bk = buckets[gi];
    const splx_frontset& fs = ts->front[set];
    int r;
    // the colour only for the visible Gaussians, once the binning has compacted their list (the geometry alone decides
    // visibility, depth and footprint: the binning does not read the colour)
    if (opts->flags & SPLX_ITER_FUSED_PROJECTION) {
      if ((r = splx_project_plan(ctx, &g, K, ts->part_offsets, &bk.plan, ts->sh_degree, &fs.proj))) return r;
      return splx_bin_sort_filtered_plan(ctx, &fs.proj, n, K, ts->part_offsets, &bk.plan, ts->cross_mask, bk.part_depth_range,
                                         &fs.bins, fs.ws, fs.ws_bytes);
    }
    if ((r = splx_project_geometry_plan(ctx, &g, K, ts->part_offsets, &bk.plan, &fs.proj))) return r;
    if ((r = splx_bin_sort_filtered_plan(ctx, &fs.proj, n, K, ts->part_offsets, &bk.plan, ts->cross_mask, bk.part_depth_range,
                                         &fs.bins, fs.ws, fs.ws_bytes))) return r;
    const uint32_t* vlist = nullptr;
    const uint64_t* nvis = nullptr;
    if ((r = splx_bin_sort_visible(fs.ws, n, fs.bins.capacity, K, &bk.plan.cams[0], &vlist, &nvis))) SPLX_FAIL(ctx, r, "splx_iteration: visible list");
    return splx_project_colour_list_plan(ctx, &g, K, ts->part_offsets, &bk.plan, ts->sh_degree, &fs.proj, vlist, nvis);
  };

  // a5-a10 of bucket gi from front set `set`, on the context's stream
  auto back = [&](int gi, int set) -> int {
    const splx_bucket& bk = buckets[gi];
    const splx_frontset& fs = ts->front[set];
    const splx_plan* plan = &bk.plan;
    int r;
    if ((r = splx_render_partial_plan(ctx, &fs.proj, &fs.bins, K, plan, &ts->partials, nullptr))) return r;
    PlanDev pd;
    if ((r = make_plan_dev(ctx, "splx_iteration", K, plan, &pd))) return r;
    ViewBufs vb;
    memset(&vb, 0, sizeof vb);
    for (int b = 0; b < plan->n_views; ++b) {
      const size_t v = (size_t)bk.view_index[b];
      vb.target[b] = host ? ts->targets + 3 * HW * v : targets[v];
      vb.image[b] = ts->images + 3 * HW * v;
      vb.T_total[b] = ts->T_totals ? ts->T_totals + HW * v : nullptr;
      vb.g_image[b] = ts->g_images ? ts->g_images + 3 * HW * v : nullptr;
    }
    if (host && gi == 0) SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(main, ctx->ev_up, 0));
    const float scale = (float)plan->n_views;     // every view's loss is its own mean
    if (!dssim) {   // a6 + a7 + a8 in one pass over the partials
      if ((r = launch_compose_fused(ctx, &ts->partials, &fs.bins, pd, ts->bg, vb, scale, ts->loss_sum, ts->g_ct, opts->sat_eps,
                                    bk.tile_state_out))) return r;
    } else {        // a6, then L_RGB + lambda L_D-SSIM (an 11 x 11 neighbourhood: its own kernels), then a8
      if ((r = launch_compose_fwd(ctx, &ts->partials, &fs.bins, pd, ts->bg, vb, opts->sat_eps, bk.tile_state_out))) return r;
      // the D-SSIM workspace is indexed by the view's position in THIS launch; launches are serialised on the stream
      if ((r = launch_dssim(ctx, plan->n_views, W, H, vb, opts->lambda_dssim, scale, ts->loss_sum, ts->dssim_ws))) return r;
      if ((r = launch_compose_bwd(ctx, &ts->partials, &fs.bins, pd, ts->bg, vb, ts->g_ct))) return r;
    }
    if (down || m_out) {   // results leave while the backward runs
      SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_img, main));
      SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(ctx->s_down, ctx->ev_img, 0));
      if (images_out)
        for (int b = 0; b < plan->n_views; ++b) {
          const size_t v = (size_t)bk.view_index[b];
          if (images_out[v])
            SPLX_CUDA_OK(ctx, cudaMemcpyAsync(images_out[v], ts->images + 3 * HW * v, 3 * HW * sizeof(float), cudaMemcpyDeviceToHost, ctx->s_down));
        }
      if (m_out)
        SPLX_CUDA_OK(ctx, cudaMemcpyAsync(m_out + gi, fs.bins.num_intersections, sizeof(uint64_t), cudaMemcpyDeviceToHost, ctx->s_down));
      // the loss after the last images: both use the one device-to-host copy engine, in this order nothing waits
      if (loss_out && gi == n_buckets - 1)
        SPLX_CUDA_OK(ctx, cudaMemcpyAsync(loss_out, ts->loss_sum, 2 * sizeof(double), cudaMemcpyDeviceToHost, ctx->s_down));
      down_used = true;
    }
    if ((r = splx_raster_backward_plan(ctx, &fs.proj, &fs.bins, K, plan, &ts->partials, ts->g_ct, ts->g2d))) return r;
    // a10: with flags (ts->touched) every bucket walks the binning's list of visible Gaussians, stores the gradient of a
    // row it is the first to reach and adds to the others; without them the first bucket stores every row of the
    // gradient (zeros where nothing is visible) and later buckets accumulate over the list
    const uint32_t* vlist = nullptr;
    const uint64_t* nvis = nullptr;
    if (ts->touched || gi > 0) {
      if ((r = splx_bin_sort_visible(fs.ws, n, fs.bins.capacity, K, &plan->cams[0], &vlist, &nvis))) SPLX_FAIL(ctx, r, "splx_iteration: visible list");
      // only the Gaussians that received a 2-D gradient: the others have a zero gradient -- with flags they stay unflagged
      // (an unflagged row counts as zero), without flags this is an accumulating launch and adding zero changes nothing
      const bool keep_all = ts->touched && ((opts->flags & SPLX_ITER_KEEP_ZERO_ROWS) || (adam && adam->sparse));
      if (!keep_all &&
          (r = splx_bin_sort_gradient_rows(ctx, fs.ws, n, fs.bins.capacity, K, &plan->cams[0], ts->g2d, &vlist, &nvis))) return r;
      return splx_project_backward_list_plan(ctx, &g, K, ts->part_offsets, plan, ts->sh_degree, &fs.proj, ts->g2d,
                                             SPLX_PB_CLEAR_G2D, &ts->grads, vlist, nvis, ts->touched);
    }
    return splx_project_backward_plan(ctx, &g, K, ts->part_offsets, plan, ts->sh_degree, &fs.proj, ts->g2d,
                                      SPLX_PB_CLEAR_G2D | SPLX_PB_OVERWRITE, &ts->grads);
  };

  if (!pipelined) {
    for (int gi = 0; gi < n_buckets; ++gi) {
      if ((rc = front(gi, 0, main))) return rc;
      if ((rc = back(gi, 0))) return rc;
    }
  } else {
    SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(ctx->s_front, ctx->ev_start, 0));     // the parameters of the previous optimiser step
    if ((rc = front(0, 0, ctx->s_front))) return rc;
    SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_front[0], ctx->s_front));
    for (int gi = 0; gi < n_buckets; ++gi) {
      if (gi + 1 < n_buckets) {
        // front set (gi + 1) % 2 was last read by the blending half of bucket gi - 1
        if (gi >= 1) SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(ctx->s_front, ctx->ev_back[(gi - 1) % 2], 0));
        if ((rc = front(gi + 1, (gi + 1) % 2, ctx->s_front))) return rc;
        SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_front[(gi + 1) % 2], ctx->s_front));
      }
      SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(main, ctx->ev_front[gi % 2], 0));
      if ((rc = back(gi, gi % 2))) return rc;
      SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_back[gi % 2], main));
    }
  }

  if (adam) {
    const float gs = 1.0f / (float)n_views;
    if (ts->touched && adam->sparse) {
      if ((rc = splx_adam_sparse(ctx, &ts->params, &ts->grads, &adam->m_soa, &adam->v_soa, ts->touched, adam->lr, adam->beta1,
                                 adam->beta2, adam->eps, adam->step, gs))) return rc;
    } else if (ts->touched) {
      if ((rc = splx_adam_groups_flagged(ctx, adam->param, adam->grad, adam->m, adam->v, adam->n_groups, adam->group_offsets,
                                         adam->widths, n, ts->touched, adam->lr, adam->beta1, adam->beta2, adam->eps, adam->step,
                                         gs))) return rc;
    } else {
      if ((rc = splx_adam_groups(ctx, adam->param, adam->grad, adam->m, adam->v, adam->n_groups, adam->group_offsets, adam->lr,
                                 adam->beta1, adam->beta2, adam->eps, adam->step, gs, 0))) return rc;
    }
  }
  if (down_used) {   // join: a caller that synchronises the context's stream finds the host buffers complete
    SPLX_CUDA_OK(ctx, cudaEventRecord(ctx->ev_down, ctx->s_down));
    SPLX_CUDA_OK(ctx, cudaStreamWaitEvent(main, ctx->ev_down, 0));
  }
  return SPLX_OK;
}

}  // extern "C"
