/* splx.h -- C ABI of libsplx.so: the single-GPU (B200, sm_100a) hot path of Splaxel's
 * pixel-level scheme (arxiv/paper_2606_18588).  Citations are PAPER.md line numbers.
 *
 * K Gaussian partitions ("simulated ranks") live as K contiguous
 * slices of one SoA parameter set.  Every call below processes ALL K partitions in one
 * launch per stage: the partition index is folded into the high bits of the tile key, so
 * one sort, one render grid (K x tiles) and one backward grid cover the K ranks.
 *
 * Conventions
 *  - extern "C", plain pointers and sizes.  Structs are read on the HOST at call time;
 *    every pointer INSIDE them that names data is a CUDA DEVICE pointer to caller-owned
 *    memory (16-byte aligned), unless the field comment says "host".  The library never
 *    frees, reallocates or keeps those pointers after the call returns.
 *  - All calls are asynchronous on the CUDA stream given to splx_create and never
 *    synchronise the device.  Scratch memory is a caller-owned workspace; the *_ws_bytes
 *    queries give its size.
 *  - Return value: SPLX_OK (0) or a negative error; splx_last_error gives text.  No
 *    exceptions cross the boundary.  There is no CPU fallback: without a CUDA device
 *    splx_create fails with SPLX_ERR_CUDA.
 *  - Gradient outputs are ACCUMULATED (+=); the caller zeroes them (lets B views sum).
 *  - fp32 everywhere; indices and keys are integers.  Tile = 16 x 16 pixels; pixel (i,j)
 *    samples the point (i+0.5, j+0.5).
 */
#ifndef SPLX_H_
#define SPLX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPLX_OK 0
#define SPLX_ERR_INVALID_ARG (-1) /* null / misaligned pointer, bad size, sh_degree not in [0,3], K not in [1,64] */
#define SPLX_ERR_WORKSPACE (-2)   /* workspace too small */
#define SPLX_ERR_CAPACITY (-3)    /* reported by splx_check_capacity: more intersections than binning.capacity */
#define SPLX_ERR_CUDA (-4)        /* a CUDA runtime call failed (text in splx_last_error) */

#define SPLX_MAX_K 64
#define SPLX_TILE 16
#define SPLX_ADAM_MAX_GROUPS 8
#define SPLX_MAX_VIEWS 8 /* views consolidated into one launch (splx_plan) */
#define SPLX_BLEND_STRIDE 12 /* floats per Gaussian in splx_projected.blend */
#define SPLX_G2D_STRIDE 12 /* floats per Gaussian in the 2-D gradient buffer, see splx_raster_backward */

typedef struct splx_ctx splx_ctx;

/* Blending / projection constants.  The paper is silent on all of them except the
 * saturation threshold (1e-4); defaults follow BASELINE.json north_star. */
typedef struct {
  float alpha_min;    /* skip a Gaussian at a pixel when alpha < alpha_min        (1/255) */
  float alpha_max;    /* alpha = min(alpha_max, o * exp(power))                   (0.99)  */
  float T_eps;        /* stop before a Gaussian that would take T below T_eps     (1e-4)  */
  float dilation;     /* added to the diagonal of Sigma2D                         (0.3)   */
  float lim_factor;   /* x/z, y/z clamped to +-lim_factor*tan(fov/2) inside J     (1.3)   */
  float radius_floor; /* radius = ceil(3 sqrt(mid + sqrt(max(radius_floor, mid^2-det)))) (0.1) */
} splx_config;

/* Pinhole camera: p_cam = R * mean + t (R row-major), u = fx x/z + cx, v = fy y/z + cy. */
typedef struct {
  float R[9];
  float t[3];
  float fx, fy, cx, cy;
  int32_t width, height;
  float near_z; /* a Gaussian whose camera-space z <= near_z is culled */
} splx_camera;

/* Gaussian parameters Theta_i: SoA over all n Gaussians of all partitions.
 * mean[n,3], log_scale[n,3] (S = exp), quat[n,4] = (w,x,y,z) un-normalised (R),
 * opacity_logit[n] (o = sigmoid), sh[n,16,3] (colour c as SH degree <= 3). 59 floats. */
typedef struct {
  const float *mean, *log_scale, *quat, *opacity_logit, *sh;
  int64_t n;
} splx_gaussians;

/* Same layout; every array is accumulated into (+=). */
typedef struct {
  float *mean, *log_scale, *quat, *opacity_logit, *sh;
  int64_t n;
} splx_gaussian_grads;

/* 2-D attributes of PAPER.md L80 (depth d, 2-D mean, Sigma2D as its inverse "conic").
 * means2d[n,2], depth[n], conic_opacity[n,4] = (A, B, C, o) with power = -0.5(A dx^2 +
 * C dy^2) - B dx dy, rgb[n,3], radius[n] (0 = culled), tiles_touched[n], clamp[n]
 * (bit c set: colour channel c was clamped at 0).  A culled Gaussian gets radius = 0 and tiles_touched = 0; its other
 * attributes are NOT written (no stage reads them: at city scale 90 % of the projected Gaussians are culled and their
 * zeros were most of the projection's memory traffic). */
typedef struct {
  float *means2d, *depth, *conic_opacity, *rgb;
  int32_t *radius;
  uint32_t *tiles_touched;
  uint8_t *clamp;
  /* blend[n,12]: the 48-byte record the blend kernels stage per list entry, written by
   * splx_project from the values above (no new arithmetic beyond the log2(e) pre-scaling of the
   * conic): (u, v, o, depth | -0.5 log2e A, -log2e B, -0.5 log2e C, bits(Gaussian index) |
   * r, g, b, 0).  Not written for a culled Gaussian. */
  float *blend;
} splx_projected;

/* Tile binning of all K partitions.  slot = k * (TX*TY) + tile; key = (slot << 32) |
 * float_bits(depth); val = Gaussian index (global, into the SoA).  keys/vals[capacity];
 * tile_ranges[K*TX*TY][2] = [first, last+1) into keys/vals, (0,0) for an empty tile;
 * num_intersections: DEVICE uint64[2]: [0] = M, the number of intersections (clamped to
 * nothing: if M > capacity the overflowing entries are dropped and splx_check_capacity
 * reports it; with M >= 2^32 nothing is emitted at all); [1] = the number of NON-EMPTY lists that were dropped
 * because their slot carried SPLX_TILE_INVISIBLE (0 whenever the caller's regions are conservative, see
 * splx_footprint_margin). */
typedef struct {
  uint64_t *keys;
  uint32_t *vals;
  uint32_t *tile_ranges;
  uint64_t capacity;
  uint64_t *num_intersections;
  /* Optional (NULL = off), DEVICE uint32[K*TX*TY + SPLX_ORDER_EXTRA], written by splx_bin_sort*: the slots with a
   * non-empty list ordered by DESCENDING list length (to ~3 %: 1024 log-linear length classes, arbitrary order inside
   * a class), then their count at index K*TX*TY, then scratch.  The blend kernels (render_partial with
   * SPLX_PLAN_SPARSE, raster_backward) then hand out their CTAs in this order -- longest list first -- instead
   * of tile order, which shortens the tail of the launch; results are unchanged (a slot's output does not depend on
   * when it is computed).  Built and used for images of up to 16384 tiles (at 4K the order costs more L2 locality
   * than the shorter tail gains: measured); beyond that the buffer is left untouched and tile order is used. */
  uint32_t *slot_order;
} splx_binning;
#define SPLX_ORDER_EXTRA 1025

/* Partial pixels of all K partitions (Eq.3-4): ct[K,H,W,4] =
 * (premultiplied C^k rgb, T^k), d[K,H,W] = D^k = sum d_i alpha_i T_i, n_contrib[K,H,W] =
 * 1 + list position of the pixel's last contributor (0 if none). */
typedef struct {
  float *ct;
  float *d;
  uint32_t *n_contrib;
} splx_partial;

/* ---- context -------------------------------------------------------------------- */
/* cfg NULL = defaults.  cuda_stream is a cudaStream_t (NULL = default stream). */
int splx_create(splx_ctx **out, int device, void *cuda_stream, const splx_config *cfg);
int splx_destroy(splx_ctx *ctx);
const char *splx_last_error(const splx_ctx *ctx); /* ctx may be NULL: last creation error */
int splx_set_stream(splx_ctx *ctx, void *cuda_stream);
/* Number of kernels this context has launched so far (host counter). */
int64_t splx_launch_count(const splx_ctx *ctx);

/* ---- a1 projection: PAPER.md L76 (Sigma = R S S^T R^T), L80 (cull by the mean,
 * Sigma2D = J W Sigma W^T J^T, depth d, 2-D mean).  One thread per Gaussian. */
int splx_project(splx_ctx *ctx, const splx_gaussians *g, const splx_camera *cam, int sh_degree,
                 const splx_projected *out);

/* ---- a2-a4 binning: PAPER.md L81 ("sorted based on ... depth d"), L165 ("in depth
 * order").  part_offsets: HOST array of K+1 Gaussian offsets (partition k owns
 * [part_offsets[k], part_offsets[k+1])).  Result: the STABLE ascending sort of all
 * (key,val) pairs in Gaussian-index emission order, i.e. within a (partition, tile) by
 * depth bits, ties by ascending Gaussian index. */
size_t splx_bin_sort_ws_bytes(int64_t n, uint64_t capacity, int K, const splx_camera *cam);
int splx_bin_sort(splx_ctx *ctx, const splx_projected *proj, int64_t n, int K,
                  const int64_t *part_offsets, const splx_camera *cam, const splx_binning *out,
                  void *ws, size_t ws_bytes);
/* Synchronises the stream and returns SPLX_ERR_CAPACITY if the last splx_bin_sort on
 * `bins` dropped entries; writes M to *m_host (may be NULL).  The only blocking call. */
int splx_check_capacity(splx_ctx *ctx, const splx_binning *bins, uint64_t *m_host);

/* ---- a5 local render: PAPER.md Eq.1 (L84), Eq.3 (L167), Eq.4 (L172).  Grid = K x tiles;
 * one warp per half tile (16 x 8 pixels, 4 pixels per lane), the tile's list staged 32 records
 * at a time in shared memory with cp.async and culled per 8 x 4 pixel block (exact: only
 * entries whose alpha stays below alpha_min on the whole block are dropped).
 * pairs (device uint64[4], may be NULL): pairs[0] += number of list entries walked, summed over
 * pixels (the oracle's unit of work, independent of the culling); pairs[1] += number of
 * (pixel, Gaussian) pairs blended; pairs[2] += alpha evaluations actually executed;
 * pairs[3] += (Gaussian, half tile) items that survived the culling. */
int splx_render_partial(splx_ctx *ctx, const splx_projected *proj, const splx_binning *bins, int K,
                        const splx_camera *cam, const splx_partial *out, uint64_t *pairs);

/* ---- a6 global composition: Eq.5.  Per pixel the K partials are
 * ordered by D^k/(1-T^k) (an empty partial, T == 1, sorts last; ties by smaller k) and
 * accumulated front to back; bg (HOST float[3]) is blended behind everything.
 * image[H,W,3]; T_total[H,W] may be NULL. */
int splx_compose(splx_ctx *ctx, int K, const splx_partial *partials, const splx_camera *cam,
                 const float bg[3], float *image, float *T_total);

/* ---- a7 loss (harness step): mean L1, PAPER.md L95 (L_RGB term).  dL_dimage[count] =
 * sign(image-target) * scale / count; loss_sum (device double, may be NULL) += sum|.|. */
int splx_l1_loss_grad(splx_ctx *ctx, const float *image, const float *target, int64_t count,
                      float scale, float *dL_dimage, double *loss_sum);

/* ---- the full loss of PAPER.md L95 (section 2, step 4): "L = L_RGB + lambda L_D-SSIM".  The paper gives neither lambda
 * nor the SSIM window; reading s33 of DESIGN.md: L_RGB = mean |image - target|; L_D-SSIM = 1 - mean SSIM, SSIM per colour
 * channel over an 11 x 11 Gaussian window (sigma 1.5, weights summing to 1), C1 = 0.01^2, C2 = 0.03^2, pixels outside
 * the image adding nothing to the window sums (zero padding).  image, target, dL_dimage: DEVICE [n_views,H,W,3]
 * (n_views <= SPLX_MAX_VIEWS; cam gives W and H only).  dL_dimage = scale / (n_views H W 3) * (sign(image - target)
 * - lambda d(sum SSIM)/dimage): pass scale = n_views to give every view its own mean, as splx_l1_loss_grad.
 * loss_sum (DEVICE double[2], may be NULL): [0] += sum |image - target|, [1] += sum SSIM, so that
 * L = loss_sum[0] / count + lambda (1 - loss_sum[1] / count) with count = H W 3 per view.  ws: DEVICE scratch of
 * n_views * splx_dssim_ws_floats(cam) floats.  lambda = 0 gives the gradient of splx_l1_loss_grad. */
size_t splx_dssim_ws_floats(const splx_camera *cam);
int splx_dssim_loss_grad(splx_ctx *ctx, int n_views, const splx_camera *cam, const float *image, const float *target,
                         float lambda, float scale, float *dL_dimage, double *loss_sum, float *ws);

/* The same loss and gradient for callers that MUST NOT allocate (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc) and cannot bring a workspace: the scratch of the two kernels (the nine derivative
 * planes that splx_dssim_loss_grad keeps in `ws`) lives in a file-scope `static __device__` array inside the library,
 * SPLX_DSSIM_STATIC_MAX_PIXELS * 9 floats = 9 MiB, which every GPU that loads libsplx.so holds until the process exits.
 * Same arguments, same kernels, same results as splx_dssim_loss_grad.  Limit: n_views * W * H <=
 * SPLX_DSSIM_STATIC_MAX_PIXELS (e.g. one 512 x 512 view); beyond it the call returns SPLX_ERR_WORKSPACE with the two
 * numbers in splx_last_error and launches nothing.  The call performs no cudaMalloc / cudaFree and calls no allocating
 * library routine (the first call on a device looks the array's address up with cudaGetSymbolAddress).  ALL calls on a
 * device share the one array, which keeps the previous call's contents: nothing in it needs to start at zero (the
 * forward kernel writes every plane element the backward kernel reads), but two calls that OVERLAP on the GPU (different
 * streams or contexts on one device) race on it -- serialise them, or use splx_dssim_loss_grad with separate workspaces. */
#define SPLX_DSSIM_STATIC_MAX_PIXELS 262144
int splx_dssim_loss_grad_static(splx_ctx *ctx, int n_views, const splx_camera *cam, const float *image, const float *target,
                                float lambda, float scale, float *dL_dimage, double *loss_sum);

/* ---- a8 composition backward: Eq.6-7.  g_ct[K,H,W,4] =
 * (dL/dC^k rgb, dL/dT^k).  dL_dT_total[H,W] may be NULL.  Overwrites g_ct. */
int splx_compose_backward(splx_ctx *ctx, int K, const splx_partial *partials,
                          const splx_camera *cam, const float bg[3], const float *dL_dimage,
                          const float *dL_dT_total, float *g_ct);

/* ---- a9 rasteriser backward: PAPER.md L184.  Walks each pixel's list in reverse from
 * n_contrib.  g2d[n,SPLX_G2D_STRIDE] += (dL/du, dL/dv, dL/dA, dL/dB, dL/dC, dL/do,
 * dL/dr, dL/dg, dL/db, 0, 0, 0) per Gaussian (warp-reduced, then vector atomics). */
int splx_raster_backward(splx_ctx *ctx, const splx_projected *proj, const splx_binning *bins,
                         int K, const splx_camera *cam, const splx_partial *partials,
                         const float *g_ct, float *g2d);

/* ---- a10 projection backward: exact derivative of splx_project.  Reads
 * g2d and accumulates into grads (+=).  flags: SPLX_PB_CLEAR_G2D zeroes the consumed g2d rows
 * (so the next view can accumulate into g2d again); SPLX_PB_OVERWRITE stores (=) instead of
 * accumulating: EVERY row of every grads array is written (zeros for culled Gaussians and for
 * SH coefficients above sh_degree), so the first view of an iteration needs no zeroed
 * gradient buffer and reads none.  All five grads arrays must be 16-byte aligned. */
#define SPLX_PB_CLEAR_G2D 1
#define SPLX_PB_OVERWRITE 2
int splx_project_backward(splx_ctx *ctx, const splx_gaussians *g, const splx_camera *cam,
                          int sh_degree, const splx_projected *proj, float *g2d, int flags,
                          const splx_gaussian_grads *grads);

/* ---- a8+a9+a10 in one call (BASELINE.json north_star "splx_backward").  ws holds g_ct
 * and g2d; splx_backward_ws_bytes gives its size.  flags: SPLX_PB_OVERWRITE as above (0 = +=). */
size_t splx_backward_ws_bytes(int64_t n, int K, const splx_camera *cam);
int splx_backward(splx_ctx *ctx, int K, const splx_partial *partials, const splx_camera *cam,
                  const float bg[3], const float *dL_dimage, const float *dL_dT_total,
                  const splx_gaussians *g, const splx_projected *proj, const splx_binning *bins,
                  int sh_degree, const splx_gaussian_grads *grads, void *ws, size_t ws_bytes,
                  int flags);

/* ---- a11 Adam (paper silent on the optimiser; north_star names Adam).  Dense,
 * bias-corrected, step is 1-based.  grad_scale multiplies grad first (1/B for B views);
 * if zero_grad != 0 the gradient is zeroed after use.  param/grad/m/v[count]. */
int splx_adam(splx_ctx *ctx, float *param, float *grad, float *m, float *v, int64_t count,
              float lr, float beta1, float beta2, float eps, int step, float grad_scale,
              int zero_grad);

/* The same update for several parameter groups that live back to back in ONE flat buffer
 * (param/grad/m/v[group_offsets[n_groups]]), in a single launch.  group_offsets: HOST array of
 * n_groups+1 float offsets, group_offsets[0] == 0, every offset a multiple of 4 (16-byte
 * vectors never straddle groups); lr: HOST array of n_groups learning rates; 1 <= n_groups <=
 * SPLX_ADAM_MAX_GROUPS.  Elementwise identical to n_groups calls of splx_adam. */
int splx_adam_groups(splx_ctx *ctx, float *param, float *grad, float *m, float *v, int n_groups,
                     const int64_t *group_offsets, const float *lr, float beta1, float beta2,
                     float eps, int step, float grad_scale, int zero_grad);

/* splx_adam_groups with the gradient rows tracked by flags: every group holds `rows` rows of widths[j] floats (HOST
 * int32[n_groups]; row r of group j at group_offsets[j] + r * widths[j]); touched (DEVICE uint8[rows]): the gradient of
 * a row whose flag is clear is ZERO by definition and its memory is never read, so a caller need neither zero nor write
 * the rows no view reached (splx_project_backward_list_plan's `touched` maintains the flags).  Still the DENSE optimiser
 * of DESIGN.md s18: every parameter takes its step (an untouched one with g = 0: its moments decay, it moves along
 * them); elementwise identical to splx_adam_groups on a buffer whose untouched rows are zero.  Flags are not cleared. */
int splx_adam_groups_flagged(splx_ctx *ctx, float *param, const float *grad, float *m, float *v, int n_groups,
                             const int64_t *group_offsets, const int32_t *widths, int64_t rows, const uint8_t *touched,
                             const float *lr, float beta1, float beta2, float eps, int step, float grad_scale);

/* ==== Optional subsystems (BASELINE.json north_star): visibility prediction
 * and conflict-free consolidation of B views into one launch.  Additive:
 * the single-view calls above are the same code run with a one-view plan. ==================== */

/* Per-(partition, tile) visibility state, one byte per slot k*tiles + tile.  A slot whose state
 * is non-zero is SKIPPED: its list is dropped in splx_bin_sort_plan (tile range = (0,0)), so it is
 * neither rendered, composed nor back-propagated (it behaves as the identity partial C=0, T=1). */
#define SPLX_TILE_INVISIBLE 1 /* outside Omega_v^k, the projection of frustum(v) ^ AABB_k (L212, L227) */
#define SPLX_TILE_SATURATED 2 /* every pixel of the tile has prod_{j in front of k} T^j < eps (L213, L231) */

/* splx_plan.flags */
#define SPLX_PLAN_SPARSE 1 /* partial pixels and g_ct of a (partition, tile) slot with an EMPTY list are
                              neither written nor read (exact: such a partial is the identity); compose calls
                              then need the binning.  Without it every slot of a participating partition is
                              written, as in the single-view calls. */

/* One launch = B views of identical size, each partition rendering (at most) one of them.  A
 * conflict-free bucket (L249) maps disjoint partition sets to its views; a single view maps every
 * participating partition to view 0.  Read on the HOST at call time. */
typedef struct {
  int32_t n_views;             /* B in [1, SPLX_MAX_VIEWS] */
  const splx_camera *cams;     /* HOST [B]; identical width and height */
  const int32_t *view_of_part; /* HOST [K]: view index of partition k, or -1 = not a participant of this launch
                                  (its Gaussians are not projected, binned, rendered or differentiated) */
  const uint8_t *tile_state;   /* DEVICE [K*tiles] or NULL (nothing skipped) */
  int32_t flags;
  const float *max_scale;      /* HOST [K] or NULL: an upper bound of exp(log_scale) over the Gaussians of partition k.  Given,
                                  splx_project_plan first tests a Gaussian's MEAN against the half spaces outside which no
                                  Gaussian that small can reach the image (the cut of splx_visible_regions, reading s21) and
                                  reads its scale and rotation only if it passes: 12 instead of 40 bytes for most culled
                                  Gaussians.  Exact as long as the bound holds (a caller that trains refreshes it). */
  int32_t open_slots;          /* 0, or an upper bound of the number of slots (k, t) with partition k participating and
                                  tile_state[k*tiles+t] lacking SPLX_TILE_INVISIBLE, given by a caller who VOUCHES that an
                                  INVISIBLE slot holds no intersection (the conservative regions of splx_visible_regions with
                                  max_scale).  splx_bin_sort* then sorts on a renumbering of the open slots -- a city view
                                  leaves 85-90 % of the slots invisible, and 16 bits instead of 17-18 are two radix passes
                                  over the intersections instead of three -- with the same keys, vals and ranges.  Should a
                                  key fall into an INVISIBLE slot all the same (or into an open slot beyond the bound), it is
                                  carried behind every list under slot number K*tiles + 1, gets no range, and is counted in
                                  num_intersections[1].  The renumbering is used where it saves a radix pass; a NEGATIVE value
                                  (bound = -open_slots) forces it (tests).  Needs slot_map. */
  const uint32_t *slot_map;    /* DEVICE [splx_slot_map_words(K, cams)] or NULL (no renumbering): the numbering of the open slots
                                  and its inverse, written ONCE by splx_slot_map for this (tile_state INVISIBLE bits,
                                  view_of_part, open_slots) -- a caller who changes one of them rebuilds it; the saturated bits
                                  that composition rewrites every iteration do not enter it */
} splx_plan;

/* The slot numbering behind splx_plan.open_slots: slot_map_out (DEVICE uint32[splx_slot_map_words]) receives, for the plan's
 * tile_state, view_of_part and |open_slots| (plan->slot_map itself is ignored), cmap[K*tiles] = number of every open slot in
 * slot order (others: |open_slots| + 1) followed by inv[|open_slots| + 2] = the way back.  One small launch on the context's
 * stream; the plan that later carries slot_map must have the same three inputs. */
size_t splx_slot_map_words(int K, const splx_camera *cam);
int splx_slot_map(splx_ctx *ctx, int K, const splx_plan *plan, uint32_t *slot_map_out);


/* Geometric visibility (L212, L227): HOST computation, no device work, ctx not needed.  n_boxes axis-aligned boxes
 * [aabb_lo[j], aabb_hi[j]] (HOST float[n_boxes][3], world space), box j belonging to partition box_part[j] (HOST
 * int32[n_boxes]; NULL = one box per partition, n_boxes == K): a partition is the UNION of its boxes (the cell of L155,
 * or a finer cover of it by sub-cells).
 *  - max_scale NULL, the plain region of L212: the convex polyhedron box ^ {z >= near_z} (no far plane) is
 *    projected; tile_state[k*tiles + t] (HOST out) = 0 if tile t's pixel-area rectangle meets the projected region of
 *    some box j of partition k, else SPLX_TILE_INVISIBLE.
 *  - max_scale given (HOST float[n_boxes]: the largest scale exp(log_scale) among the Gaussians whose MEAN lies in box j;
 *    the boxes are then boxes of means; cfg NULL = defaults), the CONSERVATIVE region of reading s21: Gaussians
 *    belong to a partition by their mean (L155) but their footprints stick out of its box (L474).  With
 *    c^2 = max(fx, fy)^2 (1 + limx^2 + limy^2), e = dilation + sqrt(radius_floor): the box is first cut down to the means
 *    that can reach the image at all, Q = box ^ {z >= near_z} ^ {-(cx + g) z - h <= fx x <= (W - cx + g) z + h} ^ {same in
 *    y}, g = 2.5 + 3 sqrt(e), h = 3 c max_scale; on Q every footprint square has half side <= 3 sqrt(c^2 max_scale^2 /
 *    z_min(Q)^2 + e) + 1, so tile t is marked visible iff its rectangle grown by m = 3 sqrt(c^2 max_scale^2 / z_min^2 + e)
 *    + 3.5 px meets the projection of Q.  Then a slot marked SPLX_TILE_INVISIBLE has an EMPTY list and a non-participant
 *    no visible Gaussian: skipping them changes no pixel and no gradient.  The finer the boxes the tighter the regions
 *    (scenes.partition_boxes covers every partition with a grid of sub-cells).
 * participants (HOST out, may be NULL): bit k set iff partition k has at least one visible tile (GetParticipants,
 * L249).  Double precision.  Returns SPLX_OK or SPLX_ERR_INVALID_ARG (K > 64, null pointers, lo > hi, near_z <= 0, a
 * negative scale, box_part out of range). */
int splx_visible_regions(int K, int n_boxes, const int32_t *box_part, const float *aabb_lo, const float *aabb_hi,
                         const float *max_scale, const splx_config *cfg, const splx_camera *cam, uint8_t *tile_state,
                         uint64_t *participants);

/* Conflict-free view consolidation (L249): greedy bucketing in view order.  View v goes to the first
 * bucket none of whose views shares a partition with participants[v] and that holds fewer than
 * max_views_per_bucket views (<= SPLX_MAX_VIEWS), else opens a new bucket.  HOST in/out.
 * bucket_of_view[n_views] and *n_buckets are written. */
int splx_schedule_views(int n_views, const uint64_t *participants, int max_views_per_bucket,
                        int32_t *bucket_of_view, int32_t *n_buckets);

/* The stages under a plan.  part_offsets: HOST [K+1] as in splx_bin_sort.  Arrays indexed by view
 * have a leading dimension B = plan->n_views: image[B,H,W,3], T_total[B,H,W], dL_dimage[B,H,W,3].
 * Arrays indexed by partition keep their [K,...] layout (a partition belongs to one view). */
int splx_project_plan(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                      const splx_plan *plan, int sh_degree, const splx_projected *out);
int splx_bin_sort_plan(splx_ctx *ctx, const splx_projected *proj, int64_t n, int K,
                       const int64_t *part_offsets, const splx_plan *plan, const splx_binning *out,
                       void *ws, size_t ws_bytes);
/* splx_project_plan in two halves ("standard 3DGS rendering procedure", steps a1 and the colour of s13):
 * splx_project_geometry_plan writes everything splx_project_plan writes EXCEPT the colour (rgb, clamp, blend[8..10]);
 * splx_project_colour_list_plan then computes the colour of the entries of `visible` (DEVICE uint32[*num_visible],
 * *num_visible a DEVICE uint64: the list splx_bin_sort_visible returns after splx_bin_sort_plan on the geometry).
 * Together bit-equal to splx_project_plan on every visible Gaussian; the work of the colour follows the visible
 * count, not the partition sizes (on a city view ~13 % of the participating Gaussians are visible, scattered over the
 * warps).  The colour must be complete before splx_render_partial_plan / splx_project_backward_* read it. */
int splx_project_geometry_plan(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                               const splx_plan *plan, const splx_projected *out);
int splx_project_colour_list_plan(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                                  const splx_plan *plan, int sh_degree, const splx_projected *out,
                                  const uint32_t *visible, const uint64_t *num_visible);
int splx_render_partial_plan(splx_ctx *ctx, const splx_projected *proj, const splx_binning *bins, int K,
                             const splx_plan *plan, const splx_partial *out, uint64_t *pairs);
/* bins: needed with SPLX_PLAN_SPARSE or tile_state_out, else may be NULL.  tile_state_out (DEVICE
 * [K*tiles], may be NULL, may alias plan->tile_state): saturation detection "at no additional
 * cost" during composition (L231): for every participating partition k and tile t,
 * out = (in & SPLX_TILE_INVISIBLE) | (SPLX_TILE_SATURATED if at EVERY pixel of the tile the product
 * of the T^j composited in front of k is < sat_eps); `in` = plan->tile_state or 0.  A partition
 * that is the identity at a pixel stands behind all others there (its front product is T_total). */
int splx_compose_plan(splx_ctx *ctx, int K, const splx_partial *partials, const splx_binning *bins,
                      const splx_plan *plan, const float bg[3], float *image, float *T_total,
                      float sat_eps, uint8_t *tile_state_out);
/* a6 + a7 + a8 in one pass over the partial pixels: splx_compose_plan, then the mean-L1 gradient of
 * splx_l1_loss_grad over the B*H*W*3 values of `image` against `targets` [B,H,W,3] (scale as there: pass B to
 * give every view its own mean), then splx_compose_backward_plan with dL_dT_total = NULL -- statement by
 * statement the same arithmetic, without the second read of the partials and without dL/dimage ever leaving
 * the SM.  image, T_total (may be NULL), g_ct, loss_sum (device double, += sum|.|, may be NULL) and
 * tile_state_out are written as by the three staged calls. */
int splx_compose_l1_backward_plan(splx_ctx *ctx, int K, const splx_partial *partials,
                                  const splx_binning *bins, const splx_plan *plan, const float bg[3],
                                  const float *targets, float scale, float *image, float *T_total,
                                  double *loss_sum, float *g_ct, float sat_eps, uint8_t *tile_state_out);
int splx_compose_backward_plan(splx_ctx *ctx, int K, const splx_partial *partials,
                               const splx_binning *bins, const splx_plan *plan, const float bg[3],
                               const float *dL_dimage, const float *dL_dT_total, float *g_ct);
int splx_raster_backward_plan(splx_ctx *ctx, const splx_projected *proj, const splx_binning *bins, int K,
                              const splx_plan *plan, const splx_partial *partials, const float *g_ct,
                              float *g2d);
/* With SPLX_PB_OVERWRITE the gradient rows of NON-participating partitions are written as zeros. */
int splx_project_backward_plan(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                               const splx_plan *plan, int sh_degree, const splx_projected *proj,
                               float *g2d, int flags, const splx_gaussian_grads *grads);
/* The list of VISIBLE Gaussians (global indices, ascending) that the last splx_bin_sort[_plan] on workspace `ws`
 * left there, and its device-side count: pointers INTO the workspace (device memory), valid until the next
 * splx_bin_sort on it.  Same n, capacity, K, cam as that call.  Host computation only. */
int splx_bin_sort_visible(const void *ws, int64_t n, uint64_t capacity, int K, const splx_camera *cam,
                          const uint32_t **visible, const uint64_t **num_visible);
/* ---- cross-boundary per-ray filtering (appendix 8.1, Fig. 25; readings: DESIGN.md s32) ----
 * "We remove a Gaussian G_i in Q_cross from the ray r of pixel p if and only if its depth d_i falls within the
 * overlapped depth interval D_overlap and p lies in the overlapped pixel region Omega_v^k ^ Omega_v^s."
 *
 * splx_cross_sets (view independent; once per change of the Gaussians): cross_mask[i] (DEVICE uint64[n], out) gets
 * bit s set iff Gaussian i of partition k != s is in Q_cross(k, s): the axis-aligned box around its
 * support_sigma-sigma ellipsoid (half extent along axis a = support_sigma * sqrt(Sigma_aa), Sigma = R S^2 R^T)
 * meets the closed CELL box [cell_lo[s], cell_hi[s]] (HOST float[K][3]).  fp32. */
int splx_cross_sets(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                    const float *cell_lo, const float *cell_hi, float support_sigma, uint64_t *cross_mask);
/* D^k of a plan (HOST computation, double precision rounded to float): part_depth_range[2k], [2k+1] (HOST out) =
 * the smallest and largest camera-space z over the corners of box k under the view plan->view_of_part[k];
 * (+inf, -inf) for a partition that renders no view. */
int splx_cross_depth_ranges(int K, const float *aabb_lo, const float *aabb_hi, const splx_plan *plan,
                            float *part_depth_range);
/* splx_bin_sort_plan with the filter: the (Gaussian i of partition k, tile t) pair is left out of the list of
 * (k, t) iff for some partition s: bit s of cross_mask[i], s renders the view k renders, depth[i] lies in the closed
 * interval D^k ^ D^s of part_depth_range (HOST float[2K]), and tile t is in Omega^s (plan->tile_state[s, t] without
 * SPLX_TILE_INVISIBLE; no tile_state = every tile).  The order of the remaining entries is unchanged, so every
 * later stage (forward and backward) simply never sees the pair.  *num_intersections counts the pairs KEPT; the
 * capacity must still hold the unfiltered count (removed pairs are sorted to the end of the key buffer: keys and
 * vals beyond *num_intersections are scratch).  cross_mask NULL = splx_bin_sort_plan. */
int splx_bin_sort_filtered_plan(splx_ctx *ctx, const splx_projected *proj, int64_t n, int K,
                                const int64_t *part_offsets, const splx_plan *plan, const uint64_t *cross_mask,
                                const float *part_depth_range, const splx_binning *out, void *ws, size_t ws_bytes);
/* The entries of that list whose g2d row ([n, SPLX_G2D_STRIDE], as splx_raster_backward* leaves it) is not all zero,
 * compacted into scratch of the same workspace (valid until the next splx_bin_sort* on it): *rows = DEVICE uint32 list (in no
 * particular order), *num_rows = its DEVICE uint64 count.  A visible Gaussian that no pixel blended -- hidden behind opaque
 * surfaces: about half of the visible ones on a city view -- has an all-zero row and, the projection backward being linear
 * in it, a zero gradient: splx_project_backward_list_plan over (*rows, *num_rows) WITH `touched` gives the same gradients
 * under the flag semantics (an unflagged row counts as zero) for half the work.  One launch on the context's stream. */
int splx_bin_sort_gradient_rows(splx_ctx *ctx, void *ws, int64_t n, uint64_t capacity, int K, const splx_camera *cam,
                                const float *g2d, const uint32_t **rows, const uint64_t **num_rows);
/* splx_project_backward_plan in += mode over the visible Gaussians only: the rows processed are the entries of
 * `visible` (device uint32[*num_visible], *num_visible a device uint64) instead of every Gaussian of the
 * participating partitions -- same result (a culled Gaussian has no gradient), work proportional to the visible
 * count.  flags: SPLX_PB_CLEAR_G2D or 0. */
int splx_project_backward_list_plan(splx_ctx *ctx, const splx_gaussians *g, int K, const int64_t *part_offsets,
                                    const splx_plan *plan, int sh_degree, const splx_projected *proj,
                                    float *g2d, int flags, const splx_gaussian_grads *grads,
                                    const uint32_t *visible, const uint64_t *num_visible, uint8_t *touched);
/* touched (device uint8[n], may be NULL): the flags of the visible-only optimiser.  A row whose flag is clear has no
 * gradient yet in this iteration: the call STORES its gradient (whatever the row held) and sets the flag; a row whose
 * flag is set is accumulated into.  With it no gradient buffer is ever zeroed or overwritten wholesale.
 *
 * splx_adam_sparse -- an OPTION outside the paper (it changes the optimiser: DESIGN.md s31): the Adam step of
 * splx_adam on the Gaussians whose flag is set only, all 59 parameters of a row with the learning rate of their
 * group (lr: HOST float[5] for mean, log_scale, quat, opacity_logit, sh); the others keep parameters and both
 * moments unchanged.  Clears the flags it consumes.  step is 1-based and global (bias correction as splx_adam). */
int splx_adam_sparse(splx_ctx *ctx, const splx_gaussian_grads *params, const splx_gaussian_grads *grads,
                     const splx_gaussian_grads *m, const splx_gaussian_grads *v, uint8_t *touched,
                     const float lr[5], float beta1, float beta2, float eps, int step, float grad_scale);
int splx_backward_plan(splx_ctx *ctx, int K, const int64_t *part_offsets, const splx_plan *plan,
                       const splx_partial *partials, const float bg[3], const float *dL_dimage,
                       const float *dL_dT_total, const splx_gaussians *g, const splx_projected *proj,
                       const splx_binning *bins, int sh_degree, const splx_gaussian_grads *grads,
                       void *ws, size_t ws_bytes, int flags);


/* ==== One whole training iteration behind one call (the sequencing of PAPER.md Fig. 9, on one GPU) =========
 * The stages above are the parity surface; a trainer calls THIS: a1-a10 for every bucket of views of an iteration
 * (and optionally a11), issued by the library on the context's stream plus three internal streams -- projection and
 * binning of bucket g+1 run beside the blending of bucket g when a second splx_frontset is given, host copies run on
 * their own streams beside the kernels.  Nothing here synchronises; every internal stream is joined back into the
 * context's stream before the call returns, so the call may be captured into a CUDA graph by the caller. */

/* Buffers of a1-a4 for one bucket in flight. */
typedef struct {
  splx_projected proj;
  splx_binning bins;
  void *ws;        /* DEVICE, splx_bin_sort_ws_bytes(n, bins.capacity, K, cam) */
  size_t ws_bytes;
} splx_frontset;

/* Every caller-owned buffer of an iteration.  DEVICE pointers unless marked HOST. */
typedef struct {
  splx_gaussian_grads params;   /* Theta, SoA over all K partitions; only splx_adam_cfg writes it */
  splx_gaussian_grads grads;    /* same layout: the FIRST bucket of an iteration stores, later ones accumulate */
  int32_t K;
  const int64_t *part_offsets;  /* HOST [K+1] */
  int32_t sh_degree;
  float bg[3];
  splx_frontset front[2];       /* front[1].ws == NULL: buckets run strictly one after the other */
  splx_partial partials;        /* [K,H,W,*] */
  float *g_ct;                  /* [K,H,W,4] */
  float *g2d;                   /* [n,SPLX_G2D_STRIDE], all zero on entry; left all zero */
  float *images;                /* [max_views,H,W,3]: image of view v of the iteration at slot v */
  float *T_totals;              /* [max_views,H,W] or NULL */
  float *targets;               /* [max_views,H,W,3]: staging of HOST targets (SPLX_ITER_HOST), else unused / NULL */
  float *g_images;              /* [max_views,H,W,3]: dL/dimage, only used when lambda_dssim > 0, else may be NULL */
  float *dssim_ws;              /* splx_dssim_ws_floats(W,H) floats per view x max_views, only when lambda_dssim > 0 */
  double *loss_sum;             /* double[2]: [0] += sum |image-target| (cleared by the call), [1] += sum SSIM */
  int32_t max_views;
  const uint64_t *cross_mask;   /* Q_cross masks [n] (splx_cross_sets) or NULL: cross-boundary filtering off */
  uint8_t *touched;             /* [n] or NULL.  Given: the call clears it, every bucket's projection backward walks the
                                   binning's list of visible Gaussians, STORES the gradient of a row it reaches first and
                                   sets its flag, accumulates into flagged rows: grads is valid on flagged rows only and
                                   no pass over all n rows ever zeroes or writes it.  NULL: the first bucket stores every
                                   row of grads (zeros where nothing is visible), later buckets accumulate. */
} splx_trainset;

/* One bucket = one launch per stage (a conflict-free set of views, L249). */
typedef struct {
  splx_plan plan;               /* plan.cams / view_of_part HOST, plan.tile_state DEVICE */
  const int32_t *view_index;    /* HOST [plan.n_views]: plan view b is view view_index[b] of the iteration */
  uint8_t *tile_state_out;      /* DEVICE [K*tiles] or NULL: saturation detection (may alias plan.tile_state) */
  const float *part_depth_range;/* HOST [2K] (splx_cross_depth_ranges) when trainset.cross_mask is set, else NULL */
} splx_bucket;

/* Optional a11 at the end of the iteration: dense Adam over the flat buffers -- splx_adam_groups, or with
 * trainset.touched splx_adam_groups_flagged (same result; the gradient rows no view reached are neither zeroed, written
 * nor read) -- or, with trainset.touched and `sparse`, the visible-only option (splx_adam_sparse on the SoA sets). */
typedef struct {
  float *param, *grad, *m, *v;          /* flat buffers holding the five groups back to back */
  int32_t n_groups;
  const int64_t *group_offsets;         /* HOST [n_groups+1] */
  const float *lr;                      /* HOST [n_groups] */
  float beta1, beta2, eps;
  int32_t step;                         /* 1-based */
  const int32_t *widths;                /* HOST [n_groups]: floats per row of every group (needed with trainset.touched) */
  int32_t sparse;                       /* with trainset.touched: 1 = the visible-only option (splx_adam_sparse), 0 = dense */
  splx_gaussian_grads m_soa, v_soa;     /* only read with sparse */
} splx_adam_cfg;

#define SPLX_ITER_HOST 1   /* targets[v] / images_out[v] / loss_out / m_out are pinned HOST pointers */
#define SPLX_ITER_KEEP_ZERO_ROWS 8     /* with trainset.touched: the projection backward runs over EVERY visible Gaussian and flags
                                          it, also one whose gradient is exactly zero (the row set of the visible-only optimiser
                                          option).  Default: over splx_bin_sort_gradient_rows' list */
#define SPLX_ITER_FUSED_PROJECTION 4   /* a1 as ONE kernel (splx_project_plan: the colour of every visible Gaussian inside the
                                          projection).  Default: the geometry half (splx_project_geometry_plan), the binning, then
                                          the colour of the binning's list of visible Gaussians (splx_project_colour_list_plan) --
                                          faster where most participating Gaussians are culled (city views: 3.9 against 4.9 ms at
                                          100 M Gaussians), slower where most are visible (aerial_1M: 0.113 against 0.072 ms).
                                          Bit-identical results. */
typedef struct {
  int32_t flags;
  float sat_eps;         /* threshold of the saturation detection (bucket.tile_state_out) */
  float lambda_dssim;    /* 0: L = mean L1 (a6+a7+a8 fused); > 0: L = mean L1 + lambda * (1 - mean SSIM) */
} splx_iter_opts;

/* n_views views in n_buckets buckets; every view belongs to exactly one bucket.  targets[v]: [H,W,3] of view v
 * (DEVICE, or pinned HOST with SPLX_ITER_HOST: copied to trainset.targets on the library's upload stream while the
 * first bucket is projected and binned).  The loss of view v is its own mean; the gradients of the views add up
 * (grad_scale 1/n_views is applied by a11).  With SPLX_ITER_HOST: images_out[v] (HOST [H,W,3] or NULL entries; the
 * array itself may be NULL) receives image v as soon as its bucket is composed, loss_out (HOST double[2] or NULL)
 * receives loss_sum; without the flag both must be NULL.  m_out (pinned HOST uint64[n_buckets] or NULL, with or
 * without the flag) receives the intersection count of every bucket: compare it with bins.capacity after a
 * synchronisation -- a bucket with more intersections dropped its farthest keys.  adam NULL = no optimiser step. */
int splx_iteration(splx_ctx *ctx, const splx_trainset *ts, int n_buckets, const splx_bucket *buckets, int n_views,
                   const float *const *targets, float *const *images_out, double *loss_out, uint64_t *m_out,
                   const splx_iter_opts *opts, const splx_adam_cfg *adam);

/* ---- measurement helper (not part of the method): the micro-benchmarks behind the ALU rooflines of the blend loops
 * (an FMA loop and an ex2 loop measured on the box).  kind 0: FP32 FMA chains, *work (HOST out) = flops
 * of the launch (2 per FMA); kind 1: ex2.approx chains, *work = ex2 evaluations.  One asynchronous launch over all SMs;
 * the caller times it with CUDA events on the context's stream.  sink: DEVICE float[1] (never written in practice). */
int splx_microbench(splx_ctx *ctx, int kind, int64_t iters, float *sink, double *work);

#ifdef __cplusplus
}
#endif
#endif /* SPLX_H_ */
