// render.cu -- step a5 (local per-partition render) and step a9 (its backward).
// PAPER.md Eq.1 (L84): alpha_i = o_i exp(-1/2 (x-mu)^T Sigma2D^-1 (x-mu));  Eq.3 (L167):
// C^m = sum c_i alpha_i prod_{j<i}(1-alpha_j);  Eq.4 (L172): T^m = prod (1-alpha_i) and the partial
// depth D^m (read as sum d_i alpha_i T_i).  Blending rules (s2): skip power > 0,
// alpha = min(alpha_max, .), skip alpha < alpha_min, stop BEFORE a Gaussian that would take T
// below T_eps.  Backward: PAPER.md L184 ("the per-Gaussian gradient backpropagates through the
// intermediate partial pixel"), with dL/dC^m and dL/dT^m coming from Eq.6-7 (compose.cu).
//
// Both kernels are instruction-issue bound (profiles/r01a_ncu_blend_kernels.md: 90 % issue-slot utilisation, DRAM 2 %),
// so the design minimises instructions per useful (pixel, Gaussian) pair:
//   * grid = (tiles, K), CTA = 2 autonomous warps, one per HALF tile (16 x 8 pixels).  A lane owns 4
//     pixels, one in each 8 x 4 block ("slot") of the half tile, so the record of a Gaussian is read
//     from shared memory once per 4 pixel evaluations and the x / y terms of the quadratic form are
//     shared between the slots.  No __syncthreads anywhere: a warp stages its own copy of the list.
//   * the tile's sorted list is staged 32 records (48 B each, splx_projected.blend) at a time with
//     16-byte cp.async into a two-deep ring, one record per lane, prefetched a batch ahead.
//   * exact culling: the lane that staged a record computes, per slot, the maximum of the Gaussian's
//     exponent over the slot's pixel rectangle (closed form for a concave quadratic on a box); a slot
//     whose best pixel stays below alpha_min is skipped for that Gaussian.  Only pairs that the
//     alpha_min rule would skip anyway are dropped, so results are bit-identical to walking the list.
//   * backward: a lane accumulates the six moments of dL/dG over its 4 pixels and the colour sums in
//     registers and stores its nine partial gradients to a shared staging block (9 conflict-free
//     stores per (Gaussian, half tile) item); every seven items the 63 rows are summed over the lanes
//     (one row per lane, rotating column: no bank conflict) and leave as two rounds of 32 distinct
//     atomics.  ~28 instructions per item instead of ~75 for a shuffle tree + selects.
#include "common.cuh"

namespace {

constexpr int WARPS = 2;                 // warps per CTA = half tiles per tile
constexpr int BLOCK = 32 * WARPS;
constexpr int NBUF = 2;                  // staging ring depth
constexpr float LN2 = 0.6931471805599453f;
constexpr float CULL_MARGIN = 0.02f;     // in log2(alpha): 1.4 % slack, far above fp32 rounding of the exponent
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Staging ring of one warp: [buffer][quarter of the record][entry].  Quarter 0 = (u, v, o, depth),
// 1 = (A', B', C', bits(index)), 2 = (r, g, b, 0).
struct Ring { float4 q[NBUF][3][32]; };

// Issue the copies of list entry `idx` (if inside [.., end)) into slot `lane` of ring buffer `buf`.
__device__ __forceinline__ void stage_issue(Ring& ring, int buf, int lane, const float* __restrict__ blend,
                                            const uint32_t* __restrict__ vals, uint32_t idx, uint32_t end) {
  if (idx < end) {
    const float* src = blend + (size_t)SPLX_BLEND_STRIDE * __ldg(vals + idx);
    cp_async16(&ring.q[buf][0][lane], src);
    cp_async16(&ring.q[buf][1][lane], src + 4);
    cp_async16(&ring.q[buf][2][lane], src + 8);
  }
  cp_async_commit();
}

// Maximum over the rectangle [x0,x1] x [y0,y1] of q(dx,dy) = A dx^2 + B dx dy + C dy^2 with
// (dx,dy) = (gx - x, gy - y), for a negative definite form (A, C < 0).  The maximiser lies on one
// of the (at most two) box edges that face the centre; on the line through the clamped centre
// coordinate the 1-D optimum is the unconstrained one clamped to the edge's extent.
__device__ __forceinline__ float quad_max_rect(float gx, float gy, float A, float B, float C, float hBC, float hBA,
                                               float x0, float x1, float y0, float y1) {
  const float dxc = gx - fminf(fmaxf(gx, x0), x1);
  const float dyc = gy - fminf(fmaxf(gy, y0), y1);
  const float dy1 = fminf(fmaxf(hBC * dxc, gy - y1), gy - y0);     // hBC = -B / (2C)
  const float q1 = A * dxc * dxc + (B * dxc + C * dy1) * dy1;
  const float dx2 = fminf(fmaxf(hBA * dyc, gx - x1), gx - x0);     // hBA = -B / (2A)
  const float q2 = C * dyc * dyc + (B * dyc + A * dx2) * dx2;
  return fmaxf(q1, q2);
}

// 4-bit mask of the slots of this warp's half tile on which the Gaussian can reach alpha_min.
// (X0, Y0) = pixel coordinates of the half tile's first pixel; slot s covers columns 8(s&1)..+7 and
// rows 4(s>>1)..+3; pixel i samples i + 0.5.
__device__ __forceinline__ unsigned cull_mask(const float4 a, const float4 b, float X0, float Y0, float log2_amin) {
  const float A = b.x, B = b.y, C = b.z, o = a.z;
  if (!(A < 0.f) || !(C < 0.f) || !(log2_amin > -1e30f)) return 0xFu;   // degenerate conic or alpha_min == 0: keep all
  const float tau = log2_amin - lg2_approx(o) - CULL_MARGIN;           // keep the slot if max exponent >= tau
  const float hBC = -0.5f * __fdividef(B, C), hBA = -0.5f * __fdividef(B, A);
  unsigned m = 0;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    const float x0 = X0 + (float)(8 * (s & 1)) + 0.5f, y0 = Y0 + (float)(4 * (s >> 1)) + 0.5f;
    const float qm = quad_max_rect(a.x, a.y, A, B, C, hBC, hBA, x0, x0 + 7.0f, y0, y0 + 3.0f);
    if (!(qm < tau)) m |= 1u << s;
  }
  return m;
}

// The alpha of one (pixel, Gaussian) pair: the same instruction sequence in the forward and the
// backward, so that both take identical skip / clamp decisions.  adx = A' dx, bdx = B' dx, cdy = C' dy.
__device__ __forceinline__ bool eval_alpha(float dx, float dy, float adx, float bdx, float cdy, float o, float amin,
                                           float amax, float& G, float& alpha, bool& clamped) {
  const float p2 = fmaf(adx, dx, fmaf(cdy, dy, __fmul_rn(bdx, dy)));
  G = ex2_approx(p2);
  const float a = __fmul_rn(o, G);
  clamped = a >= amax;
  alpha = fminf(amax, a);
  return (p2 <= 0.0f) && (alpha >= amin);
}

constexpr int FWD_MIN_CTAS = 14;   // 71 registers; a sweep 12..20 showed no effect below spilling: issue-bound
template <bool COUNT>
__global__ void __launch_bounds__(BLOCK, FWD_MIN_CTAS)
k_render_fwd(const float* __restrict__ blend, const uint32_t* __restrict__ vals, const uint32_t* __restrict__ ranges,
             int W, int H, int TX, int ntiles, splx_config cfg, const __grid_constant__ PartView pv, int sparse,
             float* __restrict__ out_ct, float* __restrict__ out_d, uint32_t* __restrict__ out_n,
             unsigned long long* pairs, const uint32_t* __restrict__ order, uint32_t nslots) {
  __shared__ Ring rings[WARPS];
  int tile = blockIdx.x, k = blockIdx.y;
  if (order) {                             // CTAs handed out longest list first (splx_binning.slot_order)
    if (blockIdx.x >= order[nslots]) return;
    const uint32_t s = order[blockIdx.x];
    k = (int)(s / (uint32_t)ntiles); tile = (int)(s - (uint32_t)k * (uint32_t)ntiles);
  }
  if (pv.v[k] < 0) return;                 // the partition does not participate in this launch
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  Ring& ring = rings[warp];
  const int X0 = (tile % TX) * SPLX_TILE, Y0 = (tile / TX) * SPLX_TILE + 8 * warp;
  const int pxi = X0 + (lane & 7), pyi = Y0 + (lane >> 3);          // slot 0 pixel; slot s adds (8(s&1), 4(s>>1))
  const float px0 = (float)pxi + 0.5f, px1 = px0 + 8.0f, py0 = (float)pyi + 0.5f, py1 = py0 + 4.0f;
  const uint32_t r0 = ranges[2 * ((size_t)k * ntiles + tile)], r1 = ranges[2 * ((size_t)k * ntiles + tile) + 1];
  if (sparse && r0 == r1) return;          // SPLX_PLAN_SPARSE: an empty list is the identity partial, never stored
  const float log2_amin = cfg.alpha_min > 0.f ? log2f(cfg.alpha_min) : -INFINITY;

  float T[4], C0[4], C1[4], C2[4], D[4];
  uint32_t last[4], wdone[4];
  unsigned done = 0;                       // bit s: slot s finished (exit rule fired, or outside the image)
  uint32_t blended = 0, evaluated = 0, items = 0;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    T[s] = 1.f; C0[s] = C1[s] = C2[s] = D[s] = 0.f; last[s] = 0; wdone[s] = 0;
    if (pxi + 8 * (s & 1) >= W || pyi + 4 * (s >> 1) >= H) done |= 1u << s;
  }
  const unsigned outside = done;

  if (r0 < r1 && !__all_sync(FULL, done == 0xFu)) {
    stage_issue(ring, 0, lane, blend, vals, r0 + lane, r1);
    int buf = 0;
    for (uint32_t start = r0; start < r1; start += 32, buf ^= 1) {
      stage_issue(ring, buf ^ 1, lane, blend, vals, start + 32 + lane, r1);
      cp_async_wait<1>();
      __syncwarp();
      unsigned m = 0;
      if (start + lane < r1) m = cull_mask(ring.q[buf][0][lane], ring.q[buf][1][lane], (float)X0, (float)Y0, log2_amin);
      const unsigned open_slots = ~__reduce_and_sync(FULL, done) & 0xFu;   // slots not yet finished in every lane
      m &= open_slots;
      unsigned live = __ballot_sync(FULL, m != 0);
      while (live) {
        const int j = __ffs(live) - 1;
        live &= live - 1;
        const unsigned mj = __shfl_sync(FULL, m, j);
        const float4 a = ring.q[buf][0][j], b = ring.q[buf][1][j], c = ring.q[buf][2][j];
        const uint32_t pos = start - r0 + (uint32_t)j + 1;     // 1-based list position, as in n_contrib
        const float dxs[2] = {__fsub_rn(a.x, px0), __fsub_rn(a.x, px1)};
        const float dys[2] = {__fsub_rn(a.y, py0), __fsub_rn(a.y, py1)};
        const float adx[2] = {__fmul_rn(b.x, dxs[0]), __fmul_rn(b.x, dxs[1])};
        const float bdx[2] = {__fmul_rn(b.y, dxs[0]), __fmul_rn(b.y, dxs[1])};
        const float cdy[2] = {__fmul_rn(b.z, dys[0]), __fmul_rn(b.z, dys[1])};
        if (COUNT) ++items;
#pragma unroll
        for (int s = 0; s < 4; ++s) {
          if (!((mj >> s) & 1)) continue;     // warp-uniform
          if (COUNT) ++evaluated;
          float G, alpha; bool clamped;
          const bool ok = eval_alpha(dxs[s & 1], dys[s >> 1], adx[s & 1], bdx[s & 1], cdy[s >> 1], a.z, cfg.alpha_min,
                                     cfg.alpha_max, G, alpha, clamped);
          // branch-free: a pixel that skips the entry blends it with weight 0
          const bool live_px = ok && !((done >> s) & 1);
          const float Tn = T[s] * (1.0f - alpha);
          const bool stop = live_px && (Tn < cfg.T_eps);      // the exit rule fires BEFORE this entry is applied
          const bool take = live_px && !(Tn < cfg.T_eps);
          const float w = take ? alpha * T[s] : 0.0f;
          C0[s] = fmaf(w, c.x, C0[s]); C1[s] = fmaf(w, c.y, C1[s]); C2[s] = fmaf(w, c.z, C2[s]);
          D[s] = fmaf(w, a.w, D[s]);
          T[s] = take ? Tn : T[s];
          last[s] = take ? pos : last[s];
          if (stop) done |= 1u << s;
          if (COUNT) { if (stop) wdone[s] = pos; if (take) ++blended; }
        }
      }
      __syncwarp();
      if (__all_sync(FULL, done == 0xFu)) break;
    }
    cp_async_wait<0>();
  }

  uint32_t walked = 0;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    if ((outside >> s) & 1) continue;
    const int x = pxi + 8 * (s & 1), y = pyi + 4 * (s >> 1);
    const size_t pix = ((size_t)k * H + y) * W + x;
    *reinterpret_cast<float4*>(out_ct + 4 * pix) = make_float4(C0[s], C1[s], C2[s], T[s]);
    out_d[pix] = D[s];
    out_n[pix] = last[s];
    if (COUNT) walked += ((done >> s) & 1) ? wdone[s] : (r1 - r0);
  }
  if (COUNT && pairs) {
    const uint32_t wsum = __reduce_add_sync(FULL, walked);
    const uint32_t bsum = __reduce_add_sync(FULL, blended);
    if (lane == 0 && wsum) {
      atomicAdd(pairs, (unsigned long long)wsum);
      atomicAdd(pairs + 1, (unsigned long long)bsum);
      atomicAdd(pairs + 2, 32ull * evaluated);
      atomicAdd(pairs + 3, (unsigned long long)items);
    }
  }
}

// Staging block of one warp in the backward: STAGE_ITEMS (Gaussian, half tile) items x 9 gradient values x 32
// lane partials.  63 rows = two rounds of 32 row sums; a lane sums its row with a rotating column so that the
// 32 lanes hit 32 different banks.
constexpr int STAGE_ITEMS = 7;
constexpr int BWD_MIN_CTAS = 10;   // 92 registers; 12 and 14 CTAs/SM with a 3-item stage measured slower
constexpr int STAGE_ROUNDS = (STAGE_ITEMS * 9 + 31) / 32;
struct __align__(128) Stage { float v[STAGE_ITEMS * 9][32]; };

// Sum the staged rows over the lanes: lane L sums row r*32 + L with eight 16-byte loads whose chunk index is
// XOR-swizzled by L & 7, so that the eight lanes of a quarter warp (one LDS.128 wavefront) read eight
// different 16-byte bank groups.  The XOR is applied to the byte address (rows are 128-byte aligned).
__device__ __noinline__ void flush_stage(Stage& st, int nb, uint32_t gid, int lane, float* __restrict__ g2d) {
  __syncwarp();
  const int rows = nb * 9;
#pragma unroll
  for (int r = 0; r < STAGE_ROUNDS; ++r) {
    const int p = r * 32 + lane;
    const int pc = p < rows ? p : 0;
    const unsigned base = (unsigned)__cvta_generic_to_shared(st.v[pc]) + 16u * (unsigned)(lane & 7);
    // the four running sums as two packed pairs: FADD2 (sm_100a add.rn.f32x2) adds two independent IEEE floats per
    // instruction -- same results, half the issue slots (the kernel is issue bound)
    unsigned long long s01 = 0ull, s23 = 0ull;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      unsigned long long f01, f23;
      asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(f01), "=l"(f23) : "r"(base ^ (16u * q)));
      asm("add.rn.f32x2 %0, %0, %1;" : "+l"(s01) : "l"(f01));
      asm("add.rn.f32x2 %0, %0, %1;" : "+l"(s23) : "l"(f23));
    }
    const float s0 = __uint_as_float((unsigned)s01), s1 = __uint_as_float((unsigned)(s01 >> 32));
    const float s2 = __uint_as_float((unsigned)s23), s3 = __uint_as_float((unsigned)(s23 >> 32));
    const int item = pc / 9, val = pc - 9 * item;
    const uint32_t idx = __shfl_sync(FULL, gid, item);
    if (p < rows) atomicAdd(g2d + (size_t)SPLX_G2D_STRIDE * idx + val, (s0 + s1) + (s2 + s3));
  }
  __syncwarp();
}

__global__ void __launch_bounds__(BLOCK, BWD_MIN_CTAS)
k_raster_bwd(const float* __restrict__ blend, const uint32_t* __restrict__ vals, const uint32_t* __restrict__ ranges,
             int W, int H, int TX, int ntiles, splx_config cfg, const float* __restrict__ ct,
             const uint32_t* __restrict__ n_contrib, const float* __restrict__ g_ct, float* __restrict__ g2d,
             const uint32_t* __restrict__ order, uint32_t nslots) {
  __shared__ Ring rings[WARPS];
  __shared__ Stage stages[WARPS];
  int tile = blockIdx.x, k = blockIdx.y;
  if (order) {                             // CTAs handed out longest list first (splx_binning.slot_order)
    if (blockIdx.x >= order[nslots]) return;
    const uint32_t s = order[blockIdx.x];
    k = (int)(s / (uint32_t)ntiles); tile = (int)(s - (uint32_t)k * (uint32_t)ntiles);
  }
  const uint32_t r0 = ranges[2 * ((size_t)k * ntiles + tile)], r1 = ranges[2 * ((size_t)k * ntiles + tile) + 1];
  if (r0 == r1) return;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  Ring& ring = rings[warp];
  const int X0 = (tile % TX) * SPLX_TILE, Y0 = (tile / TX) * SPLX_TILE + 8 * warp;
  const int pxi = X0 + (lane & 7), pyi = Y0 + (lane >> 3);
  const float px0 = (float)pxi + 0.5f, px1 = px0 + 8.0f, py0 = (float)pyi + 0.5f, py1 = py0 + 4.0f;
  const float log2_amin = cfg.alpha_min > 0.f ? log2f(cfg.alpha_min) : -INFINITY;

  // Per pixel: T = transmittance in front of the entry being visited (starts from the final one);
  // Q = <dL/dC, colour composited from everything behind> + dL/dT * (transmittance behind), so that
  // dL/dalpha_i = T_i (<dL/dC, c_i> - Q_{i+1}) and Q_i = Q_{i+1} + alpha_i (<dL/dC, c_i> - Q_{i+1}); the walk
  // starts behind the last contributor, where the colour behind is 0 and the transmittance behind is 1.
  uint32_t last[4];
  float T[4], Q[4], gC0[4], gC1[4], gC2[4];
  uint32_t lmax = 0;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    const int x = pxi + 8 * (s & 1), y = pyi + 4 * (s >> 1);
    last[s] = 0; T[s] = 1.f; Q[s] = 0.f; gC0[s] = gC1[s] = gC2[s] = 0.f;
    if (x < W && y < H) {
      const size_t pix = ((size_t)k * H + y) * W + x;
      last[s] = n_contrib[pix];
      T[s] = ct[4 * pix + 3];
      const float4 g = *reinterpret_cast<const float4*>(g_ct + 4 * pix);
      gC0[s] = g.x; gC1[s] = g.y; gC2[s] = g.z; Q[s] = g.w;
    }
    lmax = max(lmax, last[s]);
  }
  const uint32_t bmax = __reduce_max_sync(FULL, lmax);
  if (bmax == 0) return;
  // per-slot maximum of `last` over the warp: a slot is skipped for list positions beyond it
  uint32_t smax[4];
#pragma unroll
  for (int s = 0; s < 4; ++s) smax[s] = __reduce_max_sync(FULL, last[s]);

  Stage& stage = stages[warp];
  int nb = 0;                 // items staged so far (warp-uniform)
  uint32_t gid = 0;           // lane b keeps the Gaussian index of staged item b
  const int nbatch = (int)((bmax + 31) / 32);
  int buf = 0;
  stage_issue(ring, 0, lane, blend, vals, r0 + 32u * (uint32_t)(nbatch - 1) + lane, r0 + bmax);
  for (int bi = nbatch - 1; bi >= 0; --bi, buf ^= 1) {
    const uint32_t start = 32u * (uint32_t)bi;      // list position (0-based) of entry 0 of this batch
    if (bi > 0) stage_issue(ring, buf ^ 1, lane, blend, vals, r0 + start - 32 + lane, r0 + bmax);
    else cp_async_commit();
    cp_async_wait<1>();
    __syncwarp();
    unsigned m = 0;
    if (start + lane < bmax) m = cull_mask(ring.q[buf][0][lane], ring.q[buf][1][lane], (float)X0, (float)Y0, log2_amin);
    unsigned reach = 0;                              // slots in which some pixel's walk reaches this batch
#pragma unroll
    for (int s = 0; s < 4; ++s) if (smax[s] > start) reach |= 1u << s;
    m &= reach;
    unsigned live = __ballot_sync(FULL, m != 0);
    while (live) {
      const int j = 31 - __clz(live);
      live &= ~(1u << j);
      const uint32_t c1 = start + (uint32_t)j + 1;    // 1-based list position
      const unsigned mj = __shfl_sync(FULL, m, j);
      const float4 a = ring.q[buf][0][j], b = ring.q[buf][1][j], c = ring.q[buf][2][j];
      const float dxs[2] = {__fsub_rn(a.x, px0), __fsub_rn(a.x, px1)};
      const float dys[2] = {__fsub_rn(a.y, py0), __fsub_rn(a.y, py1)};
      const float adx[2] = {__fmul_rn(b.x, dxs[0]), __fmul_rn(b.x, dxs[1])};
      const float bdx[2] = {__fmul_rn(b.y, dxs[0]), __fmul_rn(b.y, dxs[1])};
      const float cdy[2] = {__fmul_rn(b.z, dys[0]), __fmul_rn(b.z, dys[1])};
      // moments of dL/dG over this lane's pixels, and the colour sums.  Branch-free per slot: a pixel
      // that does not blend this entry runs the same arithmetic with alpha = 0 (T, Q unchanged, every
      // contribution exactly 0), so the four slots interleave in the pipeline.
      float n0 = 0.f, nx = 0.f, ny = 0.f, nxx = 0.f, nxy = 0.f, nyy = 0.f, q0 = 0.f, q1 = 0.f, q2 = 0.f;
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        if (!((mj >> s) & 1)) continue;     // warp-uniform
        const float dx = dxs[s & 1], dy = dys[s >> 1];
        float G, alpha; bool clamped;
        const bool on = eval_alpha(dx, dy, adx[s & 1], bdx[s & 1], cdy[s >> 1], a.z, cfg.alpha_min, cfg.alpha_max, G, alpha, clamped) &&
                        (c1 <= last[s]);
        const float al = on ? alpha : 0.0f;
        const float rom = rcp_approx(1.0f - al);             // 1 - alpha >= 1 - alpha_max > 0
        const float Ti = on ? T[s] * rom : T[s];             // T_i = T_{i+1} / (1 - alpha_i)
        T[s] = Ti;
        const float w = al * Ti;
        q0 = fmaf(w, gC0[s], q0); q1 = fmaf(w, gC1[s], q1); q2 = fmaf(w, gC2[s], q2);     // dL/dc_i
        const float diff = fmaf(gC0[s], c.x, fmaf(gC1[s], c.y, gC2[s] * c.z)) - Q[s];
        Q[s] = fmaf(al, diff, Q[s]);
        // o * dL/dG-weight of this pixel: T_i diff G o = w diff where alpha is not clamped (w = alpha_i T_i is 0
        // for a pixel that does not blend the entry); the factor 1/o is applied once per item below
        const float gG = clamped ? 0.0f : w * diff;
        const float t1 = gG * dx, t2 = gG * dy;
        n0 += gG; nx += t1; ny += t2;
        nxx = fmaf(t1, dx, nxx); nxy = fmaf(t1, dy, nxy); nyy = fmaf(t2, dy, nyy);
      }
      // linear map from the moments to the gradients of (u, v, A, B, C, o); alpha = o 2^(A' dx^2 + B' dx dy + C' dy^2).
      // The lane's nine partial sums go to row (item, value) of the staging block; rows are summed over the
      // lanes seven items at a time (flush_stage): 9 conflict-free stores per item here instead of a shuffle tree.
      float* row = stage.v[nb * 9];
      row[lane] = LN2 * fmaf(2.0f * b.x, nx, b.y * ny);         // dL/du   (moments carry the factor o)
      row[32 + lane] = LN2 * fmaf(2.0f * b.z, ny, b.y * nx);    // dL/dv
      row[64 + lane] = -0.5f * nxx;                             // dL/dA
      row[96 + lane] = -nxy;                                    // dL/dB
      row[128 + lane] = -0.5f * nyy;                            // dL/dC
      row[160 + lane] = n0 * rcp_approx(fmaxf(a.z, 1e-30f));    // dL/do (o == 0 blends nothing: 0, not NaN)
      row[192 + lane] = q0; row[224 + lane] = q1; row[256 + lane] = q2;
      if (lane == nb) gid = __float_as_uint(b.w);
      if (++nb == STAGE_ITEMS) { flush_stage(stage, nb, gid, lane, g2d); nb = 0; }
    }
    __syncwarp();
  }
  if (nb) flush_stage(stage, nb, gid, lane, g2d);
  cp_async_wait<0>();
}

}  // namespace

int launch_render_fwd(splx_ctx* ctx, const splx_projected* pr, const splx_binning* bins, const PlanDev& plan,
                      const splx_partial* out, uint64_t* pairs) {
  const int sparse = (plan.flags & SPLX_PLAN_SPARSE) ? 1 : 0;
  const uint32_t nslots = (uint32_t)plan.ntiles * (uint32_t)plan.K;
  // longest list first only where empty slots need no visit (without SPLX_PLAN_SPARSE they get the identity partial)
  const uint32_t* order = sparse && slot_order_pays(plan) ? bins->slot_order : nullptr;
  const dim3 grid = order ? dim3(nslots, 1) : dim3(plan.ntiles, plan.K);
  if (pairs)
    k_render_fwd<true><<<grid, BLOCK, 0, ctx->stream>>>(pr->blend, bins->vals, bins->tile_ranges, plan.W, plan.H, plan.TX,
                                                        plan.ntiles, ctx->cfg, plan.pv, sparse, out->ct, out->d,
                                                        out->n_contrib, (unsigned long long*)pairs, order, nslots);
  else
    k_render_fwd<false><<<grid, BLOCK, 0, ctx->stream>>>(pr->blend, bins->vals, bins->tile_ranges, plan.W, plan.H, plan.TX,
                                                         plan.ntiles, ctx->cfg, plan.pv, sparse, out->ct, out->d,
                                                         out->n_contrib, nullptr, order, nslots);
  SPLX_LAUNCH_CHECK(ctx, "k_render_fwd");
  return SPLX_OK;
}

int launch_raster_bwd(splx_ctx* ctx, const splx_projected* pr, const splx_binning* bins, const PlanDev& plan,
                      const splx_partial* part, const float* g_ct, float* g2d) {
  const uint32_t nslots = (uint32_t)plan.ntiles * (uint32_t)plan.K;
  const uint32_t* order = slot_order_pays(plan) ? bins->slot_order : nullptr;
  // slots of non-participating partitions have empty ranges: they exit at once / are not in the order
  const dim3 grid = order ? dim3(nslots, 1) : dim3(plan.ntiles, plan.K);
  k_raster_bwd<<<grid, BLOCK, 0, ctx->stream>>>(pr->blend, bins->vals, bins->tile_ranges, plan.W, plan.H, plan.TX,
                                                plan.ntiles, ctx->cfg, part->ct, part->n_contrib, g_ct, g2d, order, nslots);
  SPLX_LAUNCH_CHECK(ctx, "k_raster_bwd");
  return SPLX_OK;
}
