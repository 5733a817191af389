// compose.cu -- step a6 (global composition), a8 (its backward) and a7 (L1 loss gradient).
// "we first sort the colors according to their partial depth D_p^m, and then
// traverse the GPUs from front to back ... to accumulate the local rendering color with partial
// transmittance":  C_p = sum_m C_p^m prod_{k<m} T_p^k  (Eq.5).  Backward, Eq.6-7 (L186-L188):
// dL/dC^m = (prod_{k<m} T^k) dL/dC,  dL/dT^m = (prod_{k<m} T^k) <dL/dC, Behind_m>.
// Readings: s3 ordering key D/(1-T); s4 ties by partition index, an empty partial
// (T == 1) is the identity and sorts last; s7 background blended behind everything.
//
// HBM-bound streaming kernels.  Grid = (tiles, B views), CTA = one 16 x 16 tile, one thread per pixel,
// float4 (C,T) + float D per partition.  A view composes only the partitions that render it
// (splx_plan.view_of_part); with SPLX_PLAN_SPARSE a (partition, tile) slot whose list is empty is
// the identity and is not even read -- the tile's participant flags are looked up once per CTA.
// Only the live partials (T < 1) of a pixel are ordered: an empty one contributes nothing wherever
// it stands, so the insertion sort runs over ~1-2 entries instead of K.
#include "common.cuh"

namespace {

constexpr int CB = SPLX_TILE * SPLX_TILE;

// s_list[0 .. *s_n) = the partitions composed into view b on this tile (they render view b and, with SPLX_PLAN_SPARSE, have a
// non-empty list here), in ascending order.  Built by the first warp: lane l looks at partitions l and l + 32.
__device__ __forceinline__ void tile_participants(const PartView& pv, int K, int b, int tile, int ntiles, int sparse,
                                                  const uint32_t* __restrict__ ranges, uint8_t* s_list, int* s_n) {
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    bool use[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int k = lane + 32 * h;
      use[h] = k < K && pv.v[k] == b;
      if (use[h] && sparse) {
        const uint2 r = *reinterpret_cast<const uint2*>(ranges + 2 * ((size_t)k * ntiles + tile));
        use[h] = r.x < r.y;
      }
    }
    const unsigned b0 = __ballot_sync(0xffffffffu, use[0]), b1 = __ballot_sync(0xffffffffu, use[1]);
    const unsigned lt = (1u << lane) - 1u;
    if (use[0]) s_list[__popc(b0 & lt)] = (uint8_t)lane;
    if (use[1]) s_list[__popc(b0) + __popc(b1 & lt)] = (uint8_t)(lane + 32);
    if (lane == 0) *s_n = __popc(b0) + __popc(b1);
  }
  __syncthreads();
}

// Collect the live partials of one pixel, sorted by (key, k).  Returns the count.  The candidates (the tile's
// participants: ~1-6 of up to 64 partitions) are fetched eight at a time, every T and D of a chunk first -- predicated,
// independent loads: one memory latency per chunk instead of a chain of dependent ones (the kernel was bound by that
// chain, profiles/r01e_ncu_full.md; round 1 had the up-front fetch for K <= 8 only, the city configurations run K = 16, 32).
template <int KMAX>
__device__ __forceinline__ int ordered_live(const float* __restrict__ ct, const float* __restrict__ d, const uint8_t* s_list,
                                            int n_use, size_t HW, size_t pix, float (&key)[KMAX], int (&idx)[KMAX]) {
  int L = 0;
  for (int c0 = 0; c0 < n_use; c0 += 8) {
    float Tk[8], dk[8];
    int kk[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const bool u = c0 + j < n_use;
      kk[j] = u ? (int)s_list[c0 + j] : 0;
      Tk[j] = u ? __ldg(ct + 4 * ((size_t)kk[j] * HW + pix) + 3) : 1.0f;
      dk[j] = u ? __ldg(d + (size_t)kk[j] * HW + pix) : 0.0f;
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (Tk[j] < 1.0f) {
        const float kv = __fdiv_rn(dk[j], __fsub_rn(1.0f, Tk[j]));
        int p = L++;
        while (p > 0 && key[p - 1] > kv) { key[p] = key[p - 1]; idx[p] = idx[p - 1]; --p; }    // stable: '>' keeps smaller k first
        key[p] = kv; idx[p] = kk[j];
      }
    }
  }
  return L;
}

template <int KMAX, bool SAT>
__global__ void __launch_bounds__(CB)
k_compose_fwd(const float* __restrict__ ct, const float* __restrict__ d, const uint32_t* __restrict__ ranges,
              const __grid_constant__ PartView pv, int K, int W, int H, int TX, int ntiles, int sparse, float bg0,
              float bg1, float bg2, const __grid_constant__ ViewBufs vb, float sat_eps,
              const uint8_t* __restrict__ state_in, uint8_t* __restrict__ state_out) {
  __shared__ uint8_t s_list[SPLX_MAX_K];
  __shared__ int s_n;
  __shared__ unsigned s_unsat[2];
  const int tile = blockIdx.x, b = blockIdx.y;
  if (SAT && threadIdx.x < 2) s_unsat[threadIdx.x] = 0u;
  tile_participants(pv, K, b, tile, ntiles, sparse, ranges, s_list, &s_n);
  const int x = (tile % TX) * SPLX_TILE + (threadIdx.x & 15), y = (tile / TX) * SPLX_TILE + (threadIdx.x >> 4);
  const size_t HW = (size_t)W * H;
  const bool inside = x < W && y < H;
  unsigned long long unsat = 0ull;
  if (inside) {
    const size_t pix = (size_t)y * W + x;
    float key[KMAX]; int idx[KMAX];
    const int L = ordered_live<KMAX>(ct, d, s_list, s_n, HW, pix, key, idx);
    float Tacc = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
    unsigned long long live = 0ull;
    for (int m = 0; m < L; ++m) {
      const float4 p = __ldg(reinterpret_cast<const float4*>(ct) + (size_t)idx[m] * HW + pix);
      if (SAT) { live |= 1ull << idx[m]; if (!(Tacc < sat_eps)) unsat |= 1ull << idx[m]; }
      C0 = fmaf(Tacc, p.x, C0); C1 = fmaf(Tacc, p.y, C1); C2 = fmaf(Tacc, p.z, C2);
      Tacc *= p.w;
    }
    float* im = vb.image[b] + 3 * pix;
    im[0] = fmaf(Tacc, bg0, C0);
    im[1] = fmaf(Tacc, bg1, C1);
    im[2] = fmaf(Tacc, bg2, C2);
    if (vb.T_total[b]) vb.T_total[b][pix] = Tacc;
    // a partition that is the identity at this pixel stands behind all live ones: its front product is T_total
    if (SAT && !(Tacc < sat_eps)) unsat |= ~live;
  }
  if (SAT) {
    const unsigned lo = __reduce_or_sync(0xffffffffu, (unsigned)unsat);
    const unsigned hi = __reduce_or_sync(0xffffffffu, (unsigned)(unsat >> 32));
    if ((threadIdx.x & 31) == 0) { if (lo) atomicOr(&s_unsat[0], lo); if (hi) atomicOr(&s_unsat[1], hi); }
    __syncthreads();
    for (int k = threadIdx.x; k < K; k += CB) {
      if (pv.v[k] != b) continue;
      const size_t slot = (size_t)k * ntiles + tile;
      const uint8_t in = state_in ? state_in[slot] : (uint8_t)0;
      const bool u = (s_unsat[k >> 5] >> (k & 31)) & 1u;
      state_out[slot] = (uint8_t)((in & SPLX_TILE_INVISIBLE) | (u ? 0 : SPLX_TILE_SATURATED));
    }
  }
}

template <int KMAX>
__global__ void __launch_bounds__(CB)
k_compose_bwd(const float* __restrict__ ct, const float* __restrict__ d, const uint32_t* __restrict__ ranges,
              const __grid_constant__ PartView pv, int K, int W, int H, int TX, int ntiles, int sparse, float bg0,
              float bg1, float bg2, const __grid_constant__ ViewBufs vb, float* __restrict__ g_ct) {
  __shared__ uint8_t s_list[SPLX_MAX_K];
  __shared__ int s_n;
  const int tile = blockIdx.x, b = blockIdx.y;
  tile_participants(pv, K, b, tile, ntiles, sparse, ranges, s_list, &s_n);
  const int x = (tile % TX) * SPLX_TILE + (threadIdx.x & 15), y = (tile / TX) * SPLX_TILE + (threadIdx.x >> 4);
  if (x >= W || y >= H) return;
  const size_t HW = (size_t)W * H, pix = (size_t)y * W + x;
  float key[KMAX]; int idx[KMAX];
  const int L = ordered_live<KMAX>(ct, d, s_list, s_n, HW, pix, key, idx);
  const float* gi = vb.g_image[b] + 3 * pix;
  const float g0 = gi[0], g1 = gi[1], g2 = gi[2];
  const float gT = vb.g_T_total[b] ? vb.g_T_total[b][pix] : 0.f;
  // T_total = product over the live partials in order (the empty ones multiply by 1)
  float Ttot = 1.f;
  for (int m = 0; m < L; ++m) Ttot *= __ldg(ct + 4 * ((size_t)idx[m] * HW + pix) + 3);
  // Empty partials stand behind all live ones: Tfront = T_total, Behind = bg, BehindT = 1.
  const float4 ge = make_float4(Ttot * g0, Ttot * g1, Ttot * g2, Ttot * (g0 * bg0 + g1 * bg1 + g2 * bg2 + gT));
  unsigned long long live = 0ull;
  for (int m = 0; m < L; ++m) live |= 1ull << idx[m];
  for (int j = 0; j < s_n; ++j) {
    const int k = s_list[j];
    if (!((live >> k) & 1ull)) reinterpret_cast<float4*>(g_ct)[(size_t)k * HW + pix] = ge;
  }
  // Live partials, back to front: Tfront_m = T_total / prod_{r>=m} T_r is avoided (no division):
  // recompute the prefix products front to back into key[] (the keys are no longer needed).
  float Tacc = 1.f;
  for (int m = 0; m < L; ++m) { key[m] = Tacc; Tacc *= __ldg(ct + 4 * ((size_t)idx[m] * HW + pix) + 3); }
  float B0 = bg0, B1 = bg1, B2 = bg2, BT = 1.f;
  for (int m = L - 1; m >= 0; --m) {
    const float4 p = __ldg(reinterpret_cast<const float4*>(ct) + (size_t)idx[m] * HW + pix);
    const float Tf = key[m];
    reinterpret_cast<float4*>(g_ct)[(size_t)idx[m] * HW + pix] =
        make_float4(Tf * g0, Tf * g1, Tf * g2, Tf * (g0 * B0 + g1 * B1 + g2 * B2 + gT * BT));
    B0 = fmaf(p.w, B0, p.x); B1 = fmaf(p.w, B1, p.y); B2 = fmaf(p.w, B2, p.z);
    BT *= p.w;
  }
}

// a6 + a7 + a8 in ONE pass over the partial pixels (splx_compose_l1_backward_plan): the forward composite, the
// mean-L1 loss gradient against the view's target and the composition backward all need the same ordered
// partials of the pixel, so the staged path's second read of the partials and the image / dL/dimage round
// trip through HBM disappear.  Arithmetic is the staged kernels', statement by statement.
template <int KMAX, bool SAT>
__global__ void __launch_bounds__(CB)
k_compose_fused(const float* __restrict__ ct, const float* __restrict__ d, const uint32_t* __restrict__ ranges,
                const __grid_constant__ PartView pv, int K, int W, int H, int TX, int ntiles, int sparse, float bg0,
                float bg1, float bg2, const __grid_constant__ ViewBufs vb, float gscale, double* loss_sum,
                float* __restrict__ g_ct, float sat_eps, const uint8_t* __restrict__ state_in,
                uint8_t* __restrict__ state_out) {
  __shared__ uint8_t s_list[SPLX_MAX_K];
  __shared__ int s_n;
  __shared__ unsigned s_unsat[2];
  __shared__ float s_loss[CB / 32];
  const int tile = blockIdx.x, b = blockIdx.y;
  if (SAT && threadIdx.x < 2) s_unsat[threadIdx.x] = 0u;
  tile_participants(pv, K, b, tile, ntiles, sparse, ranges, s_list, &s_n);
  const int x = (tile % TX) * SPLX_TILE + (threadIdx.x & 15), y = (tile / TX) * SPLX_TILE + (threadIdx.x >> 4);
  const size_t HW = (size_t)W * H;
  const bool inside = x < W && y < H;
  unsigned long long unsat = 0ull;
  float lacc = 0.f;
  if (inside) {
    const size_t pix = (size_t)y * W + x;
    float key[KMAX]; int idx[KMAX];
    const int L = ordered_live<KMAX>(ct, d, s_list, s_n, HW, pix, key, idx);
    float Tacc = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
    unsigned long long live = 0ull;
    for (int m = 0; m < L; ++m) {
      const float4 p = __ldg(reinterpret_cast<const float4*>(ct) + (size_t)idx[m] * HW + pix);
      live |= 1ull << idx[m];
      if (SAT && !(Tacc < sat_eps)) unsat |= 1ull << idx[m];
      key[m] = Tacc;                                   // T in front of the m-th partial (the keys are spent)
      C0 = fmaf(Tacc, p.x, C0); C1 = fmaf(Tacc, p.y, C1); C2 = fmaf(Tacc, p.z, C2);
      Tacc *= p.w;
    }
    const float Ttot = Tacc;
    const float i0 = fmaf(Ttot, bg0, C0), i1 = fmaf(Ttot, bg1, C1), i2 = fmaf(Ttot, bg2, C2);
    float* im = vb.image[b] + 3 * pix;
    im[0] = i0; im[1] = i1; im[2] = i2;
    if (vb.T_total[b]) vb.T_total[b][pix] = Ttot;
    if (SAT && !(Ttot < sat_eps)) unsat |= ~live;
    // a7: mean L1 against the target of view b
    const float* tg = vb.target[b] + 3 * pix;
    const float e0 = i0 - tg[0], e1 = i1 - tg[1], e2 = i2 - tg[2];
    lacc = fabsf(e0) + fabsf(e1) + fabsf(e2);
    const float g0 = e0 > 0.f ? gscale : (e0 < 0.f ? -gscale : 0.f);
    const float g1 = e1 > 0.f ? gscale : (e1 < 0.f ? -gscale : 0.f);
    const float g2 = e2 > 0.f ? gscale : (e2 < 0.f ? -gscale : 0.f);
    // a8: identity partials stand behind all live ones
    const float4 ge = make_float4(Ttot * g0, Ttot * g1, Ttot * g2, Ttot * (g0 * bg0 + g1 * bg1 + g2 * bg2));
    for (int j = 0; j < s_n; ++j) {
      const int k = s_list[j];
      if (!((live >> k) & 1ull)) reinterpret_cast<float4*>(g_ct)[(size_t)k * HW + pix] = ge;
    }
    float B0 = bg0, B1 = bg1, B2 = bg2;
    for (int m = L - 1; m >= 0; --m) {
      const float4 p = __ldg(reinterpret_cast<const float4*>(ct) + (size_t)idx[m] * HW + pix);
      const float Tf = key[m];
      reinterpret_cast<float4*>(g_ct)[(size_t)idx[m] * HW + pix] =
          make_float4(Tf * g0, Tf * g1, Tf * g2, Tf * (g0 * B0 + g1 * B1 + g2 * B2));
      B0 = fmaf(p.w, B0, p.x); B1 = fmaf(p.w, B1, p.y); B2 = fmaf(p.w, B2, p.z);
    }
  }
  if (loss_sum) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) lacc += __shfl_xor_sync(0xffffffffu, lacc, o);
    if ((threadIdx.x & 31) == 0) s_loss[threadIdx.x >> 5] = lacc;
  }
  if (SAT) {
    const unsigned lo = __reduce_or_sync(0xffffffffu, (unsigned)unsat);
    const unsigned hi = __reduce_or_sync(0xffffffffu, (unsigned)(unsat >> 32));
    if ((threadIdx.x & 31) == 0) { if (lo) atomicOr(&s_unsat[0], lo); if (hi) atomicOr(&s_unsat[1], hi); }
  }
  __syncthreads();
  if (loss_sum && threadIdx.x == 0) {
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < CB / 32; ++w) t += s_loss[w];
    atomicAdd(loss_sum, (double)t);
  }
  if (SAT) {
    for (int k = threadIdx.x; k < K; k += CB) {
      if (pv.v[k] != b) continue;
      const size_t slot = (size_t)k * ntiles + tile;
      const uint8_t in = state_in ? state_in[slot] : (uint8_t)0;
      const bool u = (s_unsat[k >> 5] >> (k & 31)) & 1u;
      state_out[slot] = (uint8_t)((in & SPLX_TILE_INVISIBLE) | (u ? 0 : SPLX_TILE_SATURATED));
    }
  }
}

// mean-L1 gradient; float4-vectorised body with a scalar tail
__global__ void __launch_bounds__(CB)
k_l1(const float* __restrict__ image, const float* __restrict__ target, int64_t count, float gscale,
     float* __restrict__ g_image, double* loss_sum) {
  const int64_t nvec = count >> 2;
  float acc = 0.f;
  for (int64_t i = (int64_t)blockIdx.x * CB + threadIdx.x; i < nvec; i += (int64_t)gridDim.x * CB) {
    const float4 a = __ldg(reinterpret_cast<const float4*>(image) + i);
    const float4 b = __ldg(reinterpret_cast<const float4*>(target) + i);
    const float dx = a.x - b.x, dy = a.y - b.y, dz = a.z - b.z, dw = a.w - b.w;
    acc += fabsf(dx) + fabsf(dy) + fabsf(dz) + fabsf(dw);
    float4 o;
    o.x = dx > 0.f ? gscale : (dx < 0.f ? -gscale : 0.f);
    o.y = dy > 0.f ? gscale : (dy < 0.f ? -gscale : 0.f);
    o.z = dz > 0.f ? gscale : (dz < 0.f ? -gscale : 0.f);
    o.w = dw > 0.f ? gscale : (dw < 0.f ? -gscale : 0.f);
    reinterpret_cast<float4*>(g_image)[i] = o;
  }
  if (blockIdx.x == 0 && threadIdx.x < (count & 3)) {
    const int64_t i = (nvec << 2) + threadIdx.x;
    const float dx = image[i] - target[i];
    acc += fabsf(dx);
    g_image[i] = dx > 0.f ? gscale : (dx < 0.f ? -gscale : 0.f);
  }
  if (loss_sum) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(loss_sum, (double)acc);
  }
}

}  // namespace

// The K partials are required to be one [K,H,W,*] allocation (splx_partial describes all K).
template <int KMAX>
static void compose_fwd_k(splx_ctx* ctx, const splx_partial* p, const uint32_t* ranges, const PlanDev& plan, int sparse,
                          const float* bg, const ViewBufs& vb, float sat_eps, uint8_t* state_out) {
  dim3 grid(plan.ntiles, plan.B);
  if (state_out)
    k_compose_fwd<KMAX, true><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, ranges, plan.pv, plan.K, plan.W, plan.H, plan.TX,
                                                           plan.ntiles, sparse, bg[0], bg[1], bg[2], vb, sat_eps,
                                                           plan.tile_state, state_out);
  else
    k_compose_fwd<KMAX, false><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, ranges, plan.pv, plan.K, plan.W, plan.H, plan.TX,
                                                            plan.ntiles, sparse, bg[0], bg[1], bg[2], vb, sat_eps, nullptr,
                                                            nullptr);
}

int launch_compose_fwd(splx_ctx* ctx, const splx_partial* p, const splx_binning* bins, const PlanDev& plan,
                       const float* bg, const ViewBufs& vb, float sat_eps, uint8_t* state_out) {
  const int sparse = (plan.flags & SPLX_PLAN_SPARSE) ? 1 : 0;
  const uint32_t* ranges = bins ? bins->tile_ranges : nullptr;
  if (plan.K <= 8) compose_fwd_k<8>(ctx, p, ranges, plan, sparse, bg, vb, sat_eps, state_out);
  else if (plan.K <= 16) compose_fwd_k<16>(ctx, p, ranges, plan, sparse, bg, vb, sat_eps, state_out);
  else if (plan.K <= 32) compose_fwd_k<32>(ctx, p, ranges, plan, sparse, bg, vb, sat_eps, state_out);
  else compose_fwd_k<SPLX_MAX_K>(ctx, p, ranges, plan, sparse, bg, vb, sat_eps, state_out);
  SPLX_LAUNCH_CHECK(ctx, "k_compose_fwd");
  return SPLX_OK;
}

template <int KMAX>
static void compose_bwd_k(splx_ctx* ctx, const splx_partial* p, const uint32_t* ranges, const PlanDev& plan, int sparse,
                          const float* bg, const ViewBufs& vb, float* g_ct) {
  dim3 grid(plan.ntiles, plan.B);
  k_compose_bwd<KMAX><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, ranges, plan.pv, plan.K, plan.W, plan.H, plan.TX,
                                                   plan.ntiles, sparse, bg[0], bg[1], bg[2], vb, g_ct);
}

int launch_compose_bwd(splx_ctx* ctx, const splx_partial* p, const splx_binning* bins, const PlanDev& plan,
                       const float* bg, const ViewBufs& vb, float* g_ct) {
  const int sparse = (plan.flags & SPLX_PLAN_SPARSE) ? 1 : 0;
  const uint32_t* ranges = bins ? bins->tile_ranges : nullptr;
  if (plan.K <= 8) compose_bwd_k<8>(ctx, p, ranges, plan, sparse, bg, vb, g_ct);
  else if (plan.K <= 16) compose_bwd_k<16>(ctx, p, ranges, plan, sparse, bg, vb, g_ct);
  else if (plan.K <= 32) compose_bwd_k<32>(ctx, p, ranges, plan, sparse, bg, vb, g_ct);
  else compose_bwd_k<SPLX_MAX_K>(ctx, p, ranges, plan, sparse, bg, vb, g_ct);
  SPLX_LAUNCH_CHECK(ctx, "k_compose_bwd");
  return SPLX_OK;
}

template <int KMAX>
static void compose_fused_k(splx_ctx* ctx, const splx_partial* p, const uint32_t* ranges, const PlanDev& plan, int sparse,
                            const float* bg, const ViewBufs& vb, float gscale, double* loss_sum, float* g_ct, float sat_eps,
                            uint8_t* state_out) {
  dim3 grid(plan.ntiles, plan.B);
  if (state_out)
    k_compose_fused<KMAX, true><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, ranges, plan.pv, plan.K, plan.W, plan.H, plan.TX,
                                                             plan.ntiles, sparse, bg[0], bg[1], bg[2], vb, gscale, loss_sum,
                                                             g_ct, sat_eps, plan.tile_state, state_out);
  else
    k_compose_fused<KMAX, false><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, ranges, plan.pv, plan.K, plan.W, plan.H, plan.TX,
                                                              plan.ntiles, sparse, bg[0], bg[1], bg[2], vb, gscale, loss_sum,
                                                              g_ct, sat_eps, nullptr, nullptr);
}

// gscale = scale / (values of ONE launch's images) as splx_l1_loss_grad forms it over B*H*W*3 values
int launch_compose_fused(splx_ctx* ctx, const splx_partial* p, const splx_binning* bins, const PlanDev& plan,
                         const float* bg, const ViewBufs& vb, float scale, double* loss_sum, float* g_ct, float sat_eps,
                         uint8_t* state_out) {
  const int sparse = (plan.flags & SPLX_PLAN_SPARSE) ? 1 : 0;
  const uint32_t* ranges = bins ? bins->tile_ranges : nullptr;
  const float gscale = scale / (float)((int64_t)plan.B * plan.W * plan.H * 3);
  if (plan.K <= 8) compose_fused_k<8>(ctx, p, ranges, plan, sparse, bg, vb, gscale, loss_sum, g_ct, sat_eps, state_out);
  else if (plan.K <= 16) compose_fused_k<16>(ctx, p, ranges, plan, sparse, bg, vb, gscale, loss_sum, g_ct, sat_eps, state_out);
  else if (plan.K <= 32) compose_fused_k<32>(ctx, p, ranges, plan, sparse, bg, vb, gscale, loss_sum, g_ct, sat_eps, state_out);
  else compose_fused_k<SPLX_MAX_K>(ctx, p, ranges, plan, sparse, bg, vb, gscale, loss_sum, g_ct, sat_eps, state_out);
  SPLX_LAUNCH_CHECK(ctx, "k_compose_fused");
  return SPLX_OK;
}

int launch_l1(splx_ctx* ctx, const float* image, const float* target, int64_t count, float scale,
              float* g_image, double* loss_sum) {
  if (count <= 0) return SPLX_OK;
  const int64_t nvec = count >> 2;
  int64_t blocks = (nvec + CB - 1) / CB;
  const int64_t cap = (int64_t)SPLX_SM_COUNT * 8;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  k_l1<<<(unsigned)blocks, CB, 0, ctx->stream>>>(image, target, count, scale / (float)count, g_image, loss_sum);
  SPLX_LAUNCH_CHECK(ctx, "k_l1");
  return SPLX_OK;
}
