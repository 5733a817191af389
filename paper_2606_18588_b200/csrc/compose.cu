// compose.cu -- step a6 (global composition), a8 (its backward) and a7 (L1 loss gradient).
// "we first sort the colors according to their partial depth D_p^m, and then
// traverse the GPUs from front to back ... to accumulate the local rendering color with partial
// transmittance":  C_p = sum_m C_p^m prod_{k<m} T_p^k  (Eq.5).  Backward, Eq.6-7 (L186-L188):
// dL/dC^m = (prod_{k<m} T^k) dL/dC,  dL/dT^m = (prod_{k<m} T^k) <dL/dC, Behind_m>.
// Readings: s3 ordering key D/(1-T); s4 ties by partition index, an empty partial
// (T == 1) is the identity and sorts last; s7 background blended behind everything.
//
// HBM-bound streaming kernels: one thread per pixel, float4 (C,T) + float D per partition.
// Only the live partials (T < 1) of a pixel are ordered: an empty one contributes nothing
// wherever it stands, so the insertion sort runs over ~1-2 entries instead of K.
#include "common.cuh"

namespace {

constexpr int CB = 256;

struct PartialPtrs { const float* ct; const float* d; };

// Collect the live partials of one pixel, sorted by (key, k).  Returns the count.
template <int KMAX>
__device__ __forceinline__ int ordered_live(const float* __restrict__ ct, const float* __restrict__ d,
                                            int K, size_t HW, size_t pix, float (&key)[KMAX], int (&idx)[KMAX]) {
  int L = 0;
  for (int k = 0; k < K; ++k) {
    const float T = __ldg(ct + 4 * ((size_t)k * HW + pix) + 3);
    if (T < 1.0f) {
      const float kk = __fdiv_rn(__ldg(d + (size_t)k * HW + pix), __fsub_rn(1.0f, T));
      int p = L++;
      while (p > 0 && key[p - 1] > kk) { key[p] = key[p - 1]; idx[p] = idx[p - 1]; --p; }  // stable: '>' keeps smaller k first
      key[p] = kk; idx[p] = k;
    }
  }
  return L;
}

template <int KMAX>
__global__ void __launch_bounds__(CB)
k_compose_fwd(const float* __restrict__ ct, const float* __restrict__ d, int K, size_t HW, float bg0, float bg1,
              float bg2, float* __restrict__ image, float* __restrict__ T_total) {
  const size_t pix = (size_t)blockIdx.x * CB + threadIdx.x;
  if (pix >= HW) return;
  float key[KMAX]; int idx[KMAX];
  const int L = ordered_live<KMAX>(ct, d, K, HW, pix, key, idx);
  float Tacc = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  for (int m = 0; m < L; ++m) {
    const float4 p = __ldg(reinterpret_cast<const float4*>(ct) + (size_t)idx[m] * HW + pix);
    C0 = fmaf(Tacc, p.x, C0); C1 = fmaf(Tacc, p.y, C1); C2 = fmaf(Tacc, p.z, C2);
    Tacc *= p.w;
  }
  image[3 * pix] = fmaf(Tacc, bg0, C0);
  image[3 * pix + 1] = fmaf(Tacc, bg1, C1);
  image[3 * pix + 2] = fmaf(Tacc, bg2, C2);
  if (T_total) T_total[pix] = Tacc;
}

template <int KMAX>
__global__ void __launch_bounds__(CB)
k_compose_bwd(const float* __restrict__ ct, const float* __restrict__ d, int K, size_t HW, float bg0, float bg1,
              float bg2, const float* __restrict__ g_image, const float* __restrict__ g_T_total,
              float* __restrict__ g_ct) {
  const size_t pix = (size_t)blockIdx.x * CB + threadIdx.x;
  if (pix >= HW) return;
  float key[KMAX]; int idx[KMAX];
  const int L = ordered_live<KMAX>(ct, d, K, HW, pix, key, idx);
  const float g0 = g_image[3 * pix], g1 = g_image[3 * pix + 1], g2 = g_image[3 * pix + 2];
  const float gT = g_T_total ? g_T_total[pix] : 0.f;
  // T_total = product over the live partials in order (the empty ones multiply by 1)
  float Ttot = 1.f;
  for (int m = 0; m < L; ++m) Ttot *= __ldg(ct + 4 * ((size_t)idx[m] * HW + pix) + 3);
  // Empty partials stand behind all live ones: Tfront = T_total, Behind = bg, BehindT = 1.
  const float4 ge = make_float4(Ttot * g0, Ttot * g1, Ttot * g2, Ttot * (g0 * bg0 + g1 * bg1 + g2 * bg2 + gT));
  for (int k = 0; k < K; ++k) {
    const float T = __ldg(ct + 4 * ((size_t)k * HW + pix) + 3);
    if (!(T < 1.0f)) reinterpret_cast<float4*>(g_ct)[(size_t)k * HW + pix] = ge;
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
int launch_compose_fwd(splx_ctx* ctx, int K, const splx_partial* p, const CamDev& cam, const float* bg,
                       float* image, float* T_total) {
  const size_t HW = (size_t)cam.W * cam.H;
  const unsigned grid = (unsigned)((HW + CB - 1) / CB);
  if (K <= 8)
    k_compose_fwd<8><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, K, HW, bg[0], bg[1], bg[2], image, T_total);
  else
    k_compose_fwd<SPLX_MAX_K><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, K, HW, bg[0], bg[1], bg[2], image, T_total);
  SPLX_LAUNCH_CHECK(ctx, "k_compose_fwd");
  return SPLX_OK;
}

int launch_compose_bwd(splx_ctx* ctx, int K, const splx_partial* p, const CamDev& cam, const float* bg,
                       const float* g_image, const float* g_T_total, float* g_ct) {
  const size_t HW = (size_t)cam.W * cam.H;
  const unsigned grid = (unsigned)((HW + CB - 1) / CB);
  if (K <= 8)
    k_compose_bwd<8><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, K, HW, bg[0], bg[1], bg[2], g_image, g_T_total, g_ct);
  else
    k_compose_bwd<SPLX_MAX_K><<<grid, CB, 0, ctx->stream>>>(p->ct, p->d, K, HW, bg[0], bg[1], bg[2], g_image, g_T_total, g_ct);
  SPLX_LAUNCH_CHECK(ctx, "k_compose_bwd");
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
