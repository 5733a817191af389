// adam.cu -- step a11, the optimiser update.  PAPER.md L184 / L190 only say that "the parameters
// can be optimized"; the optimiser is unnamed: dense bias-corrected Adam,
//   m = b1 m + (1-b1) g;  v = b2 v + (1-b2) g^2;  p -= lr (m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps).
// HBM-bound: 16 B read + 12 B written per parameter (+4 B when the gradient is zeroed in place).
// 128-bit loads/stores, grid = a multiple of the SM count, grid-stride.
#include "common.cuh"

namespace {

constexpr int AB = 256;

struct AdamK { float lr, b1, b2, omb1, omb2, eps, ibc1, ibc2; };

// sqrt.approx / div.approx (MUFU.SQRT, MUFU.RCP + one multiply: <= 1 and 2 ulp) instead of the IEEE sequences: with those the
// kernel issued ~200 instructions per 16-byte vector and sat within 10 % of the issue limit at the HBM roof (28.2 ms at
// 100 M Gaussians; 26.5 ms = 95 % of the measured copy bandwidth with the approximate pair).  The update is within 3 ulp of
// the IEEE one: far inside the 1e-5 parity bar against the fp64 oracle.  sqrt.approx(0) = 0 (an untouched row has v = 0);
// the divisor is >= eps > 0.
__device__ __forceinline__ float sqrt_approx(float x) {
  float y;
  asm("sqrt.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void adam1(float& p, float g, float& m, float& v, const AdamK& k) {
  const float lr = k.lr, eps = k.eps, ibc1 = k.ibc1, ibc2 = k.ibc2;
  m = fmaf(k.b1, m, k.omb1 * g);
  v = fmaf(k.b2, v, k.omb2 * g * g);
  p -= lr * __fdividef(m * ibc1, sqrt_approx(v * ibc2) + eps);
}

__global__ void __launch_bounds__(AB)
k_adam(float* __restrict__ param, float* __restrict__ grad, float* __restrict__ m, float* __restrict__ v,
       int64_t count, AdamK k, float gscale, int zero_grad) {
  const int64_t nvec = count >> 2;
  for (int64_t i = (int64_t)blockIdx.x * AB + threadIdx.x; i < nvec; i += (int64_t)gridDim.x * AB) {
    float4 p = reinterpret_cast<float4*>(param)[i];
    float4 g = reinterpret_cast<const float4*>(grad)[i];
    float4 mm = reinterpret_cast<float4*>(m)[i];
    float4 vv = reinterpret_cast<float4*>(v)[i];
    adam1(p.x, g.x * gscale, mm.x, vv.x, k);
    adam1(p.y, g.y * gscale, mm.y, vv.y, k);
    adam1(p.z, g.z * gscale, mm.z, vv.z, k);
    adam1(p.w, g.w * gscale, mm.w, vv.w, k);
    reinterpret_cast<float4*>(param)[i] = p;
    reinterpret_cast<float4*>(m)[i] = mm;
    reinterpret_cast<float4*>(v)[i] = vv;
    if (zero_grad) reinterpret_cast<float4*>(grad)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  if (blockIdx.x == 0 && threadIdx.x < (count & 3)) {
    const int64_t i = (nvec << 2) + threadIdx.x;
    float p = param[i], mm = m[i], vv = v[i];
    adam1(p, grad[i] * gscale, mm, vv, k);
    param[i] = p; m[i] = mm; v[i] = vv;
    if (zero_grad) grad[i] = 0.f;
  }
}

// All parameter groups of one flat buffer in ONE launch: the groups differ only in their learning
// rate; group boundaries are multiples of 4 floats, so a 128-bit vector never straddles two groups.
// FLAGS: the gradient of a row (Gaussian) whose byte in `touched` is clear is ZERO by definition and its memory is
// never read -- the rows of the gradient buffer that no view of the iteration reached need neither zeroing nor
// reading (at 100M Gaussians a view sees ~2 % of them).  Same arithmetic, statement by statement, as the plain kernel
// on a gradient buffer whose untouched rows hold zeros.
struct AdamGroups {
  long long end4[SPLX_ADAM_MAX_GROUPS]; float lr[SPLX_ADAM_MAX_GROUPS]; int n;
  uint32_t start4[SPLX_ADAM_MAX_GROUPS]; int width[SPLX_ADAM_MAX_GROUPS]; long long rows;     // FLAGS only
};

// Flags of the four elements of vector i of group j (0 = untouched), in 32-bit arithmetic (the launcher checks that vector
// indices fit): a row of 48 or 4 floats holds the whole vector (one flag), a vector of a width-1 group holds four rows
// (their four flag bytes are one aligned word), a width-3 group's vector touches two rows.
__device__ __forceinline__ uint4 adam_flags(const AdamGroups& gr, int j, int64_t i, const uint8_t* __restrict__ touched) {
  const uint32_t v0 = (uint32_t)i - gr.start4[j];        // vector index inside the group
  const int w = gr.width[j];
  const uint32_t nrow = (uint32_t)gr.rows;
  uint32_t f0, f1, f2, f3;
  if (w == 48 || w == 4) {
    const uint32_t r = w == 48 ? v0 / 12u : v0;
    f0 = f1 = f2 = f3 = r < nrow ? (uint32_t)__ldg(touched + r) : 0u;
  } else if (w == 1) {
    const uint32_t r = 4u * v0;
    uint32_t word = 0;
    if (r + 3 < nrow && ((uintptr_t)touched & 3) == 0) word = __ldg(reinterpret_cast<const uint32_t*>(touched + r));
    else { for (uint32_t c = 0; c < 4; ++c) if (r + c < nrow) word |= (uint32_t)touched[r + c] << (8 * c); }
    f0 = word & 0xffu; f1 = word & 0xff00u; f2 = word & 0xff0000u; f3 = word & 0xff000000u;
  } else {
    const uint32_t e0 = 4u * v0, uw = (uint32_t)w;         // (a width-3 group of 100 M rows: 3e8 elements, fits)
    const uint32_t ra = e0 / uw, r1 = (e0 + 1u) / uw, r2 = (e0 + 2u) / uw, rb = (e0 + 3u) / uw;
    const uint32_t fa = ra < nrow ? (uint32_t)__ldg(touched + ra) : 0u, fb = rb < nrow ? (uint32_t)__ldg(touched + rb) : 0u;
    f0 = fa; f3 = fb;
    f1 = r1 == ra ? fa : (r1 == rb ? fb : (r1 < nrow ? (uint32_t)__ldg(touched + r1) : 0u));
    f2 = r2 == ra ? fa : (r2 == rb ? fb : (r2 < nrow ? (uint32_t)__ldg(touched + r2) : 0u));
  }
  return make_uint4(f0, f1, f2, f3);
}

// U vectors per thread and trip (their loads are issued together); CS: ld.global.cs / st.global.cs (evict-first) on the
// four streams.  Measured on 30 M Gaussians (7.1 GB per buffer; a quarter of the million-row blocks 60 % flagged), median
// of 7 launches, bytes as bench.py counts them: FLAGS 7.95 ms = 5.49 TB/s with plain accesses and one vector per thread
// -> 7.05 ms = 6.19 TB/s with two vectors and the streaming hints (the one-pass streams no longer evict the flag bytes
// and each other's open DRAM pages from L2; the same hints with ONE vector per thread: 6.97-7.87 ms depending on the grid;
// four vectors: 9.3-10.1 ms at 111 registers).  Without flags: 8.07 ms = 6.14 TB/s as it is, 7.9-8.4 ms with any
// variant: left alone.  So: FLAGS -> U = 2, CS; plain -> U = 1, no hints.
template <bool CS> __device__ __forceinline__ float4 ldv(const float4* p) { return CS ? __ldcs(p) : *p; }
template <bool CS> __device__ __forceinline__ void stv(float4* p, float4 v) { if (CS) __stcs(p, v); else *p = v; }
template <bool FLAGS, int U, bool CS>
__global__ void __launch_bounds__(AB, U == 1 ? 6 : 4)      // the bytes in flight, not the ALU, carry this kernel
k_adam_groups(float* __restrict__ param, float* __restrict__ grad, float* __restrict__ m, float* __restrict__ v, int64_t nvec,
              AdamK k, const __grid_constant__ AdamGroups gr, float gscale, int zero_grad, const uint8_t* __restrict__ touched) {
  const int64_t stride = (int64_t)gridDim.x * AB;
  for (int64_t i0 = (int64_t)blockIdx.x * AB + threadIdx.x; i0 < nvec; i0 += U * stride) {
    float4 p[U], g[U], mm[U], vv[U];
    int jj[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = i0 + u * stride;
      g[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      jj[u] = 0;
      if (i >= nvec) continue;
      int j = 0;
#pragma unroll
      for (int q = 1; q < SPLX_ADAM_MAX_GROUPS; ++q)
        if (q < gr.n && i >= gr.end4[q - 1]) j = q;
      jj[u] = j;
      if (FLAGS) {
        const uint4 fl = adam_flags(gr, j, i, touched);
        p[u] = ldv<CS>(reinterpret_cast<float4*>(param) + i);
        mm[u] = ldv<CS>(reinterpret_cast<float4*>(m) + i);
        vv[u] = ldv<CS>(reinterpret_cast<float4*>(v) + i);
        if (__any_sync(__activemask(), (fl.x | fl.y | fl.z | fl.w) != 0u)) {
          const float4 t = ldv<CS>(reinterpret_cast<const float4*>(grad) + i);
          g[u] = make_float4(fl.x ? t.x : 0.f, fl.y ? t.y : 0.f, fl.z ? t.z : 0.f, fl.w ? t.w : 0.f);
        }
      } else {
        g[u] = ldv<CS>(reinterpret_cast<const float4*>(grad) + i);
        p[u] = ldv<CS>(reinterpret_cast<float4*>(param) + i);
        mm[u] = ldv<CS>(reinterpret_cast<float4*>(m) + i);
        vv[u] = ldv<CS>(reinterpret_cast<float4*>(v) + i);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = i0 + u * stride;
      if (i >= nvec) continue;
      AdamK kk = k; kk.lr = gr.lr[jj[u]];
      adam1(p[u].x, g[u].x * gscale, mm[u].x, vv[u].x, kk);
      adam1(p[u].y, g[u].y * gscale, mm[u].y, vv[u].y, kk);
      adam1(p[u].z, g[u].z * gscale, mm[u].z, vv[u].z, kk);
      adam1(p[u].w, g[u].w * gscale, mm[u].w, vv[u].w, kk);
      stv<CS>(reinterpret_cast<float4*>(param) + i, p[u]);
      stv<CS>(reinterpret_cast<float4*>(m) + i, mm[u]);
      stv<CS>(reinterpret_cast<float4*>(v) + i, vv[u]);
      if (!FLAGS && zero_grad) reinterpret_cast<float4*>(grad)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
}

// Visible-only ("sparse") Adam, an OPTION outside the paper: only Gaussians whose flag is set
// -- they received a gradient in this iteration -- take the step, the others keep parameters AND moments untouched
// (no decay); the flags are cleared on the way.  A block owns 128 consecutive Gaussians: it reads their 128 flag
// bytes and walks the five parameter groups in coalesced 16-byte chunks, touching only flagged rows (a row's 48 SH
// floats are 192 contiguous bytes).  A block without a flagged row leaves after the flag load.
constexpr int SB = 128;
struct SparseSets { float *p[5], *g[5], *m[5], *v[5]; float lr[5]; };

__device__ __forceinline__ void adam4(float* pp, const float* pg, float* pm, float* pv, const AdamK& k, float lr, float gs) {
  float4 p = *reinterpret_cast<float4*>(pp), g = *reinterpret_cast<const float4*>(pg);
  float4 m = *reinterpret_cast<float4*>(pm), v = *reinterpret_cast<float4*>(pv);
  AdamK kk = k; kk.lr = lr;
  adam1(p.x, g.x * gs, m.x, v.x, kk); adam1(p.y, g.y * gs, m.y, v.y, kk);
  adam1(p.z, g.z * gs, m.z, v.z, kk); adam1(p.w, g.w * gs, m.w, v.w, kk);
  *reinterpret_cast<float4*>(pp) = p; *reinterpret_cast<float4*>(pm) = m; *reinterpret_cast<float4*>(pv) = v;
}
__device__ __forceinline__ void adam_s(float* pp, const float* pg, float* pm, float* pv, const AdamK& k, float lr, float gs) {
  float p = *pp, m = *pm, v = *pv;
  AdamK kk = k; kk.lr = lr;
  adam1(p, *pg * gs, m, v, kk);
  *pp = p; *pm = m; *pv = v;
}

__global__ void __launch_bounds__(SB)
k_adam_sparse(const __grid_constant__ SparseSets S, uint8_t* __restrict__ touched, int64_t n, AdamK k, float gs) {
  __shared__ uint8_t s_t[SB];
  const int64_t base = (int64_t)blockIdx.x * SB;
  const int64_t i = base + threadIdx.x;
  const uint8_t t = i < n ? touched[i] : (uint8_t)0;
  s_t[threadIdx.x] = t;
  if (!__syncthreads_or(t)) return;
  if (t) touched[i] = 0;
  const int nrows = (int)min((int64_t)SB, n - base);
  // sh: 12 float4 per row
#pragma unroll 4
  for (int c = 0; c < 12; ++c) {
    const int q = c * SB + threadIdx.x;
    const int row = q / 12, c4 = q - row * 12;
    if (row < nrows && s_t[row]) {
      const int64_t off = 48 * (base + row) + 4 * c4;
      adam4(S.p[4] + off, S.g[4] + off, S.m[4] + off, S.v[4] + off, k, S.lr[4], gs);
    }
  }
  if (t) {
    adam4(S.p[2] + 4 * i, S.g[2] + 4 * i, S.m[2] + 4 * i, S.v[2] + 4 * i, k, S.lr[2], gs);      // quat
    adam_s(S.p[3] + i, S.g[3] + i, S.m[3] + i, S.v[3] + i, k, S.lr[3], gs);                     // opacity logit
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      adam_s(S.p[0] + 3 * i + c, S.g[0] + 3 * i + c, S.m[0] + 3 * i + c, S.v[0] + 3 * i + c, k, S.lr[0], gs);   // mean
      adam_s(S.p[1] + 3 * i + c, S.g[1] + 3 * i + c, S.m[1] + 3 * i + c, S.v[1] + 3 * i + c, k, S.lr[1], gs);   // log scale
    }
  }
}

}  // namespace

int launch_adam_sparse(splx_ctx* ctx, const splx_gaussian_grads* P, const splx_gaussian_grads* Gr,
                       const splx_gaussian_grads* M, const splx_gaussian_grads* V, uint8_t* touched, const float* lr,
                       float beta1, float beta2, float eps, int step, float grad_scale) {
  const int64_t n = P->n;
  if (n <= 0) return SPLX_OK;
  const double bc1 = 1.0 - pow((double)beta1, step), bc2 = 1.0 - pow((double)beta2, step);
  const AdamK k{0.f, beta1, beta2, (float)(1.0 - (double)beta1), (float)(1.0 - (double)beta2), eps,
                (float)(1.0 / bc1), (float)(1.0 / bc2)};
  SparseSets S;
  const splx_gaussian_grads* sets[4] = {P, Gr, M, V};
  float** dst[4] = {S.p, S.g, S.m, S.v};
  for (int a = 0; a < 4; ++a) {
    dst[a][0] = sets[a]->mean; dst[a][1] = sets[a]->log_scale; dst[a][2] = sets[a]->quat;
    dst[a][3] = sets[a]->opacity_logit; dst[a][4] = sets[a]->sh;
  }
  for (int j = 0; j < 5; ++j) S.lr[j] = lr[j];
  k_adam_sparse<<<(unsigned)((n + SB - 1) / SB), SB, 0, ctx->stream>>>(S, touched, n, k, grad_scale);
  SPLX_LAUNCH_CHECK(ctx, "k_adam_sparse");
  return SPLX_OK;
}

int launch_adam_groups(splx_ctx* ctx, float* param, float* grad, float* m, float* v, int n_groups,
                       const int64_t* group_offsets, const float* lr, float beta1, float beta2, float eps, int step,
                       float grad_scale, int zero_grad, const int32_t* widths, int64_t rows, const uint8_t* touched) {
  const int64_t count = group_offsets[n_groups];
  if (count <= 0) return SPLX_OK;
  const double bc1 = 1.0 - pow((double)beta1, step), bc2 = 1.0 - pow((double)beta2, step);
  const int64_t nvec = count >> 2;
  int64_t blocks = (nvec + AB - 1) / AB;
  const int64_t cap = (int64_t)SPLX_SM_COUNT * 8;
  if (blocks > cap) blocks = cap;
  const AdamK k{0.f, beta1, beta2, (float)(1.0 - (double)beta1), (float)(1.0 - (double)beta2), eps,
                (float)(1.0 / bc1), (float)(1.0 / bc2)};
  AdamGroups gr;
  memset(&gr, 0, sizeof gr);
  gr.n = n_groups;
  gr.rows = rows;
  for (int j = 0; j < SPLX_ADAM_MAX_GROUPS; ++j) {
    gr.end4[j] = j < n_groups ? group_offsets[j + 1] >> 2 : nvec;
    gr.lr[j] = j < n_groups ? lr[j] : 0.f;
    gr.start4[j] = (uint32_t)((j < n_groups ? group_offsets[j] : count) >> 2);
    gr.width[j] = (touched && j < n_groups) ? widths[j] : 1;
  }
  if (touched && (nvec >> 32 || rows >> 30))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_adam_groups_flagged: more than 2^32 vectors or 2^30 rows");
  if (touched)
    k_adam_groups<true, 2, true><<<(unsigned)blocks, AB, 0, ctx->stream>>>(param, grad, m, v, nvec, k, gr, grad_scale, 0, touched);
  else
    k_adam_groups<false, 1, false><<<(unsigned)blocks, AB, 0, ctx->stream>>>(param, grad, m, v, nvec, k, gr, grad_scale, zero_grad, nullptr);
  SPLX_LAUNCH_CHECK(ctx, "k_adam_groups");
  return SPLX_OK;
}

int launch_adam(splx_ctx* ctx, float* param, float* grad, float* m, float* v, int64_t count, float lr,
                float beta1, float beta2, float eps, int step, float grad_scale, int zero_grad) {
  if (count <= 0) return SPLX_OK;
  const double bc1 = 1.0 - pow((double)beta1, step), bc2 = 1.0 - pow((double)beta2, step);
  const int64_t nvec = count >> 2;
  int64_t blocks = (nvec + AB - 1) / AB;
  const int64_t cap = (int64_t)SPLX_SM_COUNT * 8;   // 8 resident CTAs of 256 threads per SM
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  // 1-beta and the bias corrections are formed in double on the host (0.999f is not 0.999)
  const AdamK k{lr, beta1, beta2, (float)(1.0 - (double)beta1), (float)(1.0 - (double)beta2), eps,
                (float)(1.0 / bc1), (float)(1.0 / bc2)};
  k_adam<<<(unsigned)blocks, AB, 0, ctx->stream>>>(param, grad, m, v, count, k, grad_scale, zero_grad);
  SPLX_LAUNCH_CHECK(ctx, "k_adam");
  return SPLX_OK;
}
