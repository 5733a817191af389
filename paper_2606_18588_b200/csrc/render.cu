// render.cu -- step a5 (local per-partition render) and step a9 (its backward).
// PAPER.md Eq.1 (L84): alpha_i = o_i exp(-1/2 (x-mu)^T Sigma2D^-1 (x-mu));  Eq.3 (L167):
// C^m = sum c_i alpha_i prod_{j<i}(1-alpha_j);  Eq.4 (L172): T^m = prod (1-alpha_i) and the partial
// depth D^m (read as sum d_i alpha_i T_i).  Blending rules (s2): skip power > 0,
// alpha = min(alpha_max, .), skip alpha < alpha_min, stop BEFORE a Gaussian that would take T
// below T_eps.  Backward: PAPER.md L184 ("the per-Gaussian gradient backpropagates through the
// intermediate partial pixel"), with dL/dC^m and dL/dT^m coming from Eq.6-7 (compose.cu).
//
// Grid = (tiles, K): one CTA per (partition, tile), 256 threads = 16x16 pixels, the tile's sorted
// list staged 256 Gaussians at a time in shared memory.  A warp owns an 8x4 pixel block (not a
// 32x1 row) so that small footprints leave whole warps idle in the backward, where a warp that
// has no contributor for a Gaussian skips its reduction.  Neither kernel is HBM-bound: the
// forward is FP32/MUFU issue bound, the backward FP32 + shuffle + atomics.
#include "common.cuh"

namespace {

constexpr int BLOCK = 256;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

struct Splat {          // one staged list entry; conic pre-scaled so that alpha = o * 2^p2
  float2 xy;
  float4 con;           // (-0.5 log2e A, -log2e B, -0.5 log2e C, o)
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// The same instruction sequence in the forward and the backward, so that both take identical
// skip / clamp decisions for every (pixel, Gaussian) pair.
__device__ __forceinline__ bool eval_alpha(float px, float py, const float2 xy, const float4 con,
                                           float amin, float amax, float& dx, float& dy, float& G,
                                           float& alpha, bool& clamped) {
  dx = __fsub_rn(xy.x, px);
  dy = __fsub_rn(xy.y, py);
  const float p2 = fmaf(__fmul_rn(con.x, dx), dx, fmaf(__fmul_rn(con.z, dy), dy, __fmul_rn(__fmul_rn(con.y, dx), dy)));
  G = ex2_approx(p2);
  const float a = __fmul_rn(con.w, G);
  clamped = a >= amax;
  alpha = fminf(amax, a);
  return (p2 <= 0.0f) && (alpha >= amin);
}

__device__ __forceinline__ void pixel_of_thread(int tile, int TX, int& px, int& py) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tx = tile % TX, ty = tile / TX;
  px = tx * SPLX_TILE + (warp & 1) * 8 + (lane & 7);
  py = ty * SPLX_TILE + (warp >> 1) * 4 + (lane >> 3);
}

__device__ __forceinline__ Splat stage(const float* means2d, const float* conic_opacity, uint32_t g) {
  Splat s;
  s.xy = *reinterpret_cast<const float2*>(means2d + 2 * (size_t)g);
  const float4 co = *reinterpret_cast<const float4*>(conic_opacity + 4 * (size_t)g);
  s.con = make_float4(co.x * (-0.5f * LOG2E), co.y * (-LOG2E), co.z * (-0.5f * LOG2E), co.w);
  return s;
}

__global__ void __launch_bounds__(BLOCK)
k_render_fwd(const float* __restrict__ means2d, const float* __restrict__ conic_opacity,
             const float* __restrict__ rgb, const float* __restrict__ depth,
             const uint32_t* __restrict__ vals, const uint32_t* __restrict__ ranges, int W, int H, int TX,
             int ntiles, splx_config cfg, float* __restrict__ out_ct, float* __restrict__ out_d,
             uint32_t* __restrict__ out_n, unsigned long long* pairs) {
  __shared__ Splat s_sp[BLOCK];
  __shared__ float4 s_cd[BLOCK];   // rgb, depth
  const int tile = blockIdx.x, k = blockIdx.y;
  int pxi, pyi;
  pixel_of_thread(tile, TX, pxi, pyi);
  const bool inside = pxi < W && pyi < H;
  const float px = (float)pxi + 0.5f, py = (float)pyi + 0.5f;
  const uint32_t r0 = ranges[2 * ((size_t)k * ntiles + tile)], r1 = ranges[2 * ((size_t)k * ntiles + tile) + 1];
  float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f;
  uint32_t walked = 0, last = 0, blended = 0;
  bool done = !inside;
  for (uint32_t start = r0; start < r1; start += BLOCK) {
    if (__syncthreads_count(done) == BLOCK) break;
    const uint32_t idx = start + threadIdx.x;
    if (idx < r1) {
      const uint32_t g = vals[idx];
      s_sp[threadIdx.x] = stage(means2d, conic_opacity, g);
      s_cd[threadIdx.x] = make_float4(rgb[3 * (size_t)g], rgb[3 * (size_t)g + 1], rgb[3 * (size_t)g + 2], depth[g]);
    }
    __syncthreads();
    const int nb = min((uint32_t)BLOCK, r1 - start);
    for (int j = 0; !done && j < nb; ++j) {
      ++walked;
      float dx, dy, G, alpha; bool clamped;
      if (!eval_alpha(px, py, s_sp[j].xy, s_sp[j].con, cfg.alpha_min, cfg.alpha_max, dx, dy, G, alpha, clamped)) continue;
      const float Tn = T * (1.0f - alpha);
      if (Tn < cfg.T_eps) { done = true; continue; }
      const float w = alpha * T;
      const float4 cd = s_cd[j];
      C0 = fmaf(w, cd.x, C0); C1 = fmaf(w, cd.y, C1); C2 = fmaf(w, cd.z, C2); D = fmaf(w, cd.w, D);
      T = Tn;
      last = walked;
      ++blended;
    }
  }
  if (inside) {
    const size_t pix = ((size_t)k * H + pyi) * W + pxi;
    *reinterpret_cast<float4*>(out_ct + 4 * pix) = make_float4(C0, C1, C2, T);
    out_d[pix] = D;
    out_n[pix] = last;
  }
  if (pairs) {
    const uint32_t wsum = __reduce_add_sync(0xffffffffu, inside ? walked : 0u);
    const uint32_t bsum = __reduce_add_sync(0xffffffffu, blended);
    if ((threadIdx.x & 31) == 0 && wsum) {
      atomicAdd(pairs, (unsigned long long)wsum);
      atomicAdd(pairs + 1, (unsigned long long)bsum);
    }
  }
}

// Reduce 9 per-lane values over the warp with 14 shuffles instead of 45: at each butterfly step a
// lane keeps one half of its values and hands the other half to its partner.  Afterwards lane
// 4*j (j = 0..7) holds the warp total of v[j] and every lane holds the total of v8.
__device__ __forceinline__ float warp_reduce9(float (&v)[8], float& v8, int lane) {
  const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
  float a[4], b[2], c;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float send = h16 ? v[i] : v[i + 4], keep = h16 ? v[i + 4] : v[i];
    a[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
  }
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    const float send = h8 ? a[i] : a[i + 2], keep = h8 ? a[i + 2] : a[i];
    b[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  {
    const float send = h4 ? b[0] : b[1], keep = h4 ? b[1] : b[0];
    c = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  c += __shfl_xor_sync(0xffffffffu, c, 2);
  c += __shfl_xor_sync(0xffffffffu, c, 1);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v8 += __shfl_xor_sync(0xffffffffu, v8, o);
  return c;   // lane L: total of v[((L>>4)&1)*4 + ((L>>3)&1)*2 + ((L>>2)&1)]
}

__global__ void __launch_bounds__(BLOCK)
k_raster_bwd(const float* __restrict__ means2d, const float* __restrict__ conic_opacity,
             const float* __restrict__ rgb, const uint32_t* __restrict__ vals,
             const uint32_t* __restrict__ ranges, int W, int H, int TX, int ntiles, splx_config cfg,
             const float* __restrict__ ct, const uint32_t* __restrict__ n_contrib,
             const float* __restrict__ g_ct, float* __restrict__ g2d) {
  __shared__ Splat s_sp[BLOCK];
  __shared__ float4 s_ci[BLOCK];   // rgb, Gaussian index (as bits)
  __shared__ uint32_t s_max[BLOCK / 32];
  const int tile = blockIdx.x, k = blockIdx.y;
  const uint32_t r0 = ranges[2 * ((size_t)k * ntiles + tile)], r1 = ranges[2 * ((size_t)k * ntiles + tile) + 1];
  if (r0 == r1) return;
  int pxi, pyi;
  pixel_of_thread(tile, TX, pxi, pyi);
  const bool inside = pxi < W && pyi < H;
  const float px = (float)pxi + 0.5f, py = (float)pyi + 0.5f;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t last = 0;
  float T = 1.f, Tfin = 1.f, gC0 = 0.f, gC1 = 0.f, gC2 = 0.f, gT = 0.f;
  if (inside) {
    const size_t pix = ((size_t)k * H + pyi) * W + pxi;
    last = n_contrib[pix];
    Tfin = ct[4 * pix + 3];
    const float4 g = *reinterpret_cast<const float4*>(g_ct + 4 * pix);
    gC0 = g.x; gC1 = g.y; gC2 = g.z; gT = g.w;
  }
  T = Tfin;
  const uint32_t wmax = __reduce_max_sync(0xffffffffu, last);
  if (lane == 0) s_max[warp] = wmax;
  __syncthreads();
  uint32_t bmax = 0;
#pragma unroll
  for (int w = 0; w < BLOCK / 32; ++w) bmax = max(bmax, s_max[w]);
  if (bmax == 0) return;
  float S0 = 0.f, S1 = 0.f, S2 = 0.f;   // colour behind the current Gaussian (relative to its T)
  const float gTfin = gT * Tfin;
  for (int b = (int)((bmax - 1) / BLOCK); b >= 0; --b) {
    __syncthreads();
    const uint32_t pos = (uint32_t)b * BLOCK + threadIdx.x;
    if (pos < bmax) {
      const uint32_t g = vals[r0 + pos];
      s_sp[threadIdx.x] = stage(means2d, conic_opacity, g);
      s_ci[threadIdx.x] = make_float4(rgb[3 * (size_t)g], rgb[3 * (size_t)g + 1], rgb[3 * (size_t)g + 2], __uint_as_float(g));
    }
    __syncthreads();
    const int jtop = (int)min((uint32_t)BLOCK, bmax - (uint32_t)b * BLOCK) - 1;
    for (int j = jtop; j >= 0; --j) {
      const uint32_t c = (uint32_t)b * BLOCK + j + 1;   // 1-based list position, as in n_contrib
      float dx, dy, G, alpha; bool clamped;
      const Splat sp = s_sp[j];
      bool on = (c <= last) && eval_alpha(px, py, sp.xy, sp.con, cfg.alpha_min, cfg.alpha_max, dx, dy, G, alpha, clamped);
      if (!__any_sync(0xffffffffu, on)) continue;
      float v[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f}, v8 = 0.f;
      const float4 ci = s_ci[j];
      if (on) {
        const float om = 1.0f - alpha;
        const float rom = __fdividef(1.0f, om);
        T *= rom;                              // T_i = T_{i+1} / (1 - alpha_i)
        const float w = alpha * T;
        v[6] = w * gC0; v[7] = w * gC1; v8 = w * gC2;                       // dL/dc_i
        float dLda = T * (gC0 * (ci.x - S0) + gC1 * (ci.y - S1) + gC2 * (ci.z - S2)) - gTfin * rom;
        S0 = fmaf(alpha, ci.x - S0, S0); S1 = fmaf(alpha, ci.y - S1, S1); S2 = fmaf(alpha, ci.z - S2, S2);
        if (!clamped) {
          const float gG = dLda * G;           // dL/do
          const float gp = sp.con.w * gG;      // dL/dpower
          const float gl = gp * LN2;
          v[0] = gl * fmaf(2.0f * sp.con.x, dx, sp.con.y * dy);   // dL/du
          v[1] = gl * fmaf(2.0f * sp.con.z, dy, sp.con.y * dx);   // dL/dv
          v[2] = -0.5f * dx * dx * gp;                             // dL/dA
          v[3] = -dx * dy * gp;                                    // dL/dB
          v[4] = -0.5f * dy * dy * gp;                             // dL/dC
          v[5] = gG;
        }
      }
      const float tot = warp_reduce9(v, v8, lane);
      const uint32_t g = __float_as_uint(ci.w);
      float* dst = g2d + (size_t)SPLX_G2D_STRIDE * g;
      if ((lane & 3) == 0) {
        const int idx = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
        atomicAdd(dst + idx, tot);
      } else if (lane == 1) {
        atomicAdd(dst + 8, v8);
      }
    }
  }
}

}  // namespace

int launch_render_fwd(splx_ctx* ctx, const splx_projected* pr, const splx_binning* bins, int K,
                      const CamDev& cam, const splx_partial* out, uint64_t* pairs) {
  const int ntiles = cam.TX * cam.TY;
  dim3 grid(ntiles, K);
  k_render_fwd<<<grid, BLOCK, 0, ctx->stream>>>(pr->means2d, pr->conic_opacity, pr->rgb, pr->depth, bins->vals,
                                                bins->tile_ranges, cam.W, cam.H, cam.TX, ntiles, ctx->cfg,
                                                out->ct, out->d, out->n_contrib, (unsigned long long*)pairs);
  SPLX_LAUNCH_CHECK(ctx, "k_render_fwd");
  return SPLX_OK;
}

int launch_raster_bwd(splx_ctx* ctx, const splx_projected* pr, const splx_binning* bins, int K,
                      const CamDev& cam, const splx_partial* part, const float* g_ct, float* g2d) {
  const int ntiles = cam.TX * cam.TY;
  dim3 grid(ntiles, K);
  k_raster_bwd<<<grid, BLOCK, 0, ctx->stream>>>(pr->means2d, pr->conic_opacity, pr->rgb, bins->vals,
                                                bins->tile_ranges, cam.W, cam.H, cam.TX, ntiles, ctx->cfg,
                                                part->ct, part->n_contrib, g_ct, g2d);
  SPLX_LAUNCH_CHECK(ctx, "k_raster_bwd");
  return SPLX_OK;
}
