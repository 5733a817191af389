// dssim.cu -- the loss of PAPER.md L95 (section 2, step 4): "L = L_RGB + lambda L_D-SSIM", forward and gradient.
// The paper states neither lambda nor the SSIM window; reading s33: L_RGB = mean |image - target|,
// L_D-SSIM = 1 - mean SSIM, SSIM per colour channel over an 11 x 11 Gaussian window (sigma 1.5, weights summing to
// 1), C1 = 0.01^2, C2 = 0.03^2, zero padding (pixels outside the image add nothing to the window sums).
//
// Two HBM-bound kernels over 16 x 16 pixel tiles (+ 5 pixel halo), all three channels of a tile staged once in shared
// memory with coalesced row loads, the 11 x 11 window applied as a horizontal then a vertical 11-tap pass:
//   k_dssim_fwd: five window sums (mu_x, mu_y, E[x^2], E[y^2], E[xy]) -> SSIM(p) and its derivatives with respect
//                to the three sums that contain the image (mu_x, E[x^2], E[xy]) -> 3 maps in the workspace; block
//                sums of |x - y| and SSIM leave as two double atomics per CTA.
//   k_dssim_bwd: the three maps filtered with the same (symmetric) window give d(sum SSIM)/dx(q) =
//                F[d_mu](q) + 2 x(q) F[d_e2](q) + y(q) F[d_e12](q); dL/dx = s (sign(x - y) - lambda d(sum SSIM)/dx).
#include "common.cuh"

namespace {

constexpr int DR = 5;                       // window radius
constexpr int DT = SPLX_TILE;               // 16 x 16 output pixels per CTA
constexpr int DH = DT + 2 * DR;             // 26 rows / columns with the halo
constexpr int DROW = DH * 3;                // floats per staged row (three interleaved channels)
constexpr float DC1 = 0.01f * 0.01f, DC2 = 0.03f * 0.03f;

struct Win { float w[2 * DR + 1]; };

static Win make_window() {
  Win W;
  double s = 0.0, v[2 * DR + 1];
  for (int i = -DR; i <= DR; ++i) { v[i + DR] = exp(-(double)(i * i) / (2.0 * 1.5 * 1.5)); s += v[i + DR]; }
  for (int i = 0; i <= 2 * DR; ++i) W.w[i] = (float)(v[i] / s);
  return W;
}

// Stage rows [y0-5, y0+21) x columns [x0-5, x0+21) x 3 channels of `src` ([H][W][3]) into s[DH][DROW]; zeros outside.
__device__ __forceinline__ void stage_region(float* __restrict__ s, const float* __restrict__ src, int x0, int y0, int W, int H) {
  for (int e = threadIdx.x; e < DH * DROW; e += DT * DT) {
    const int r = e / DROW, c = e - r * DROW;
    const int y = y0 - DR + r, xc = (x0 - DR) * 3 + c;          // xc: float column inside the image row
    float v = 0.f;
    if (y >= 0 && y < H && xc >= 0 && xc < 3 * W) v = __ldg(src + (size_t)y * W * 3 + xc);
    s[e] = v;
  }
}

__global__ void __launch_bounds__(DT * DT)
k_dssim_fwd(const __grid_constant__ ViewBufs vb, int W, int H, int TX, const __grid_constant__ Win win,
            float* __restrict__ ws, size_t ws_view_stride, double* loss_sum) {
  __shared__ float s_x[DH * DROW], s_y[DH * DROW];
  __shared__ float s_h[5][DH][DT];          // horizontal pass of one channel
  __shared__ float s_red[2][DT * DT / 32];
  const int b = blockIdx.y, tile = blockIdx.x;
  const int x0 = (tile % TX) * DT, y0 = (tile / TX) * DT;
  const int tx = threadIdx.x & (DT - 1), ty = threadIdx.x >> 4;
  const float* x = vb.image[b];
  const float* y = vb.target[b];
  stage_region(s_x, x, x0, y0, W, H);
  stage_region(s_y, y, x0, y0, W, H);
  __syncthreads();
  const int px = x0 + tx, py = y0 + ty;
  const bool inside = px < W && py < H;
  const size_t HW = (size_t)W * H;
  float* wsb = ws + (size_t)b * ws_view_stride;
  float l1 = 0.f, ss = 0.f;
#pragma unroll 1
  for (int c = 0; c < 3; ++c) {
    for (int e = threadIdx.x; e < DH * DT; e += DT * DT) {          // 26 rows x 16 columns
      const int r = e >> 4, col = e & (DT - 1);
      float hx = 0.f, hy = 0.f, hxx = 0.f, hyy = 0.f, hxy = 0.f;
#pragma unroll
      for (int k = 0; k <= 2 * DR; ++k) {
        const float a = s_x[r * DROW + (col + k) * 3 + c], bb = s_y[r * DROW + (col + k) * 3 + c], w = win.w[k];
        const float wa = w * a, wb = w * bb;
        hx += wa; hy += wb; hxx = fmaf(wa, a, hxx); hyy = fmaf(wb, bb, hyy); hxy = fmaf(wa, bb, hxy);
      }
      s_h[0][r][col] = hx; s_h[1][r][col] = hy; s_h[2][r][col] = hxx; s_h[3][r][col] = hyy; s_h[4][r][col] = hxy;
    }
    __syncthreads();
    float mx = 0.f, my = 0.f, exx = 0.f, eyy = 0.f, exy = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * DR; ++k) {
      const float w = win.w[k];
      mx = fmaf(w, s_h[0][ty + k][tx], mx); my = fmaf(w, s_h[1][ty + k][tx], my);
      exx = fmaf(w, s_h[2][ty + k][tx], exx); eyy = fmaf(w, s_h[3][ty + k][tx], eyy);
      exy = fmaf(w, s_h[4][ty + k][tx], exy);
    }
    if (inside) {
      const float sxx = exx - mx * mx, syy = eyy - my * my, sxy = exy - mx * my;
      const float A1 = 2.f * mx * my + DC1, A2 = 2.f * sxy + DC2, B1 = mx * mx + my * my + DC1, B2 = sxx + syy + DC2;
      const float iB1 = 1.0f / B1, iB2 = 1.0f / B2;
      const float S = A1 * A2 * iB1 * iB2;
      ss += S;
      const float a = s_x[(ty + DR) * DROW + (tx + DR) * 3 + c], bb = s_y[(ty + DR) * DROW + (tx + DR) * 3 + c];
      l1 += fabsf(a - bb);
      // workspace: nine planes [map][channel][H][W] (planar, so that these stores and the backward's loads are coalesced)
      const size_t p = (size_t)c * HW + (size_t)py * W + px;
      wsb[p] = 2.f * my * (A2 - A1) * iB1 * iB2 - S * 2.f * mx * (iB1 - iB2);      // dS/dmu_x
      wsb[3 * HW + p] = -S * iB2;                                                  // dS/dE[x^2]
      wsb[6 * HW + p] = 2.f * A1 * iB1 * iB2;                                      // dS/dE[xy]
    }
    __syncthreads();
  }
  if (loss_sum) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { l1 += __shfl_xor_sync(0xffffffffu, l1, o); ss += __shfl_xor_sync(0xffffffffu, ss, o); }
    if ((threadIdx.x & 31) == 0) { s_red[0][threadIdx.x >> 5] = l1; s_red[1][threadIdx.x >> 5] = ss; }
    __syncthreads();
    if (threadIdx.x < 2) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < DT * DT / 32; ++w) t += s_red[threadIdx.x][w];
      atomicAdd(loss_sum + threadIdx.x, (double)t);
    }
  }
}

__global__ void __launch_bounds__(DT * DT)
k_dssim_bwd(const __grid_constant__ ViewBufs vb, int W, int H, int TX, const __grid_constant__ Win win,
            const float* __restrict__ ws, size_t ws_view_stride, float gscale, float lambda) {
  __shared__ float s_d[3][DH][DH + 1];      // the three derivative maps of one channel, tile + halo
  __shared__ float s_h[3][DH][DT];
  const int b = blockIdx.y, tile = blockIdx.x;
  const int x0 = (tile % TX) * DT, y0 = (tile / TX) * DT;
  const int tx = threadIdx.x & (DT - 1), ty = threadIdx.x >> 4;
  const size_t HW = (size_t)W * H;
  const float* wsb = ws + (size_t)b * ws_view_stride;
  const int px = x0 + tx, py = y0 + ty;
  const bool inside = px < W && py < H;
  float g[3] = {0.f, 0.f, 0.f};
  float xa[3] = {0.f, 0.f, 0.f}, ya[3] = {0.f, 0.f, 0.f};
  if (inside) {
    const size_t p = ((size_t)py * W + px) * 3;
#pragma unroll
    for (int c = 0; c < 3; ++c) { xa[c] = vb.image[b][p + c]; ya[c] = vb.target[b][p + c]; }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    for (int e = threadIdx.x; e < 3 * DH * DH; e += DT * DT) {
      const int m = e / (DH * DH), q = e - m * (DH * DH);
      const int r = q / DH, col = q - r * DH;
      const int y = y0 - DR + r, x = x0 - DR + col;
      float v = 0.f;
      if (y >= 0 && y < H && x >= 0 && x < W) v = __ldg(wsb + (size_t)(3 * m + c) * HW + (size_t)y * W + x);
      s_d[m][r][col] = v;
    }
    __syncthreads();
    for (int e = threadIdx.x; e < DH * DT; e += DT * DT) {
      const int r = e >> 4, col = e & (DT - 1);
      float h0 = 0.f, h1 = 0.f, h2 = 0.f;
#pragma unroll
      for (int k = 0; k <= 2 * DR; ++k) {
        const float w = win.w[k];
        h0 = fmaf(w, s_d[0][r][col + k], h0); h1 = fmaf(w, s_d[1][r][col + k], h1); h2 = fmaf(w, s_d[2][r][col + k], h2);
      }
      s_h[0][r][col] = h0; s_h[1][r][col] = h1; s_h[2][r][col] = h2;
    }
    __syncthreads();
    float f0 = 0.f, f1 = 0.f, f2 = 0.f;
#pragma unroll
    for (int k = 0; k <= 2 * DR; ++k) {
      const float w = win.w[k];
      f0 = fmaf(w, s_h[0][ty + k][tx], f0); f1 = fmaf(w, s_h[1][ty + k][tx], f1); f2 = fmaf(w, s_h[2][ty + k][tx], f2);
    }
    const float e = xa[c] - ya[c];
    const float sgn = e > 0.f ? 1.f : (e < 0.f ? -1.f : 0.f);
    g[c] = gscale * (sgn - lambda * (f0 + 2.f * xa[c] * f1 + ya[c] * f2));
    __syncthreads();
  }
  if (inside) {
    float* out = vb.g_image[b] + ((size_t)py * W + px) * 3;
    out[0] = g[0]; out[1] = g[1]; out[2] = g[2];
  }
}

}  // namespace

size_t dssim_ws_floats(int W, int H) { return (size_t)9 * W * H; }

// vb.image / vb.target / vb.g_image (written) of views 0..B-1; ws: B x dssim_ws_floats(W, H) floats.
// dL/dimage = scale / (B H W 3) (sign(image - target) - lambda d(sum SSIM)/dimage), as splx_l1_loss_grad scales.
int launch_dssim(splx_ctx* ctx, int B, int W, int H, const ViewBufs& vb, float lambda, float scale, double* loss_sum, float* ws) {
  static const Win win = make_window();
  const int TX = (W + DT - 1) / DT, TY = (H + DT - 1) / DT;
  const dim3 grid(TX * TY, B);
  const size_t stride = dssim_ws_floats(W, H);
  k_dssim_fwd<<<grid, DT * DT, 0, ctx->stream>>>(vb, W, H, TX, win, ws, stride, loss_sum);
  SPLX_LAUNCH_CHECK(ctx, "k_dssim_fwd");
  const float gscale = scale / (float)((int64_t)B * W * H * 3);
  k_dssim_bwd<<<grid, DT * DT, 0, ctx->stream>>>(vb, W, H, TX, win, ws, stride, gscale, lambda);
  SPLX_LAUNCH_CHECK(ctx, "k_dssim_bwd");
  return SPLX_OK;
}

// ---- splx_dssim_loss_grad_static: the entry point that allocates nothing (include/splx.h) ----------------------------
// The scratch is a file-scope device array.  In HOST code its name is a host-side stand-in, not a device address: the
// address comes from cudaGetSymbolAddress, looked up once per device with that device current, and only that pointer
// is handed to the kernels.
static __device__ __align__(256) float g_dssim_scratch[(size_t)9 * SPLX_DSSIM_STATIC_MAX_PIXELS];

namespace {
constexpr int MAX_DEVICES = 64;
float* g_scratch_ptr[MAX_DEVICES];      // device address of g_dssim_scratch on device d, nullptr until looked up
}  // namespace

extern "C" int splx_dssim_loss_grad_static(splx_ctx* ctx, int n_views, const splx_camera* cam, const float* image,
                                           const float* target, float lambda, float scale, float* dL_dimage, double* loss_sum) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if (!cam || cam->width <= 0 || cam->height <= 0 || n_views < 1 || n_views > SPLX_MAX_VIEWS || !image || !target ||
      !dL_dimage || !(lambda >= 0.f))
    SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_dssim_loss_grad_static: null argument, bad size, n_views not in [1,%d] or lambda < 0",
              SPLX_MAX_VIEWS);
  const long long pixels = (long long)n_views * cam->width * cam->height;
  if (pixels > (long long)SPLX_DSSIM_STATIC_MAX_PIXELS)
    SPLX_FAIL(ctx, SPLX_ERR_WORKSPACE, "splx_dssim_loss_grad_static: n_views * W * H = %lld pixels exceed the static scratch of %d "
              "pixels (SPLX_DSSIM_STATIC_MAX_PIXELS); use splx_dssim_loss_grad with a workspace", pixels, SPLX_DSSIM_STATIC_MAX_PIXELS);
  if (ctx->device < 0 || ctx->device >= MAX_DEVICES) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_dssim_loss_grad_static: device %d", ctx->device);
  float* ws = g_scratch_ptr[ctx->device];
  if (!ws) {   // set-up, once per device: the symbol's address ON THE CONTEXT'S DEVICE
    int cur = -1;
    SPLX_CUDA_OK(ctx, cudaGetDevice(&cur));
    if (cur != ctx->device) SPLX_CUDA_OK(ctx, cudaSetDevice(ctx->device));
    const cudaError_t e = cudaGetSymbolAddress((void**)&ws, g_dssim_scratch);
    if (cur != ctx->device) cudaSetDevice(cur);
    if (e != cudaSuccess || !ws) SPLX_FAIL(ctx, SPLX_ERR_CUDA, "cudaGetSymbolAddress(g_dssim_scratch) failed: %s", cudaGetErrorString(e));
    g_scratch_ptr[ctx->device] = ws;
  }
  const ViewBufs vb = contiguous_views(n_views, (size_t)cam->width * cam->height, target, const_cast<float*>(image), nullptr,
                                       dL_dimage, nullptr);
  return launch_dssim(ctx, n_views, cam->width, cam->height, vb, lambda, scale, loss_sum, ws);
}
