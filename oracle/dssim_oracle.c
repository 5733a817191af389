/* dssim_oracle.c -- CPU oracle of the D-SSIM loss term.  TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it; it shares no code with
 * the CUDA path.
 *
 * PAPER.md L95 (section 2, step 4): "L = L_RGB + lambda L_D-SSIM".  The paper gives neither lambda nor the
 * window; reading s33 of DESIGN.md: L_D-SSIM = 1 - mean SSIM(image, target), SSIM of Wang et
 * al. (2004) per colour channel with an 11 x 11 Gaussian window (sigma 1.5, weights normalised to sum 1),
 * C1 = 0.01^2, C2 = 0.03^2 (dynamic range 1), the window sums running over the pixels INSIDE the image only
 * (zero padding: an outside pixel adds nothing to any of the five sums), mean over all H*W*3 values; lambda = 0.2.
 *
 * This file is that definition written out: the five window sums as direct 121-term double loops per pixel (no
 * separable passes, no tiling), SSIM from them, and the derivative of the mean SSIM with respect to the first image
 * by the chain rule through the three window sums that contain it (mu_x, E[x^2], E[xy]), again as direct loops.
 * fp64 throughout.  Pins: tests/test_oracle_dssim.py (identical images, constant images closed form, central
 * differences, a torch conv2d + autograd restatement). */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define R 5               /* window radius: 11 x 11 */
#define SIGMA 1.5
#define C1 (0.01 * 0.01)
#define C2 (0.03 * 0.03)

static void window(double w[2 * R + 1]) {
  double s = 0.0;
  for (int i = -R; i <= R; ++i) { w[i + R] = exp(-(double)(i * i) / (2.0 * SIGMA * SIGMA)); s += w[i + R]; }
  for (int i = 0; i <= 2 * R; ++i) w[i] /= s;        /* the 2-D window w[i] w[j] then sums to 1 */
}

/* x, y: [H][W][C] (x = rendered image, y = target).  Returns mean SSIM over H*W*C.
 * ssim_map (may be NULL): [H][W][C].  g_x (may be NULL): d(mean SSIM)/dx, [H][W][C]. */
double orc_ssim(int W, int H, int C, const double* x, const double* y, double* ssim_map, double* g_x) {
  double w[2 * R + 1];
  window(w);
  const size_t n = (size_t)W * H * C;
  /* derivative of SSIM(p) with respect to the three window sums that contain x */
  double* d_mu = (double*)calloc(n, sizeof(double));
  double* d_e2 = (double*)calloc(n, sizeof(double));
  double* d_e12 = (double*)calloc(n, sizeof(double));
  double total = 0.0;
  for (int py = 0; py < H; ++py)
    for (int px = 0; px < W; ++px)
      for (int c = 0; c < C; ++c) {
        double mx = 0, my = 0, exx = 0, eyy = 0, exy = 0;
        for (int dy = -R; dy <= R; ++dy)
          for (int dx = -R; dx <= R; ++dx) {
            const int qy = py + dy, qx = px + dx;
            if (qy < 0 || qy >= H || qx < 0 || qx >= W) continue;     /* zero padding */
            const double ww = w[dy + R] * w[dx + R];
            const double a = x[((size_t)qy * W + qx) * C + c], b = y[((size_t)qy * W + qx) * C + c];
            mx += ww * a; my += ww * b; exx += ww * a * a; eyy += ww * b * b; exy += ww * a * b;
          }
        const double sxx = exx - mx * mx, syy = eyy - my * my, sxy = exy - mx * my;
        const double A1 = 2 * mx * my + C1, A2 = 2 * sxy + C2, B1 = mx * mx + my * my + C1, B2 = sxx + syy + C2;
        const double S = (A1 * A2) / (B1 * B2);
        const size_t p = ((size_t)py * W + px) * C + c;
        if (ssim_map) ssim_map[p] = S;
        total += S;
        /* with (mu_x, E[x^2], E[xy]) as the independent variables:
         *   dA1/dmu = 2 mu_y, dA2/dmu = -2 mu_y, dB1/dmu = 2 mu_x, dB2/dmu = -2 mu_x,
         *   dB2/dE[x^2] = 1, dA2/dE[xy] = 2 */
        d_mu[p] = (2 * my * A2 - 2 * my * A1) / (B1 * B2) - S * (2 * mx / B1 - 2 * mx / B2);
        d_e2[p] = -S / B2;
        d_e12[p] = 2 * A1 / (B1 * B2);
      }
  if (g_x) {
    for (int qy = 0; qy < H; ++qy)
      for (int qx = 0; qx < W; ++qx)
        for (int c = 0; c < C; ++c) {
          const size_t q = ((size_t)qy * W + qx) * C + c;
          double acc = 0.0;
          for (int dy = -R; dy <= R; ++dy)
            for (int dx = -R; dx <= R; ++dx) {
              const int py = qy + dy, px = qx + dx;       /* pixels p whose window holds q */
              if (py < 0 || py >= H || px < 0 || px >= W) continue;
              const size_t p = ((size_t)py * W + px) * C + c;
              acc += w[dy + R] * w[dx + R] * (d_mu[p] + 2 * x[q] * d_e2[p] + y[q] * d_e12[p]);
            }
          g_x[q] = acc / (double)n;
        }
  }
  free(d_mu); free(d_e2); free(d_e12);
  return total / (double)n;
}
