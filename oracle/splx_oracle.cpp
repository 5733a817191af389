// splx_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of the Splaxel pixel-level hot
// path (arxiv/paper_2606_18588), written from PAPER.md and from the readings
// listed in DESIGN.md ("Readings of the paper", s1..s26).  It exists so that
// the CUDA path can be checked against something that a reader can compare
// with the paper by eye.  It shares no code with the CUDA path: only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load it.  All floating point data crosses this boundary as double;
// every fp32 value is exactly representable, so the same routines serve the
// teacher-forced checks (fp32 GPU outputs in) and the finite-difference pins
// (double in).  Integer decisions that the kernel takes in fp32 (tile rect,
// depth key bits) are taken in fp32 here too, as stated at each site.
//
// Stage map (one function per step of SURVEY.md s8(a)):
//   orc_project          PAPER.md L76, L80 (s2 step 1): Sigma = R S S^T R^T,
//                        Sigma2D = J W Sigma W^T J^T, 2-D mean, depth d
//   orc_bin_sort         PAPER.md L81 (s2 step 2: sort by depth d), L165
//   orc_render_partial   PAPER.md L84 Eq.1, L93 Eq.2, L167 Eq.3, L172 Eq.4
//   orc_compose          PAPER.md L176-L178 Eq.5
//   orc_compose_bwd      PAPER.md L186-L188 Eq.6-7
//   orc_raster_bwd       PAPER.md L184 (gradient through the partial pixel)
//   orc_project_bwd      PAPER.md L95 (back-propagated to all parameters)
//   orc_adam             optimiser step (paper silent; Adam per north_star)
//   orc_l1               PAPER.md L95 (L_RGB term only)
//
// Pins (tests/test_oracle_*.py): closed forms, brute force, finite
// differences, fp64 autograd on a dense restatement, torch.optim.Adam.
// Parity unpinned (nothing printed in the paper fixes them):
//   * the SH sign/ordering convention (self-consistent only),
//   * the per-pixel partition order for partitions that are not separated
//     in depth (only the depth-separated invariant of L180 is pinned).

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

constexpr int TILE = 16;  // reading s1

struct Cam {
  double R[9], t[3], fx, fy, cx, cy;
  int W, H;
  double near_z;
};
// cam layout: R[0..8] row-major (p_cam = R*mean + t), t[9..11], fx, fy, cx, cy, W, H, near_z
Cam load_cam(const double* c) {
  Cam k;
  for (int i = 0; i < 9; ++i) k.R[i] = c[i];
  for (int i = 0; i < 3; ++i) k.t[i] = c[9 + i];
  k.fx = c[12]; k.fy = c[13]; k.cx = c[14]; k.cy = c[15];
  k.W = (int)c[16]; k.H = (int)c[17]; k.near_z = c[18];
  return k;
}
struct Cfg {
  double alpha_min, alpha_max, T_eps, dilation, lim_factor, radius_floor;
};
// cfg layout: alpha_min (1/255), alpha_max (0.99), T_eps (1e-4), dilation (0.3),
//             lim_factor (1.3), radius_floor (0.1)     -- readings s2, s9
Cfg load_cfg(const double* c) { return Cfg{c[0], c[1], c[2], c[3], c[4], c[5]}; }

inline int tiles_x(int W) { return (W + TILE - 1) / TILE; }
inline int tiles_y(int H) { return (H + TILE - 1) / TILE; }

// Unit quaternion (w,x,y,z) -> rotation matrix (row-major).
void quat_to_rot(const double q[4], double Rm[9]) {
  const double w = q[0], x = q[1], y = q[2], z = q[3];
  Rm[0] = 1 - 2 * (y * y + z * z); Rm[1] = 2 * (x * y - w * z);     Rm[2] = 2 * (x * z + w * y);
  Rm[3] = 2 * (x * y + w * z);     Rm[4] = 1 - 2 * (x * x + z * z); Rm[5] = 2 * (y * z - w * x);
  Rm[6] = 2 * (x * z - w * y);     Rm[7] = 2 * (y * z + w * x);     Rm[8] = 1 - 2 * (x * x + y * y);
}

// Real spherical-harmonic basis up to degree 3 (reading s13).  The constants
// are the orthonormal ones: Y00 = 1/2 sqrt(1/pi) etc.; tests pin them by
// quadrature.  Y[l] for l < (deg+1)^2; dY[l][3] = gradient of the polynomial
// with respect to the (unconstrained) direction components.
void sh_basis(int deg, const double d[3], double Y[16], double dY[16][3]) {
  const double PI = 3.14159265358979323846;
  const double x = d[0], y = d[1], z = d[2];
  for (int l = 0; l < 16; ++l) { Y[l] = 0; dY[l][0] = dY[l][1] = dY[l][2] = 0; }
  Y[0] = 0.5 * std::sqrt(1.0 / PI);
  if (deg < 1) return;
  const double k1 = std::sqrt(3.0 / (4.0 * PI));
  Y[1] = -k1 * y; dY[1][1] = -k1;
  Y[2] = k1 * z;  dY[2][2] = k1;
  Y[3] = -k1 * x; dY[3][0] = -k1;
  if (deg < 2) return;
  const double k2a = 0.5 * std::sqrt(15.0 / PI), k2b = 0.25 * std::sqrt(5.0 / PI),
               k2c = 0.25 * std::sqrt(15.0 / PI);
  Y[4] = k2a * x * y;   dY[4][0] = k2a * y;  dY[4][1] = k2a * x;
  Y[5] = -k2a * y * z;  dY[5][1] = -k2a * z; dY[5][2] = -k2a * y;
  Y[6] = k2b * (2 * z * z - x * x - y * y);
  dY[6][0] = -2 * k2b * x; dY[6][1] = -2 * k2b * y; dY[6][2] = 4 * k2b * z;
  Y[7] = -k2a * x * z;  dY[7][0] = -k2a * z; dY[7][2] = -k2a * x;
  Y[8] = k2c * (x * x - y * y); dY[8][0] = 2 * k2c * x; dY[8][1] = -2 * k2c * y;
  if (deg < 3) return;
  const double k3a = 0.25 * std::sqrt(35.0 / (2.0 * PI)), k3b = 0.5 * std::sqrt(105.0 / PI),
               k3c = 0.25 * std::sqrt(21.0 / (2.0 * PI)), k3d = 0.25 * std::sqrt(7.0 / PI),
               k3e = 0.25 * std::sqrt(105.0 / PI);
  Y[9] = -k3a * y * (3 * x * x - y * y);
  dY[9][0] = -k3a * 6 * x * y; dY[9][1] = -k3a * (3 * x * x - 3 * y * y);
  Y[10] = k3b * x * y * z;
  dY[10][0] = k3b * y * z; dY[10][1] = k3b * x * z; dY[10][2] = k3b * x * y;
  Y[11] = -k3c * y * (4 * z * z - x * x - y * y);
  dY[11][0] = k3c * 2 * x * y; dY[11][1] = -k3c * (4 * z * z - x * x - 3 * y * y);
  dY[11][2] = -k3c * 8 * y * z;
  Y[12] = k3d * z * (2 * z * z - 3 * x * x - 3 * y * y);
  dY[12][0] = -k3d * 6 * x * z; dY[12][1] = -k3d * 6 * y * z;
  dY[12][2] = k3d * (6 * z * z - 3 * x * x - 3 * y * y);
  Y[13] = -k3c * x * (4 * z * z - x * x - y * y);
  dY[13][0] = -k3c * (4 * z * z - 3 * x * x - y * y); dY[13][1] = k3c * 2 * x * y;
  dY[13][2] = -k3c * 8 * x * z;
  Y[14] = k3e * z * (x * x - y * y);
  dY[14][0] = k3e * 2 * x * z; dY[14][1] = -k3e * 2 * y * z; dY[14][2] = k3e * (x * x - y * y);
  Y[15] = -k3a * x * (x * x - 3 * y * y);
  dY[15][0] = -k3a * (3 * x * x - 3 * y * y); dY[15][1] = k3a * 6 * x * y;
}

// Tile rectangle of a projected Gaussian (reading s11).  Pixel (i,j) samples
// the point (i+0.5, j+0.5), so a footprint [u-r, u+r] covers pixel columns
// i with u-0.5-r <= i <= u-0.5+r.  This decision is taken in fp32 from the
// fp32-rounded (u, v) because the kernel takes it in fp32: two subtractions,
// an exact scaling by 1/16, floor.  No multiply-add occurs, so the result does
// not depend on FMA contraction.
void tile_rect(double u, double v, int radius, int W, int H, int rect[4]) {
  const int TX = tiles_x(W), TY = tiles_y(H);
  const float uf = (float)u, vf = (float)v, rf = (float)radius;
  const float ux = uf - 0.5f, vy = vf - 0.5f;
  const float x0f = std::floor((ux - rf) * 0.0625f);
  const float x1f = std::floor(((ux + rf) + 15.0f) * 0.0625f);
  const float y0f = std::floor((vy - rf) * 0.0625f);
  const float y1f = std::floor(((vy + rf) + 15.0f) * 0.0625f);
  auto clampi = [](float f, int hi) {
    if (!(f > 0.0f)) return 0;           // also catches NaN
    if (f >= (float)hi) return hi;
    return (int)f;
  };
  rect[0] = clampi(x0f, TX); rect[1] = clampi(y0f, TY);
  rect[2] = clampi(x1f, TX); rect[3] = clampi(y1f, TY);
}

inline uint32_t float_bits(float f) { uint32_t b; std::memcpy(&b, &f, 4); return b; }

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------
// O1 projection.  PAPER.md L76 (Sigma = R S S^T R^T), L80 (frustum cull by the
// mean; Sigma2D = J W Sigma W^T J^T; depth d; 2-D mean).  Readings s5, s8-s11,
// s13, s14.  A culled Gaussian gets radius = 0, tiles_touched = 0, zeros.
// Outputs (all caller-allocated): means2d[n,2], depth[n], conic_opacity[n,4],
// rgb[n,3], radius[n], tiles_touched[n], clamp[n] (bit c set when channel c
// was clamped at 0), rect[n,4] = x0,y0,x1,y1, radius_margin[n] = distance of
// 3*sqrt(lambda) to the integer below its ceiling, relative (for the
// fragile-Gaussian protocol; +inf when culled).
// ---------------------------------------------------------------------------
void orc_project(int64_t n, const double* mean, const double* log_scale, const double* quat,
                 const double* opacity_logit, const double* sh, int sh_degree,
                 const double* cam_, const double* cfg_, double* means2d, double* depth,
                 double* conic_opacity, double* rgb, int32_t* radius, uint32_t* tiles_touched,
                 uint8_t* clamp, int32_t* rect, double* radius_margin) {
  const Cam cam = load_cam(cam_);
  const Cfg cfg = load_cfg(cfg_);
  const int nsh = (sh_degree + 1) * (sh_degree + 1);
  // camera centre o = -R^T t
  double o[3];
  for (int j = 0; j < 3; ++j)
    o[j] = -(cam.R[0 * 3 + j] * cam.t[0] + cam.R[1 * 3 + j] * cam.t[1] + cam.R[2 * 3 + j] * cam.t[2]);
  for (int64_t i = 0; i < n; ++i) {
    means2d[2 * i] = means2d[2 * i + 1] = 0; depth[i] = 0;
    for (int c = 0; c < 4; ++c) conic_opacity[4 * i + c] = 0;
    for (int c = 0; c < 3; ++c) rgb[3 * i + c] = 0;
    radius[i] = 0; tiles_touched[i] = 0; clamp[i] = 0;
    for (int c = 0; c < 4; ++c) rect[4 * i + c] = 0;
    radius_margin[i] = std::numeric_limits<double>::infinity();

    const double* mu = mean + 3 * i;
    double p[3];
    for (int r = 0; r < 3; ++r)
      p[r] = cam.R[3 * r] * mu[0] + cam.R[3 * r + 1] * mu[1] + cam.R[3 * r + 2] * mu[2] + cam.t[r];
    if (p[2] <= cam.near_z) continue;  // s8: cull by the mean's camera depth only

    // Sigma = Rot S S^T Rot^T  (L76)
    double s[3] = {std::exp(log_scale[3 * i]), std::exp(log_scale[3 * i + 1]),
                   std::exp(log_scale[3 * i + 2])};
    const double* q = quat + 4 * i;
    const double qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    const double qh[4] = {q[0] / qn, q[1] / qn, q[2] / qn, q[3] / qn};
    double Rot[9]; quat_to_rot(qh, Rot);
    double Mm[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) Mm[3 * r + c] = Rot[3 * r + c] * s[c];
    double Sig[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += Mm[3 * r + k] * Mm[3 * c + k];
      Sig[3 * r + c] = a;
    }
    // J: Jacobian of (x,y,z) -> (fx x/z, fy y/z), evaluated at a point whose
    // x/z, y/z are clamped to +-1.3 tan(fov/2)  (s9)
    const double z = p[2];
    const double limx = cfg.lim_factor * cam.W / (2.0 * cam.fx);
    const double limy = cfg.lim_factor * cam.H / (2.0 * cam.fy);
    const double tx = std::min(limx, std::max(-limx, p[0] / z)) * z;
    const double ty = std::min(limy, std::max(-limy, p[1] / z)) * z;
    const double J[6] = {cam.fx / z, 0, -cam.fx * tx / (z * z), 0, cam.fy / z, -cam.fy * ty / (z * z)};
    double Tm[6];  // J * W, W = camera rotation (L80)
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += J[3 * r + k] * cam.R[3 * k + c];
      Tm[3 * r + c] = a;
    }
    double TS[6];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += Tm[3 * r + k] * Sig[3 * k + c];
      TS[3 * r + c] = a;
    }
    double cov[4];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 2; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += TS[3 * r + k] * Tm[3 * c + k];
      cov[2 * r + c] = a;
    }
    const double a = cov[0] + cfg.dilation, b = cov[1], c = cov[3] + cfg.dilation;
    const double det = a * c - b * b;
    if (det <= 0) continue;
    const double mid = 0.5 * (a + c);
    const double lam = mid + std::sqrt(std::max(cfg.radius_floor, mid * mid - det));
    const double r3 = 3.0 * std::sqrt(lam);
    const int rad = (int)std::ceil(r3);
    const double u = cam.fx * p[0] / z + cam.cx, v = cam.fy * p[1] / z + cam.cy;
    int rc[4]; tile_rect(u, v, rad, cam.W, cam.H, rc);
    const int tt = (rc[2] - rc[0]) * (rc[3] - rc[1]);
    if (tt <= 0) continue;

    means2d[2 * i] = u; means2d[2 * i + 1] = v; depth[i] = z;  // s5: depth = camera-space z
    conic_opacity[4 * i + 0] = c / det;
    conic_opacity[4 * i + 1] = -b / det;
    conic_opacity[4 * i + 2] = a / det;
    conic_opacity[4 * i + 3] = 1.0 / (1.0 + std::exp(-opacity_logit[i]));
    radius[i] = rad; tiles_touched[i] = (uint32_t)tt;
    for (int k = 0; k < 4; ++k) rect[4 * i + k] = rc[k];
    radius_margin[i] = ((double)rad - r3) / r3;

    // colour: SH evaluated along the direction from the camera centre (s13)
    double d[3] = {mu[0] - o[0], mu[1] - o[1], mu[2] - o[2]};
    const double dn = std::sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    for (int k = 0; k < 3; ++k) d[k] /= dn;
    double Y[16], dY[16][3]; sh_basis(sh_degree, d, Y, dY);
    for (int ch = 0; ch < 3; ++ch) {
      double val = 0.5;
      for (int l = 0; l < nsh; ++l) val += Y[l] * sh[(i * 16 + l) * 3 + ch];
      if (val < 0) { clamp[i] |= (uint8_t)(1u << ch); val = 0; }
      rgb[3 * i + ch] = val;
    }
  }
}

// ---------------------------------------------------------------------------
// The depth as the SORT KEY sees it.  Reading s12: key = (tile << 32) | float_bits(depth), an integer decision taken in
// fp32 -- by both sides in the same precision and the same operation order, so that two Gaussians whose depths differ
// by less than an fp32 rounding are ordered alike by the oracle and by the kernel:
//   z32 = fl(fma(R22, mz, fma(R21, my, fl(R20 * mx))) + t2)        (all operands rounded to fp32 first)
// Only the ORDER uses it; the depth that enters the partial depth D (Eq.4) stays the fp64 value of orc_project.
// ---------------------------------------------------------------------------
void orc_depth_key(int64_t n, const double* mean, const double* cam_, double* depth32) {
  const Cam cam = load_cam(cam_);
  const float r0 = (float)cam.R[6], r1 = (float)cam.R[7], r2 = (float)cam.R[8], t2 = (float)cam.t[2];
  for (int64_t i = 0; i < n; ++i) {
    const float mx = (float)mean[3 * i], my = (float)mean[3 * i + 1], mz = (float)mean[3 * i + 2];
    const float z = std::fmaf(r2, mz, std::fmaf(r1, my, r0 * mx)) + t2;
    depth32[i] = (double)z;
  }
}

// ---------------------------------------------------------------------------
// O2 tile binning + depth sort.  PAPER.md L81 ("sorted based on their distance
// from the camera, i.e., depth d"), L165 ("sorted locally by depth").  The
// mechanism (tile|depth 64-bit keys, stable order, per-tile ranges) is reading
// s12.  Takes the projected (means2d, radius, depth); the rect is recomputed.
// orc_count_tiles returns M and fills tiles_touched; orc_bin_sort fills
// offsets[n] (inclusive prefix sum), keys[M], vals[M], ranges[TX*TY,2].
// ---------------------------------------------------------------------------
uint64_t orc_count_tiles(int64_t n, const double* means2d, const int32_t* radius, int W, int H,
                         uint32_t* tiles_touched) {
  uint64_t M = 0;
  for (int64_t i = 0; i < n; ++i) {
    uint32_t tt = 0;
    if (radius[i] > 0) {
      int rc[4]; tile_rect(means2d[2 * i], means2d[2 * i + 1], radius[i], W, H, rc);
      tt = (uint32_t)((rc[2] - rc[0]) * (rc[3] - rc[1]));
    }
    tiles_touched[i] = tt; M += tt;
  }
  return M;
}

void orc_bin_sort(int64_t n, const double* means2d, const int32_t* radius, const double* depth,
                  int W, int H, uint32_t* offsets, uint64_t* keys, uint32_t* vals,
                  uint32_t* ranges) {
  const int TX = tiles_x(W), TY = tiles_y(H);
  struct Item { uint64_t key; uint32_t val; };
  std::vector<Item> items;
  uint64_t run = 0;
  for (int64_t i = 0; i < n; ++i) {
    if (radius[i] > 0) {
      int rc[4]; tile_rect(means2d[2 * i], means2d[2 * i + 1], radius[i], W, H, rc);
      for (int ty = rc[1]; ty < rc[3]; ++ty)
        for (int tx = rc[0]; tx < rc[2]; ++tx) {
          const uint64_t tile = (uint64_t)ty * TX + tx;
          items.push_back(Item{(tile << 32) | float_bits((float)depth[i]), (uint32_t)i});
          ++run;
        }
    }
    offsets[i] = (uint32_t)run;
  }
  std::stable_sort(items.begin(), items.end(),
                   [](const Item& a, const Item& b) { return a.key < b.key; });
  for (int t = 0; t < TX * TY; ++t) ranges[2 * t] = ranges[2 * t + 1] = 0;
  for (size_t k = 0; k < items.size(); ++k) {
    keys[k] = items[k].key; vals[k] = items[k].val;
    const uint32_t t = (uint32_t)(items[k].key >> 32);
    if (k == 0 || (uint32_t)(items[k - 1].key >> 32) != t) ranges[2 * t] = (uint32_t)k;
    ranges[2 * t + 1] = (uint32_t)k + 1;
  }
}

// ---------------------------------------------------------------------------
// O3 local (per-partition) render.  PAPER.md Eq.1 (L84), Eq.3 (L167), Eq.4
// (L172, read as D = sum d_i alpha_i T_i: reading s3), blending rules of
// reading s2: skip power>0, alpha = min(alpha_max, o*exp(power)), skip
// alpha < alpha_min, stop BEFORE applying a Gaussian that would take T below
// T_eps.  A pixel walks the sorted list of its tile and nothing else.
// tile_list (n_tiles entries) restricts the work to those tiles; NULL = all.
// Outputs per pixel: ct[H,W,4] = (C.rgb premultiplied, T), d[H,W],
// n_contrib[H,W] = 1 + list position of the last contributor (0 if none),
// margin[H,W] = smallest relative distance of any decision taken for this
// pixel to its threshold (fragile-pixel protocol), t_exit[H,W] = T at the early
// exit if the walk ended by it, else -1.  Returns the number of list entries
// walked (pair evaluations), summed over the processed pixels.
// Pixels of tiles not in tile_list are left untouched.
// ---------------------------------------------------------------------------
uint64_t orc_render_partial(const double* means2d, const double* conic_opacity, const double* rgb,
                            const double* depth, const uint32_t* vals, const uint32_t* ranges,
                            int W, int H, const double* cfg_, const int32_t* tile_list,
                            int64_t n_tiles, double* ct, double* d, uint32_t* n_contrib,
                            double* margin, double* t_exit) {
  const Cfg cfg = load_cfg(cfg_);
  const int TX = tiles_x(W), TY = tiles_y(H);
  uint64_t walked = 0;
  const int64_t nt = tile_list ? n_tiles : (int64_t)TX * TY;
  for (int64_t it = 0; it < nt; ++it) {
    const int t = tile_list ? tile_list[it] : (int)it;
    const int ty = t / TX, tx = t % TX;
    const uint32_t r0 = ranges[2 * t], r1 = ranges[2 * t + 1];
    for (int j = ty * TILE; j < std::min(H, (ty + 1) * TILE); ++j)
      for (int i = tx * TILE; i < std::min(W, (tx + 1) * TILE); ++i) {
        double T = 1, C[3] = {0, 0, 0}, D = 0, mg = std::numeric_limits<double>::infinity();
        double te = -1; uint32_t nc = 0;
        const double px = i + 0.5, py = j + 0.5;  // s10
        for (uint32_t pos = r0; pos < r1; ++pos) {
          ++walked;
          const uint32_t g = vals[pos];
          const double dx = means2d[2 * g] - px, dy = means2d[2 * g + 1] - py;
          const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1],
                       Cc = conic_opacity[4 * g + 2], op = conic_opacity[4 * g + 3];
          const double t1 = A * dx * dx, t2 = Cc * dy * dy, t3 = B * dx * dy;
          const double power = -0.5 * (t1 + t2) - t3;  // exponent of Eq.1
          const double mag = 0.5 * (std::fabs(t1) + std::fabs(t2)) + std::fabs(t3);
          if (mag > 0) mg = std::min(mg, std::fabs(power) / mag);
          if (power > 0) continue;
          const double alpha = std::min(cfg.alpha_max, op * std::exp(power));  // Eq.1
          if (cfg.alpha_min > 0) mg = std::min(mg, std::fabs(alpha - cfg.alpha_min) / cfg.alpha_min);
          if (alpha < cfg.alpha_min) continue;
          const double Tn = T * (1 - alpha);
          if (cfg.T_eps > 0) mg = std::min(mg, std::fabs(Tn - cfg.T_eps) / cfg.T_eps);
          if (Tn < cfg.T_eps) { te = T; break; }
          const double w = alpha * T;  // alpha_i T_i, T_i = prod_{j<i}(1-alpha_j)
          for (int c = 0; c < 3; ++c) C[c] += w * rgb[3 * g + c];  // Eq.3
          D += w * depth[g];                                        // Eq.4 (s3)
          T = Tn;
          nc = pos - r0 + 1;
        }
        const int64_t pix = (int64_t)j * W + i;
        ct[4 * pix] = C[0]; ct[4 * pix + 1] = C[1]; ct[4 * pix + 2] = C[2]; ct[4 * pix + 3] = T;
        d[pix] = D; n_contrib[pix] = nc; margin[pix] = mg; t_exit[pix] = te;
      }
  }
  return walked;
}

// ---------------------------------------------------------------------------
// O4 global composition.  PAPER.md L176-L178, Eq.5: per pixel, sort the
// partials by partial depth, accumulate front to back with the partial
// transmittances.  Ordering key = D/(1-T) (reading s3), +inf for a partition
// that blended nothing (T == 1; it is the identity element wherever it lands),
// stable by partition index (s4).  bg is blended behind everything (s7).
// ct[K,H,W,4], d[K,H,W] -> image[H,W,3], T_total[H,W], order[H,W,K] (the
// permutation used, front first), order_margin[H,W] = smallest relative gap
// between adjacent finite keys (+inf if fewer than two).
// tile_list restricts the pixels as in orc_render_partial.
// ---------------------------------------------------------------------------
static void compose_order(int K, const double* ct, const double* d, int64_t HW, int64_t pix,
                          int* perm, double* gap) {
  double key[64];
  for (int k = 0; k < K; ++k) {
    const double T = ct[((int64_t)k * HW + pix) * 4 + 3];
    key[k] = (T < 1.0) ? d[(int64_t)k * HW + pix] / (1.0 - T) : std::numeric_limits<double>::infinity();
    perm[k] = k;
  }
  std::stable_sort(perm, perm + K, [&](int a, int b) { return key[a] < key[b]; });
  double g = std::numeric_limits<double>::infinity();
  for (int k = 0; k + 1 < K; ++k) {
    const double ka = key[perm[k]], kb = key[perm[k + 1]];
    if (std::isfinite(ka) && std::isfinite(kb)) {
      const double den = std::max(std::fabs(ka), std::fabs(kb));
      g = std::min(g, den > 0 ? (kb - ka) / den : 0.0);
    }
  }
  if (gap) *gap = g;
}

void orc_compose(int K, const double* ct, const double* d, int W, int H, const double* bg,
                 const int32_t* tile_list, int64_t n_tiles, double* image, double* T_total,
                 int32_t* order, double* order_margin) {
  const int TX = tiles_x(W), TY = tiles_y(H);
  const int64_t HW = (int64_t)W * H;
  const int64_t nt = tile_list ? n_tiles : (int64_t)TX * TY;
  for (int64_t it = 0; it < nt; ++it) {
    const int t = tile_list ? tile_list[it] : (int)it;
    const int ty = t / TX, tx = t % TX;
    for (int j = ty * TILE; j < std::min(H, (ty + 1) * TILE); ++j)
      for (int i = tx * TILE; i < std::min(W, (tx + 1) * TILE); ++i) {
        const int64_t pix = (int64_t)j * W + i;
        int perm[64]; double gap;
        compose_order(K, ct, d, HW, pix, perm, &gap);
        double Tacc = 1, C[3] = {0, 0, 0};
        for (int m = 0; m < K; ++m) {  // Eq.5: C = sum_m C^m prod_{k<m} T^k
          const double* p = ct + ((int64_t)perm[m] * HW + pix) * 4;
          for (int c = 0; c < 3; ++c) C[c] += Tacc * p[c];
          Tacc *= p[3];
          order[pix * K + m] = perm[m];
        }
        for (int c = 0; c < 3; ++c) image[3 * pix + c] = C[c] + Tacc * bg[c];
        T_total[pix] = Tacc;
        order_margin[pix] = gap;
      }
  }
}

// ---------------------------------------------------------------------------
// O6 composition backward.  PAPER.md L186 Eq.6, L188 Eq.7: for partition m at
// composition rank r, dL/dC^m = (prod_{k<m} T^k) dL/dC and
// dL/dT^m = (prod_{k<m} T^k) <dL/dC, Behind_m> where Behind_m is the colour
// composited from everything behind m (including bg).  g_T_total (may be
// NULL) is an optional gradient on T_total.  No gradient flows through D or
// through the order.  Output g_ct[K,H,W,4] = (dL/dC^k.rgb, dL/dT^k).
// ---------------------------------------------------------------------------
void orc_compose_bwd(int K, const double* ct, const double* d, int W, int H, const double* bg,
                     const double* g_image, const double* g_T_total, const int32_t* tile_list,
                     int64_t n_tiles, double* g_ct) {
  const int TX = tiles_x(W), TY = tiles_y(H);
  const int64_t HW = (int64_t)W * H;
  const int64_t nt = tile_list ? n_tiles : (int64_t)TX * TY;
  for (int64_t it = 0; it < nt; ++it) {
    const int t = tile_list ? tile_list[it] : (int)it;
    const int ty = t / TX, tx = t % TX;
    for (int j = ty * TILE; j < std::min(H, (ty + 1) * TILE); ++j)
      for (int i = tx * TILE; i < std::min(W, (tx + 1) * TILE); ++i) {
        const int64_t pix = (int64_t)j * W + i;
        int perm[64];
        compose_order(K, ct, d, HW, pix, perm, nullptr);
        double Tfront[64], Tacc = 1;
        for (int m = 0; m < K; ++m) { Tfront[m] = Tacc; Tacc *= ct[((int64_t)perm[m] * HW + pix) * 4 + 3]; }
        const double* g = g_image + 3 * pix;
        const double gT = g_T_total ? g_T_total[pix] : 0.0;
        double Behind[3] = {bg[0], bg[1], bg[2]}, BehindT = 1;
        for (int m = K - 1; m >= 0; --m) {
          const int k = perm[m];
          const double* p = ct + ((int64_t)k * HW + pix) * 4;
          double* o = g_ct + ((int64_t)k * HW + pix) * 4;
          for (int c = 0; c < 3; ++c) o[c] = Tfront[m] * g[c];                              // Eq.7
          o[3] = Tfront[m] * (g[0] * Behind[0] + g[1] * Behind[1] + g[2] * Behind[2] + gT * BehindT);  // Eq.6
          for (int c = 0; c < 3; ++c) Behind[c] = p[c] + p[3] * Behind[c];
          BehindT *= p[3];
        }
      }
  }
}

// ---------------------------------------------------------------------------
// O7 rasteriser backward for one partition.  PAPER.md L184: "the per-Gaussian
// gradient backpropagates through the intermediate partial pixel".  Given
// g_ct = (dL/dC^k, dL/dT^k) per pixel, redo the forward walk keeping the
// contributors, then walk them in reverse:
//   dL/dalpha_i = <gC, T_i c_i - R_i/(1-alpha_i)> - gT * T_fin/(1-alpha_i),
//   R_i = sum_{j>i} alpha_j T_j c_j,   dL/dc_i += alpha_i T_i gC,
// and chain alpha = min(alpha_max, o*G), G = exp(power), through o, the conic
// and the 2-D mean.  A clamped alpha passes no gradient (true derivative of
// the min; reading s15).  Outputs are ACCUMULATED (+=): g_means2d[n,2],
// g_conic[n,3] (A, B, C), g_opacity[n], g_rgb[n,3].
// ---------------------------------------------------------------------------
void orc_raster_bwd(const double* means2d, const double* conic_opacity, const double* rgb,
                    const uint32_t* vals, const uint32_t* ranges, int W, int H, const double* cfg_,
                    const int32_t* tile_list, int64_t n_tiles, const double* g_ct,
                    double* g_means2d, double* g_conic, double* g_opacity, double* g_rgb) {
  const Cfg cfg = load_cfg(cfg_);
  const int TX = tiles_x(W), TY = tiles_y(H);
  const int64_t nt = tile_list ? n_tiles : (int64_t)TX * TY;
  struct Contrib { uint32_t g; double alpha, T, G, dx, dy; bool clamped; };
  std::vector<Contrib> list;
  for (int64_t it = 0; it < nt; ++it) {
    const int t = tile_list ? tile_list[it] : (int)it;
    const int ty = t / TX, tx = t % TX;
    const uint32_t r0 = ranges[2 * t], r1 = ranges[2 * t + 1];
    for (int j = ty * TILE; j < std::min(H, (ty + 1) * TILE); ++j)
      for (int i = tx * TILE; i < std::min(W, (tx + 1) * TILE); ++i) {
        const int64_t pix = (int64_t)j * W + i;
        const double px = i + 0.5, py = j + 0.5;
        list.clear();
        double T = 1;
        for (uint32_t pos = r0; pos < r1; ++pos) {
          const uint32_t g = vals[pos];
          const double dx = means2d[2 * g] - px, dy = means2d[2 * g + 1] - py;
          const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1],
                       Cc = conic_opacity[4 * g + 2], op = conic_opacity[4 * g + 3];
          const double power = -0.5 * (A * dx * dx + Cc * dy * dy) - B * dx * dy;
          if (power > 0) continue;
          const double G = std::exp(power);
          const bool clamped = op * G >= cfg.alpha_max;
          const double alpha = clamped ? cfg.alpha_max : op * G;
          if (alpha < cfg.alpha_min) continue;
          const double Tn = T * (1 - alpha);
          if (Tn < cfg.T_eps) break;
          list.push_back(Contrib{g, alpha, T, G, dx, dy, clamped});
          T = Tn;
        }
        const double T_fin = T;
        const double* gC = g_ct + 4 * pix;
        const double gT = gC[3];
        double Rs[3] = {0, 0, 0};  // suffix colour sum_{j>i} w_j c_j
        for (size_t k = list.size(); k-- > 0;) {
          const Contrib& cb = list[k];
          const uint32_t g = cb.g;
          const double w = cb.alpha * cb.T;
          double dL_dalpha = 0;
          for (int c = 0; c < 3; ++c) {
            dL_dalpha += gC[c] * (cb.T * rgb[3 * g + c] - Rs[c] / (1 - cb.alpha));
            g_rgb[3 * g + c] += w * gC[c];
          }
          dL_dalpha -= gT * T_fin / (1 - cb.alpha);
          for (int c = 0; c < 3; ++c) Rs[c] += w * rgb[3 * g + c];
          if (cb.clamped) continue;
          const double A = conic_opacity[4 * g], B = conic_opacity[4 * g + 1],
                       Cc = conic_opacity[4 * g + 2], op = conic_opacity[4 * g + 3];
          g_opacity[g] += cb.G * dL_dalpha;
          const double dL_dpower = op * cb.G * dL_dalpha;
          g_means2d[2 * g] += dL_dpower * (-A * cb.dx - B * cb.dy);
          g_means2d[2 * g + 1] += dL_dpower * (-Cc * cb.dy - B * cb.dx);
          g_conic[3 * g] += -0.5 * cb.dx * cb.dx * dL_dpower;
          g_conic[3 * g + 1] += -cb.dx * cb.dy * dL_dpower;
          g_conic[3 * g + 2] += -0.5 * cb.dy * cb.dy * dL_dpower;
        }
      }
  }
}

// ---------------------------------------------------------------------------
// O8 projection backward: the exact derivative of orc_project wherever it is
// differentiable (the loss is "backpropagated ... to update all
// Gaussian parameters").  Inputs are the 2-D gradients of O7; a Gaussian with
// radius == 0 (culled in the forward) receives nothing.  Outputs ACCUMULATE
// into g_mean[n,3], g_log_scale[n,3], g_quat[n,4], g_opacity_logit[n],
// g_sh[n,16,3].  Pinned by central finite differences and by fp64 autograd
// on a dense restatement (tests/test_oracle_grad.py).
// ---------------------------------------------------------------------------
void orc_project_bwd(int64_t n, const double* mean, const double* log_scale, const double* quat,
                     const double* opacity_logit, const double* sh, int sh_degree,
                     const double* cam_, const double* cfg_, const int32_t* radius,
                     const uint8_t* clamp, const double* g_means2d, const double* g_conic,
                     const double* g_opacity, const double* g_rgb, double* g_mean,
                     double* g_log_scale, double* g_quat, double* g_opacity_logit, double* g_sh) {
  const Cam cam = load_cam(cam_);
  const Cfg cfg = load_cfg(cfg_);
  const int nsh = (sh_degree + 1) * (sh_degree + 1);
  double o[3];
  for (int j = 0; j < 3; ++j)
    o[j] = -(cam.R[0 * 3 + j] * cam.t[0] + cam.R[1 * 3 + j] * cam.t[1] + cam.R[2 * 3 + j] * cam.t[2]);
  for (int64_t i = 0; i < n; ++i) {
    if (radius[i] <= 0) continue;
    const double* mu = mean + 3 * i;
    // ---- recompute the forward intermediates ----
    double p[3];
    for (int r = 0; r < 3; ++r)
      p[r] = cam.R[3 * r] * mu[0] + cam.R[3 * r + 1] * mu[1] + cam.R[3 * r + 2] * mu[2] + cam.t[r];
    const double z = p[2];
    double s[3] = {std::exp(log_scale[3 * i]), std::exp(log_scale[3 * i + 1]),
                   std::exp(log_scale[3 * i + 2])};
    const double* q = quat + 4 * i;
    const double qn = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    const double qh[4] = {q[0] / qn, q[1] / qn, q[2] / qn, q[3] / qn};
    double Rot[9]; quat_to_rot(qh, Rot);
    double Mm[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) Mm[3 * r + c] = Rot[3 * r + c] * s[c];
    double Sig[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += Mm[3 * r + k] * Mm[3 * c + k];
      Sig[3 * r + c] = a;
    }
    const double limx = cfg.lim_factor * cam.W / (2.0 * cam.fx);
    const double limy = cfg.lim_factor * cam.H / (2.0 * cam.fy);
    const double xz = p[0] / z, yz = p[1] / z;
    const bool clx = (xz < -limx) || (xz > limx), cly = (yz < -limy) || (yz > limy);
    const double Lx = std::min(limx, std::max(-limx, xz)), Ly = std::min(limy, std::max(-limy, yz));
    const double tx = Lx * z, ty = Ly * z;
    const double J[6] = {cam.fx / z, 0, -cam.fx * tx / (z * z), 0, cam.fy / z, -cam.fy * ty / (z * z)};
    double Tm[6];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += J[3 * r + k] * cam.R[3 * k + c];
      Tm[3 * r + c] = a;
    }
    double TS[6];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += Tm[3 * r + k] * Sig[3 * k + c];
      TS[3 * r + c] = a;
    }
    const double ca = TS[0] * Tm[0] + TS[1] * Tm[1] + TS[2] * Tm[2] + cfg.dilation;
    const double cb = TS[0] * Tm[3] + TS[1] * Tm[4] + TS[2] * Tm[5];
    const double cc = TS[3] * Tm[3] + TS[4] * Tm[4] + TS[5] * Tm[5] + cfg.dilation;
    const double det = ca * cc - cb * cb;
    const double A = cc / det, B = -cb / det, C = ca / det;  // conic Q = P^-1

    // ---- opacity: sigmoid ----
    const double op = 1.0 / (1.0 + std::exp(-opacity_logit[i]));
    g_opacity_logit[i] += op * (1 - op) * g_opacity[i];

    // ---- colour: SH and view direction ----
    double dp[3] = {0, 0, 0};   // dL/dp (camera-space mean)
    double dmu[3] = {0, 0, 0};  // dL/dmu collected directly in world space
    {
      double dvec[3] = {mu[0] - o[0], mu[1] - o[1], mu[2] - o[2]};
      const double dn = std::sqrt(dvec[0] * dvec[0] + dvec[1] * dvec[1] + dvec[2] * dvec[2]);
      double dir[3] = {dvec[0] / dn, dvec[1] / dn, dvec[2] / dn};
      double Y[16], dY[16][3]; sh_basis(sh_degree, dir, Y, dY);
      double gr[3];
      for (int ch = 0; ch < 3; ++ch) gr[ch] = (clamp[i] >> ch & 1) ? 0.0 : g_rgb[3 * i + ch];
      double gdir[3] = {0, 0, 0};
      for (int l = 0; l < nsh; ++l) {
        double dot = 0;
        for (int ch = 0; ch < 3; ++ch) {
          g_sh[(i * 16 + l) * 3 + ch] += Y[l] * gr[ch];
          dot += sh[(i * 16 + l) * 3 + ch] * gr[ch];
        }
        for (int k = 0; k < 3; ++k) gdir[k] += dY[l][k] * dot;
      }
      // dir = dvec/|dvec|:  d dir/d dvec = (I - dir dir^T)/|dvec|
      const double dd = dir[0] * gdir[0] + dir[1] * gdir[1] + dir[2] * gdir[2];
      for (int k = 0; k < 3; ++k) dmu[k] += (gdir[k] - dir[k] * dd) / dn;
    }

    // ---- conic -> cov2d:  Q = P^-1,  dL/dP = -Q Gm Q ----
    const double gA = g_conic[3 * i], gB = g_conic[3 * i + 1], gCc = g_conic[3 * i + 2];
    const double Gm[4] = {gA, 0.5 * gB, 0.5 * gB, gCc};
    const double Q[4] = {A, B, B, C};
    double QG[4], dP[4];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 2; ++c)
      QG[2 * r + c] = Q[2 * r] * Gm[c] + Q[2 * r + 1] * Gm[2 + c];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 2; ++c)
      dP[2 * r + c] = -(QG[2 * r] * Q[c] + QG[2 * r + 1] * Q[2 + c]);
    const double Gc[4] = {dP[0], dP[1], dP[2], dP[3]};  // symmetric; gb/2 on the off-diagonals

    // ---- cov2d = Tm Sigma Tm^T:  dL/dSigma = Tm^T Gc Tm,  dL/dTm = 2 Gc Tm Sigma ----
    double GT[6];  // Gc * Tm (2x3)
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c)
      GT[3 * r + c] = Gc[2 * r] * Tm[c] + Gc[2 * r + 1] * Tm[3 + c];
    double dSig[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c)
      dSig[3 * r + c] = Tm[r] * GT[c] + Tm[3 + r] * GT[3 + c];
    double dTm[6];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += GT[3 * r + k] * Sig[3 * k + c];
      dTm[3 * r + c] = 2 * a;
    }
    // Tm = J W:  dL/dJ = dL/dTm W^T
    double dJ[6];
    for (int r = 0; r < 2; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += dTm[3 * r + k] * cam.R[3 * c + k];
      dJ[3 * r + c] = a;
    }
    // J entries as functions of p (clamped components follow the clamp's true derivative)
    const double z2 = z * z, z3 = z2 * z;
    dp[2] += dJ[0] * (-cam.fx / z2) + dJ[4] * (-cam.fy / z2);
    if (!clx) { dp[0] += dJ[2] * (-cam.fx / z2); dp[2] += dJ[2] * (2 * cam.fx * p[0] / z3); }
    else      { dp[2] += dJ[2] * (cam.fx * Lx / z2); }
    if (!cly) { dp[1] += dJ[5] * (-cam.fy / z2); dp[2] += dJ[5] * (2 * cam.fy * p[1] / z3); }
    else      { dp[2] += dJ[5] * (cam.fy * Ly / z2); }
    // 2-D mean: u = fx x/z + cx, v = fy y/z + cy
    const double gu = g_means2d[2 * i], gv = g_means2d[2 * i + 1];
    dp[0] += cam.fx / z * gu;
    dp[1] += cam.fy / z * gv;
    dp[2] += -cam.fx * p[0] / z2 * gu - cam.fy * p[1] / z2 * gv;
    // p = W mu + t
    for (int k = 0; k < 3; ++k)
      dmu[k] += cam.R[k] * dp[0] + cam.R[3 + k] * dp[1] + cam.R[6 + k] * dp[2];
    for (int k = 0; k < 3; ++k) g_mean[3 * i + k] += dmu[k];

    // ---- Sigma = Mm Mm^T, Mm = Rot diag(s) ----
    double dMm[9];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) {
      double a = 0; for (int k = 0; k < 3; ++k) a += (dSig[3 * r + k] + dSig[3 * k + r]) * Mm[3 * k + c];
      dMm[3 * r + c] = a;
    }
    double dRot[9];
    for (int c = 0; c < 3; ++c) {
      double ds = 0;
      for (int r = 0; r < 3; ++r) { ds += Rot[3 * r + c] * dMm[3 * r + c]; dRot[3 * r + c] = s[c] * dMm[3 * r + c]; }
      g_log_scale[3 * i + c] += s[c] * ds;
    }
    // Rot(q_hat): polynomial derivative, then through the normalisation
    const double w = qh[0], x = qh[1], y = qh[2], zq = qh[3];
    const double dRw[9] = {0, -2 * zq, 2 * y, 2 * zq, 0, -2 * x, -2 * y, 2 * x, 0};
    const double dRx[9] = {0, 2 * y, 2 * zq, 2 * y, -4 * x, -2 * w, 2 * zq, 2 * w, -4 * x};
    const double dRy[9] = {-4 * y, 2 * x, 2 * w, 2 * x, 0, 2 * zq, -2 * w, 2 * zq, -4 * y};
    const double dRz[9] = {-4 * zq, -2 * w, 2 * x, 2 * w, -4 * zq, 2 * y, 2 * x, 2 * y, 0};
    double gq[4] = {0, 0, 0, 0};
    for (int k = 0; k < 9; ++k) {
      gq[0] += dRot[k] * dRw[k]; gq[1] += dRot[k] * dRx[k];
      gq[2] += dRot[k] * dRy[k]; gq[3] += dRot[k] * dRz[k];
    }
    const double qd = qh[0] * gq[0] + qh[1] * gq[1] + qh[2] * gq[2] + qh[3] * gq[3];
    for (int k = 0; k < 4; ++k) g_quat[4 * i + k] += (gq[k] - qh[k] * qd) / qn;
  }
}

// ---------------------------------------------------------------------------
// O5 loss (harness step a7).  PAPER.md L95: L = L_RGB + lambda L_D-SSIM; only
// the RGB term, as a mean L1 (reading s17).  Returns L; g_image = sign/(3HW).
// ---------------------------------------------------------------------------
double orc_l1(int64_t count, const double* image, const double* target, double* g_image) {
  double L = 0;
  for (int64_t i = 0; i < count; ++i) {
    const double dlt = image[i] - target[i];
    L += std::fabs(dlt);
    if (g_image) g_image[i] = (dlt > 0 ? 1.0 : (dlt < 0 ? -1.0 : 0.0)) / (double)count;
  }
  return L / (double)count;
}

// ---------------------------------------------------------------------------
// O9 Adam (reading s18): m = b1 m + (1-b1) g;  v = b2 v + (1-b2) g^2;
// p -= lr * (m/(1-b1^t)) / (sqrt(v/(1-b2^t)) + eps).  Dense; step is 1-based.
// ---------------------------------------------------------------------------
void orc_adam(int64_t count, double* param, const double* grad, double* m, double* v, double lr,
              double beta1, double beta2, double eps, int step) {
  const double bc1 = 1.0 - std::pow(beta1, step), bc2 = 1.0 - std::pow(beta2, step);
  for (int64_t i = 0; i < count; ++i) {
    m[i] = beta1 * m[i] + (1 - beta1) * grad[i];
    v[i] = beta2 * v[i] + (1 - beta2) * grad[i] * grad[i];
    param[i] -= lr * (m[i] / bc1) / (std::sqrt(v[i] / bc2) + eps);
  }
}

// SH basis exposed for the quadrature pin.
void orc_sh_basis(int deg, const double* dir, double* Y) {
  double dY[16][3]; sh_basis(deg, dir, Y, dY);
}

}  // extern "C"
