// cross.cu -- cross-boundary per-ray filtering, the parts outside the binning (appendix 8.1,
// Fig. 25; readings DESIGN.md s32): "let Q_cross denote the set of Gaussians whose spatial support spans both
// partitions" -> k_cross_sets (device, view independent); "the overlapped depth interval D_overlap" ->
// splx_cross_depth_ranges (host, per plan).  The removal itself happens where the lists are made: sort.cu.
#include <algorithm>
#include <cmath>
#include <limits>

#include "common.cuh"

namespace {

struct CellBoxes { float lo[SPLX_MAX_K][3], hi[SPLX_MAX_K][3]; };
struct CrossRuns { int K; int64_t off[SPLX_MAX_K + 1]; };

// One thread per Gaussian: 40 B in, 8 B out -- a plain streaming kernel (bound by HBM; a fraction of a
// projection pass, and run only when the Gaussians change, not per view).
__global__ void __launch_bounds__(256)
k_cross_sets(const float* __restrict__ mean, const float* __restrict__ log_scale, const float* __restrict__ quat, int64_t n,
             const __grid_constant__ CrossRuns runs, const __grid_constant__ CellBoxes boxes, float sigma,
             uint64_t* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int k = 0;                                      // partition of Gaussian i: last k with off[k] <= i
  {
    int lo = 0, hi = runs.K - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (runs.off[mid] <= i) lo = mid; else hi = mid - 1;
    }
    k = lo;
  }
  const float mx = mean[3 * i], my = mean[3 * i + 1], mz = mean[3 * i + 2];
  const float sx = expf(log_scale[3 * i]), sy = expf(log_scale[3 * i + 1]), sz = expf(log_scale[3 * i + 2]);
  const float4 q = *reinterpret_cast<const float4*>(quat + 4 * i);
  const float qn = rsqrtf(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
  const float w = q.x * qn, x = q.y * qn, y = q.z * qn, z = q.w * qn;
  const float r00 = 1.f - 2.f * (y * y + z * z), r01 = 2.f * (x * y - w * z), r02 = 2.f * (x * z + w * y);
  const float r10 = 2.f * (x * y + w * z), r11 = 1.f - 2.f * (x * x + z * z), r12 = 2.f * (y * z - w * x);
  const float r20 = 2.f * (x * z - w * y), r21 = 2.f * (y * z + w * x), r22 = 1.f - 2.f * (x * x + y * y);
  const float s2x = sx * sx, s2y = sy * sy, s2z = sz * sz;
  // Sigma_aa = sum_j R_aj^2 s_j^2
  const float hx = sigma * sqrtf(r00 * r00 * s2x + r01 * r01 * s2y + r02 * r02 * s2z);
  const float hy = sigma * sqrtf(r10 * r10 * s2x + r11 * r11 * s2y + r12 * r12 * s2z);
  const float hz = sigma * sqrtf(r20 * r20 * s2x + r21 * r21 * s2y + r22 * r22 * s2z);
  uint64_t m = 0;
  for (int s = 0; s < runs.K; ++s) {
    if (s == k) continue;
    const bool meet = mx - hx <= boxes.hi[s][0] && mx + hx >= boxes.lo[s][0] && my - hy <= boxes.hi[s][1] &&
                      my + hy >= boxes.lo[s][1] && mz - hz <= boxes.hi[s][2] && mz + hz >= boxes.lo[s][2];
    if (meet) m |= 1ull << s;
  }
  out[i] = m;
}

}  // namespace

int launch_cross_sets(splx_ctx* ctx, const splx_gaussians* g, int K, const int64_t* part_offsets, const float* cell_lo,
                      const float* cell_hi, float support_sigma, uint64_t* cross_mask) {
  if (g->n == 0) return SPLX_OK;
  CrossRuns runs;
  CellBoxes boxes;
  memset(&runs, 0, sizeof runs);
  memset(&boxes, 0, sizeof boxes);
  runs.K = K;
  for (int k = 0; k <= K; ++k) runs.off[k] = part_offsets[k];
  for (int k = 0; k < K; ++k)
    for (int a = 0; a < 3; ++a) { boxes.lo[k][a] = cell_lo[3 * k + a]; boxes.hi[k][a] = cell_hi[3 * k + a]; }
  const int64_t blocks = (g->n + 255) / 256;
  k_cross_sets<<<(unsigned)blocks, 256, 0, ctx->stream>>>(g->mean, g->log_scale, g->quat, g->n, runs, boxes, support_sigma,
                                                          cross_mask);
  SPLX_LAUNCH_CHECK(ctx, "k_cross_sets");
  return SPLX_OK;
}

extern "C" int splx_cross_depth_ranges(int K, const float* aabb_lo, const float* aabb_hi, const splx_plan* plan,
                                       float* part_depth_range) {
  if (K < 1 || K > SPLX_MAX_K || !aabb_lo || !aabb_hi || !plan || !plan->cams || !plan->view_of_part || !part_depth_range ||
      plan->n_views < 1 || plan->n_views > SPLX_MAX_VIEWS)
    return SPLX_ERR_INVALID_ARG;
  for (int k = 0; k < K; ++k) {
    const int v = plan->view_of_part[k];
    if (v < -1 || v >= plan->n_views) return SPLX_ERR_INVALID_ARG;
    if (v < 0) {
      part_depth_range[2 * k] = std::numeric_limits<float>::infinity();
      part_depth_range[2 * k + 1] = -std::numeric_limits<float>::infinity();
      continue;
    }
    const splx_camera& c = plan->cams[v];
    double zmin = 1e300, zmax = -1e300;
    for (int i = 0; i < 8; ++i) {
      const double wx = (i & 1) ? aabb_hi[3 * k] : aabb_lo[3 * k], wy = (i & 2) ? aabb_hi[3 * k + 1] : aabb_lo[3 * k + 1],
                   wz = (i & 4) ? aabb_hi[3 * k + 2] : aabb_lo[3 * k + 2];
      const double z = (double)c.R[6] * wx + (double)c.R[7] * wy + (double)c.R[8] * wz + (double)c.t[2];
      zmin = std::min(zmin, z); zmax = std::max(zmax, z);
    }
    part_depth_range[2 * k] = (float)zmin;
    part_depth_range[2 * k + 1] = (float)zmax;
  }
  return SPLX_OK;
}
