// visibility.cu -- HOST side of the two optional subsystems: geometric visibility prediction
// ("the camera frustum is a convex polyhedron ... each GPU partition is also convex,
// designed explicitly as an axis-aligned bounding box ... the overlapping volume ... is also a convex
// polyhedron ... Projecting this convex 3D space onto the image plane yields a convex visible region
// ... efficiently determined by projecting only the intersection vertices ... without rendering";
// L227: done "at initialization stage") and conflict-free view consolidation (L249, greedy
// bucketing over GetParticipants(v)).  Both are small, static, per-view host computations in the
// paper as well; the device consumes their result as the per-(partition, tile) state bytes of
// splx_plan.  The transmittance half of the prediction (L231) runs on the device: compose.cu.
#include <algorithm>
#include <vector>

#include "common.cuh"

namespace {

struct P2 { double x, y; };
struct P3 { double x, y, z; };

// Keep the part of a convex polygon with z >= zmin (Sutherland-Hodgman against one plane).
void clip_near(const std::vector<P3>& in, double zmin, std::vector<P3>& out) {
  out.clear();
  const size_t n = in.size();
  for (size_t i = 0; i < n; ++i) {
    const P3& a = in[i];
    const P3& b = in[(i + 1) % n];
    const bool ia = a.z >= zmin, ib = b.z >= zmin;
    if (ia) out.push_back(a);
    if (ia != ib) {
      const double s = (zmin - a.z) / (b.z - a.z);
      out.push_back(P3{a.x + s * (b.x - a.x), a.y + s * (b.y - a.y), zmin});
    }
  }
}

double cross(const P2& o, const P2& a, const P2& b) { return (a.x - o.x) * (b.y - o.y) - (a.y - o.y) * (b.x - o.x); }

// Andrew's monotone chain; returns the hull counter-clockwise without repeated end point
// (1 point, 2 points for degenerate inputs).
std::vector<P2> convex_hull(std::vector<P2> pts) {
  std::sort(pts.begin(), pts.end(), [](const P2& a, const P2& b) { return a.x < b.x || (a.x == b.x && a.y < b.y); });
  pts.erase(std::unique(pts.begin(), pts.end(), [](const P2& a, const P2& b) { return a.x == b.x && a.y == b.y; }), pts.end());
  const size_t n = pts.size();
  if (n < 3) return pts;
  std::vector<P2> h(2 * n);
  size_t k = 0;
  for (size_t i = 0; i < n; ++i) {
    while (k >= 2 && cross(h[k - 2], h[k - 1], pts[i]) <= 0) --k;
    h[k++] = pts[i];
  }
  for (size_t i = n - 1, t = k + 1; i-- > 0;) {
    while (k >= t && cross(h[k - 2], h[k - 1], pts[i]) <= 0) --k;
    h[k++] = pts[i];
  }
  h.resize(k - 1);
  return h;
}

// Closed convex polygon (>= 1 vertex) against the closed rectangle [x0,x1] x [y0,y1]: separating axes =
// the rectangle's two axes and the normals of the polygon's edges.
bool hull_meets_rect(const std::vector<P2>& h, double x0, double x1, double y0, double y1) {
  double lx = h[0].x, hx = h[0].x, ly = h[0].y, hy = h[0].y;
  for (const P2& p : h) { lx = std::min(lx, p.x); hx = std::max(hx, p.x); ly = std::min(ly, p.y); hy = std::max(hy, p.y); }
  if (hx < x0 || lx > x1 || hy < y0 || ly > y1) return false;
  const size_t n = h.size();
  if (n < 2) return true;
  const P2 rc[4] = {{x0, y0}, {x1, y0}, {x1, y1}, {x0, y1}};
  for (size_t i = 0; i < n; ++i) {
    const P2& a = h[i];
    const P2& b = h[(i + 1) % n];
    const double nx = b.y - a.y, ny = -(b.x - a.x);      // a normal of edge a->b
    double pl = 1e300, ph = -1e300, rl = 1e300, rh = -1e300;
    for (const P2& p : h) { const double s = nx * p.x + ny * p.y; pl = std::min(pl, s); ph = std::max(ph, s); }
    for (const P2& p : rc) { const double s = nx * p.x + ny * p.y; rl = std::min(rl, s); rh = std::max(rh, s); }
    if (ph < rl || rh < pl) return false;
    if (n == 2) break;                                    // a segment has one edge
  }
  return true;
}

}  // namespace

extern "C" {

int splx_visible_regions(int K, const float* aabb_lo, const float* aabb_hi, const splx_camera* cam,
                         uint8_t* tile_state, uint64_t* participants) {
  if (K < 1 || K > SPLX_MAX_K || !aabb_lo || !aabb_hi || !cam || !tile_state) return SPLX_ERR_INVALID_ARG;
  if (cam->width <= 0 || cam->height <= 0 || !(cam->fx > 0.f) || !(cam->fy > 0.f)) return SPLX_ERR_INVALID_ARG;
  const int W = cam->width, H = cam->height;
  const int TX = (W + SPLX_TILE - 1) / SPLX_TILE, TY = (H + SPLX_TILE - 1) / SPLX_TILE;
  const size_t ntiles = (size_t)TX * TY;
  uint64_t part = 0;
  // faces of the box as corner-index quads (corner c: bit 0 -> x, bit 1 -> y, bit 2 -> z taken from hi)
  static const int face[6][4] = {{0, 2, 6, 4}, {1, 3, 7, 5}, {0, 1, 5, 4}, {2, 3, 7, 6}, {0, 1, 3, 2}, {4, 5, 7, 6}};
  std::vector<P3> poly, clipped;
  for (int k = 0; k < K; ++k) {
    const float* lo = aabb_lo + 3 * k;
    const float* hi = aabb_hi + 3 * k;
    uint8_t* st = tile_state + (size_t)k * ntiles;
    for (int a = 0; a < 3; ++a) if (!(lo[a] <= hi[a])) return SPLX_ERR_INVALID_ARG;
    P3 c[8];
    for (int i = 0; i < 8; ++i) {
      const double w[3] = {(i & 1) ? hi[0] : lo[0], (i & 2) ? hi[1] : lo[1], (i & 4) ? hi[2] : lo[2]};
      double p[3];
      for (int r = 0; r < 3; ++r)
        p[r] = (double)cam->R[3 * r] * w[0] + (double)cam->R[3 * r + 1] * w[1] + (double)cam->R[3 * r + 2] * w[2] + (double)cam->t[r];
      c[i] = P3{p[0], p[1], p[2]};
    }
    std::vector<P2> pts;
    for (int f = 0; f < 6; ++f) {
      poly.assign({c[face[f][0]], c[face[f][1]], c[face[f][2]], c[face[f][3]]});
      clip_near(poly, (double)cam->near_z, clipped);
      for (const P3& p : clipped) pts.push_back(P2{(double)cam->fx * p.x / p.z + (double)cam->cx, (double)cam->fy * p.y / p.z + (double)cam->cy});
    }
    if (pts.empty()) {   // the box lies behind the near plane
      std::fill(st, st + ntiles, (uint8_t)SPLX_TILE_INVISIBLE);
      continue;
    }
    const std::vector<P2> hull = convex_hull(pts);
    bool any = false;
    for (int ty = 0; ty < TY; ++ty)
      for (int tx = 0; tx < TX; ++tx) {
        const double x0 = 16.0 * tx, x1 = std::min(16.0 * (tx + 1), (double)W);
        const double y0 = 16.0 * ty, y1 = std::min(16.0 * (ty + 1), (double)H);
        const bool vis = hull_meets_rect(hull, x0, x1, y0, y1);
        st[(size_t)ty * TX + tx] = vis ? 0 : SPLX_TILE_INVISIBLE;
        any |= vis;
      }
    if (any) part |= 1ull << k;
  }
  if (participants) *participants = part;
  return SPLX_OK;
}

int splx_schedule_views(int n_views, const uint64_t* participants, int max_views_per_bucket, int32_t* bucket_of_view,
                        int32_t* n_buckets) {
  if (n_views < 0 || (n_views > 0 && (!participants || !bucket_of_view)) || !n_buckets || max_views_per_bucket < 1 ||
      max_views_per_bucket > SPLX_MAX_VIEWS)
    return SPLX_ERR_INVALID_ARG;
  std::vector<uint64_t> used;     // partitions already claimed by each bucket
  std::vector<int> count;
  for (int v = 0; v < n_views; ++v) {
    int b = -1;
    for (size_t j = 0; j < used.size(); ++j)
      if ((used[j] & participants[v]) == 0 && count[j] < max_views_per_bucket) { b = (int)j; break; }
    if (b < 0) { used.push_back(0); count.push_back(0); b = (int)used.size() - 1; }
    used[b] |= participants[v];
    count[b] += 1;
    bucket_of_view[v] = b;
  }
  *n_buckets = (int32_t)used.size();
  return SPLX_OK;
}

}  // extern "C"
