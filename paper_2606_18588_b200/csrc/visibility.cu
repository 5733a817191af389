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
#include <cmath>
#include <vector>

#include "common.cuh"

namespace {

struct P2 { double x, y; };
struct P3 { double x, y, z; };

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

// ---- conservative regions (reading s21) -------------------------------------------------------------------------
// Gaussians belong to a partition by their mean (L155) but their footprints stick out of its box (L474), and the
// binning keeps every Gaussian whose square of tiles meets the image (s8, s11).  For a Gaussian with scale <= s and
// camera-space mean (x, y, z), z > near:
//   radius = ceil(3 sqrt(lambda)),  lambda = mid + sqrt(max(floor, mid^2 - det)) <= lambda_max(Sigma2D) + sqrt(floor),
//   Sigma2D = J W Sigma W^T J^T + dilation I (L80, s9)  =>  lambda_max <= |J|_2^2 s^2 + dilation,
//   |J|_2^2 <= c^2 / z^2,  c^2 = max(fx, fy)^2 (1 + limx^2 + limy^2)   (J J^T has eigenvalues f^2/z^2 and f^2 (1 + Lx^2 +
//   Ly^2)/z^2 for fx = fy = f; |Lx| <= limx, |Ly| <= limy are the clamps of s9),
// so radius <= 3 c s / z + 3 sqrt(e) + 1 with e = dilation + sqrt(floor).  Its square of tiles covers the pixel columns
// within radius + 1.5 of u = fx x / z + cx (pixel centres at +0.5, one pixel of rounding); it can meet the image
// [0, W] only if  -(cx + g) z - h <= fx x <= (W - cx + g) z + h,  g = 2.5 + 3 sqrt(e),  h = 3 c s  -- LINEAR in (x, z),
// likewise in (y, z).  Hence only means inside the convex polyhedron  Q = box ^ {z >= near} ^ {those four half spaces}
// matter; on Q the radius is at most  m - 2.5,  m = 3 sqrt(c^2 s^2 / z_min(Q)^2 + e) + 3.5, and every tile such a
// Gaussian is binned to lies within m pixels of the projection of Q.  A slot outside that region has an EMPTY list.
struct Plane { double n[3], d; };     // inside: n . p + d >= 0   (camera space)

// vertices of the bounded convex polyhedron { p : all planes >= 0 }: every triple of planes that meets in one point
// satisfying the others (11 planes: 165 triples; host, double).  Slightly outside points are accepted: conservative.
static void polytope_vertices(const std::vector<Plane>& pl, std::vector<P3>& out) {
  out.clear();
  const size_t n = pl.size();
  for (size_t i = 0; i < n; ++i)
    for (size_t j = i + 1; j < n; ++j)
      for (size_t k = j + 1; k < n; ++k) {
        const double* a = pl[i].n; const double* b = pl[j].n; const double* c = pl[k].n;
        const double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
        const double det = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
        const double na = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]), nb = std::sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]),
                     nc = std::sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
        if (std::fabs(det) <= 1e-10 * na * nb * nc) continue;           // (nearly) parallel planes
        const double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
        const double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        double p[3];
        for (int r = 0; r < 3; ++r) p[r] = -(pl[i].d * bc[r] + pl[j].d * ca[r] + pl[k].d * ab[r]) / det;
        const double scale = 1.0 + std::fabs(p[0]) + std::fabs(p[1]) + std::fabs(p[2]);
        bool inside = true;
        for (size_t q = 0; q < n && inside; ++q) {
          const double nn = std::sqrt(pl[q].n[0] * pl[q].n[0] + pl[q].n[1] * pl[q].n[1] + pl[q].n[2] * pl[q].n[2]);
          inside = pl[q].n[0] * p[0] + pl[q].n[1] * p[1] + pl[q].n[2] * p[2] + pl[q].d >= -1e-9 * nn * scale;
        }
        if (inside) out.push_back(P3{p[0], p[1], p[2]});
      }
}

int splx_visible_regions(int K, int n_boxes, const int32_t* box_part, const float* aabb_lo, const float* aabb_hi,
                         const float* max_scale, const splx_config* cfg, const splx_camera* cam, uint8_t* tile_state,
                         uint64_t* participants) {
  if (K < 1 || K > SPLX_MAX_K || n_boxes < 0 || (!box_part && n_boxes != K) || !aabb_lo || !aabb_hi || !cam || !tile_state)
    return SPLX_ERR_INVALID_ARG;
  if (cam->width <= 0 || cam->height <= 0 || !(cam->fx > 0.f) || !(cam->fy > 0.f) || !(cam->near_z > 0.f)) return SPLX_ERR_INVALID_ARG;
  const int W = cam->width, H = cam->height;
  const int TX = (W + SPLX_TILE - 1) / SPLX_TILE, TY = (H + SPLX_TILE - 1) / SPLX_TILE;
  const size_t ntiles = (size_t)TX * TY;
  const double fx = cam->fx, fy = cam->fy, cx = cam->cx, cy = cam->cy, near_z = cam->near_z;
  const double lim_factor = cfg ? cfg->lim_factor : 1.3, dilation = cfg ? cfg->dilation : 0.3, rfloor = cfg ? cfg->radius_floor : 0.1;
  const double limx = lim_factor * W / (2.0 * fx), limy = lim_factor * H / (2.0 * fy);
  const double c2 = std::max(fx, fy) * std::max(fx, fy) * (1.0 + limx * limx + limy * limy);
  const double e = dilation + std::sqrt(rfloor), g = 2.5 + 3.0 * std::sqrt(e);
  uint64_t part = 0;
  std::fill(tile_state, tile_state + (size_t)K * ntiles, (uint8_t)SPLX_TILE_INVISIBLE);
  std::vector<Plane> planes;
  std::vector<P3> verts;
  for (int j = 0; j < n_boxes; ++j) {
    const int k = box_part ? box_part[j] : j;
    if (k < 0 || k >= K) return SPLX_ERR_INVALID_ARG;
    const float* lo = aabb_lo + 3 * j;
    const float* hi = aabb_hi + 3 * j;
    uint8_t* st = tile_state + (size_t)k * ntiles;
    for (int a = 0; a < 3; ++a) if (!(lo[a] <= hi[a])) return SPLX_ERR_INVALID_ARG;
    if (max_scale && !(max_scale[j] >= 0.f)) return SPLX_ERR_INVALID_ARG;
    planes.clear();
    // the box, in camera space: world = R^T (p - t), so world_a = col_a(R) . p - col_a(R) . t
    for (int a = 0; a < 3; ++a) {
      const double n[3] = {cam->R[a], cam->R[3 + a], cam->R[6 + a]};
      const double nt = n[0] * cam->t[0] + n[1] * cam->t[1] + n[2] * cam->t[2];
      planes.push_back(Plane{{n[0], n[1], n[2]}, -nt - (double)lo[a]});
      planes.push_back(Plane{{-n[0], -n[1], -n[2]}, nt + (double)hi[a]});
    }
    planes.push_back(Plane{{0.0, 0.0, 1.0}, -near_z});
    double s = 0.0;
    if (max_scale) {       // the half spaces outside which no Gaussian of this box can reach the image
      s = max_scale[j];
      const double h = 3.0 * std::sqrt(c2) * s;
      planes.push_back(Plane{{-fx, 0.0, (double)W - cx + g}, h});
      planes.push_back(Plane{{fx, 0.0, cx + g}, h});
      planes.push_back(Plane{{0.0, -fy, (double)H - cy + g}, h});
      planes.push_back(Plane{{0.0, fy, cy + g}, h});
    }
    polytope_vertices(planes, verts);
    if (verts.empty()) continue;   // behind the near plane, or (conservative mode) out of reach of the image
    double zmin = 1e300;
    std::vector<P2> pts;
    for (const P3& p : verts) {
      const double z = std::max(p.z, near_z);
      zmin = std::min(zmin, z);
      pts.push_back(P2{fx * p.x / z + cx, fy * p.y / z + cy});
    }
    const std::vector<P2> hull = convex_hull(pts);
    const double mg = max_scale ? 3.0 * std::sqrt(c2 * s * s / (zmin * zmin) + e) + 3.5 : 0.0;
    // only the tiles under the hull's bounding rectangle (grown by the margin) can meet it
    double lx = hull[0].x, hx = hull[0].x, ly = hull[0].y, hy = hull[0].y;
    for (const P2& p : hull) { lx = std::min(lx, p.x); hx = std::max(hx, p.x); ly = std::min(ly, p.y); hy = std::max(hy, p.y); }
    if (hx + mg < 0.0 || lx - mg > (double)W || hy + mg < 0.0 || ly - mg > (double)H) continue;
    const int tx0 = std::max(0, (int)std::floor((lx - mg) / 16.0)), tx1 = std::min(TX - 1, (int)std::floor((hx + mg) / 16.0));
    const int ty0 = std::max(0, (int)std::floor((ly - mg) / 16.0)), ty1 = std::min(TY - 1, (int)std::floor((hy + mg) / 16.0));
    bool any = false;
    for (int ty = ty0; ty <= ty1; ++ty)
      for (int tx = tx0; tx <= tx1; ++tx) {
        if (st[(size_t)ty * TX + tx] == 0) { any = true; continue; }      // another box of the partition already reaches it
        const double x0 = 16.0 * tx - mg, x1 = std::min(16.0 * (tx + 1), (double)W) + mg;
        const double y0 = 16.0 * ty - mg, y1 = std::min(16.0 * (ty + 1), (double)H) + mg;
        if (hull_meets_rect(hull, x0, x1, y0, y1)) { st[(size_t)ty * TX + tx] = 0; any = true; }
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
