// project.cu -- step a1 (projection) and step a10 (its exact derivative).
// Sigma = R S S^T R^T.  L80: frustum cull by the mean; Sigma2D = J W Sigma W^T J^T;
// 2-D attributes depth d, 2-D mean, Sigma2D.  Readings: s5 depth = camera z,
// s8 cull rule, s9 dilation / radius / J clamp, s10 pixel centres, s11 tile rect, s13 SH colour,
// s14 parameterisation, s15 true derivative at clamps.
//
// Both kernels are HBM-bound streaming kernels: one thread per Gaussian, 236 B of parameters in
// for a visible Gaussian (44 B for a culled one: the 192 B of SH are only read when visible).
#include "common.cuh"

namespace {

constexpr int PROJ_THREADS = 256;

// Real SH constants (orthonormal basis, Condon-Shortley phase; index l(l+1)+m).
constexpr float kY0 = 0.28209479177387814f;
constexpr float kK1 = 0.4886025119029199f;
constexpr float kK2a = 1.0925484305920792f;
constexpr float kK2b = 0.31539156525252005f;
constexpr float kK2c = 0.5462742152960396f;
constexpr float kK3a = 0.5900435899266435f;
constexpr float kK3b = 2.890611442640554f;
constexpr float kK3c = 0.4570457994644658f;
constexpr float kK3d = 0.3731763325901154f;
constexpr float kK3e = 1.445305721320277f;

struct Geo {  // forward intermediates shared by both directions
  float p[3];
  float s[3], qh[4], qn, Rot[9], Mm[9];
  float Tm[6];    // J * W
  float N[6];     // Tm * Mm  (2x3):  Sigma2D = N N^T + dilation I
  float a, b, c, det;
  float Lx, Ly;   // clamped x/z, y/z used inside J
  bool clx, cly;
};

__device__ __forceinline__ float det2_accurate(float a, float c, float b) {
  // a*c - b*b with one rounding error instead of a cancellation (Kahan's fma scheme)
  const float w = b * b;
  const float e = fmaf(-b, b, w);
  const float f = fmaf(a, c, -w);
  return f + e;
}

// Raw per-Gaussian inputs of the geometry chain, loaded up front so that the loads are independent.
struct GeoIn { float m[3], ls[3]; float4 q; };

__device__ __forceinline__ GeoIn load_geo(const splx_gaussians& g, int64_t i) {
  GeoIn in;
#pragma unroll
  for (int k = 0; k < 3; ++k) { in.m[k] = g.mean[3 * i + k]; in.ls[k] = g.log_scale[3 * i + k]; }
  in.q = *reinterpret_cast<const float4*>(g.quat + 4 * i);
  return in;
}

__device__ __forceinline__ bool geometry(const GeoIn& in, const CamDev& cam, float dilation, Geo& G) {
  const float mx = in.m[0], my = in.m[1], mz = in.m[2];
#pragma unroll
  for (int r = 0; r < 2; ++r)
    G.p[r] = cam.R[3 * r] * mx + cam.R[3 * r + 1] * my + cam.R[3 * r + 2] * mz + cam.t[r];
  // the depth is the sort key (s12): a fixed fp32 operation order, so that two Gaussians whose depths differ by less
  // than a rounding are ordered by every build of this kernel -- and by the oracle -- alike
  G.p[2] = __fadd_rn(__fmaf_rn(cam.R[8], mz, __fmaf_rn(cam.R[7], my, __fmul_rn(cam.R[6], mx))), cam.t[2]);
  if (!(G.p[2] > cam.near_z)) return false;
#pragma unroll
  for (int k = 0; k < 3; ++k) G.s[k] = expf(in.ls[k]);
  const float4 q = in.q;
  G.qn = sqrtf(q.x * q.x + q.y * q.y + q.z * q.z + q.w * q.w);
  const float inv = 1.0f / G.qn;
  const float w = q.x * inv, x = q.y * inv, y = q.z * inv, z = q.w * inv;
  G.qh[0] = w; G.qh[1] = x; G.qh[2] = y; G.qh[3] = z;
  G.Rot[0] = 1.f - 2.f * (y * y + z * z); G.Rot[1] = 2.f * (x * y - w * z); G.Rot[2] = 2.f * (x * z + w * y);
  G.Rot[3] = 2.f * (x * y + w * z); G.Rot[4] = 1.f - 2.f * (x * x + z * z); G.Rot[5] = 2.f * (y * z - w * x);
  G.Rot[6] = 2.f * (x * z - w * y); G.Rot[7] = 2.f * (y * z + w * x); G.Rot[8] = 1.f - 2.f * (x * x + y * y);
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c) G.Mm[3 * r + c] = G.Rot[3 * r + c] * G.s[c];
  const float pz = G.p[2], iz = 1.0f / pz;
  const float xz = G.p[0] * iz, yz = G.p[1] * iz;
  G.clx = (xz < -cam.limx) || (xz > cam.limx);
  G.cly = (yz < -cam.limy) || (yz > cam.limy);
  G.Lx = fminf(cam.limx, fmaxf(-cam.limx, xz));
  G.Ly = fminf(cam.limy, fmaxf(-cam.limy, yz));
  const float j00 = cam.fx * iz, j02 = -cam.fx * G.Lx * iz;  // -fx * (Lx z) / z^2
  const float j11 = cam.fy * iz, j12 = -cam.fy * G.Ly * iz;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    G.Tm[c] = j00 * cam.R[c] + j02 * cam.R[6 + c];
    G.Tm[3 + c] = j11 * cam.R[3 + c] + j12 * cam.R[6 + c];
  }
#pragma unroll
  for (int r = 0; r < 2; ++r)
#pragma unroll
    for (int c = 0; c < 3; ++c)
      G.N[3 * r + c] = G.Tm[3 * r] * G.Mm[c] + G.Tm[3 * r + 1] * G.Mm[3 + c] + G.Tm[3 * r + 2] * G.Mm[6 + c];
  G.a = G.N[0] * G.N[0] + G.N[1] * G.N[1] + G.N[2] * G.N[2] + dilation;
  G.b = G.N[0] * G.N[3] + G.N[1] * G.N[4] + G.N[2] * G.N[5];
  G.c = G.N[3] * G.N[3] + G.N[4] * G.N[4] + G.N[5] * G.N[5] + dilation;
  G.det = det2_accurate(G.a, G.c, G.b);
  return G.det > 0.0f;
}

// Y_l(dir), l < (deg+1)^2
__device__ __forceinline__ void sh_eval(int deg, float x, float y, float z, float* Y) {
  Y[0] = kY0;
  if (deg < 1) return;
  Y[1] = -kK1 * y; Y[2] = kK1 * z; Y[3] = -kK1 * x;
  if (deg < 2) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  Y[4] = kK2a * x * y; Y[5] = -kK2a * y * z; Y[6] = kK2b * (2.f * zz - xx - yy);
  Y[7] = -kK2a * x * z; Y[8] = kK2c * (xx - yy);
  if (deg < 3) return;
  Y[9] = -kK3a * y * (3.f * xx - yy);
  Y[10] = kK3b * x * y * z;
  Y[11] = -kK3c * y * (4.f * zz - xx - yy);
  Y[12] = kK3d * z * (2.f * zz - 3.f * xx - 3.f * yy);
  Y[13] = -kK3c * x * (4.f * zz - xx - yy);
  Y[14] = kK3e * z * (xx - yy);
  Y[15] = -kK3a * x * (xx - 3.f * yy);
}

// Run of the launch this block works on (warp-uniform binary search over <= 64 entries).
__device__ __forceinline__ int find_run(const RunTable& rt, int b) {
  int lo = 0, hi = rt.n - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (rt.block_prefix[mid] <= b) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// Position of chunk q of row `row` inside the row's NV chunks of the staged copy.  Degree 3 (12 chunks = 192 B, no
// padding): XOR with the row so that the row-wise LDS.128 of a quarter warp spreads over the bank groups (chunks 0-7
// conflict-free, chunks 8-11 two-way); smaller rows are left in place.
template <int NV>
__device__ __forceinline__ int sh_swz(int q, int row) {
  if (NV == 12) return q < 8 ? (q ^ (row & 7)) : 8 + ((q - 8) ^ (row & 3));
  return q;
}

// colour: SH along the direction from the camera centre to the mean (s13).  The coefficients come from `sh4`
// (the Gaussian's row in global memory, chunk q at sh4[q]) or, STAGED, from the warp's shared-memory copy of its 32
// rows (chunk q of row `lane` at sh4[lane * NV + sh_swz<NV>(q, lane)]).
template <int DEG, bool STAGED>
__device__ __forceinline__ void colour(const float4* sh4, int lane, const CamDev& cam, const float* m, int64_t i,
                                       const splx_projected& out, float4* bl) {
  float dx = m[0] - cam.o[0], dy = m[1] - cam.o[1], dz = m[2] - cam.o[2];
  const float dinv = rsqrtf(dx * dx + dy * dy + dz * dz);
  dx *= dinv; dy *= dinv; dz *= dinv;
  constexpr int NSH = (DEG + 1) * (DEG + 1);
  float Y[NSH];
  sh_eval(DEG, dx, dy, dz, Y);
  float c[3] = {0.5f, 0.5f, 0.5f};
  constexpr int NV = (NSH * 3 + 3) / 4;
#pragma unroll
  for (int q = 0; q < NV; ++q) {
    const float4 f = STAGED ? sh4[lane * NV + sh_swz<NV>(q, lane)] : __ldg(sh4 + q);
    const float e[4] = {f.x, f.y, f.z, f.w};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int idx = 4 * q + t;
      if (idx < NSH * 3) c[idx % 3] = fmaf(Y[idx / 3], e[t], c[idx % 3]);
    }
  }
  uint8_t cl = 0;
#pragma unroll
  for (int ch = 0; ch < 3; ++ch) {
    if (c[ch] < 0.f) { cl |= (uint8_t)(1u << ch); c[ch] = 0.f; }
    out.rgb[3 * i + ch] = c[ch];
  }
  bl[2] = make_float4(c[0], c[1], c[2], 0.f);
  out.clamp[i] = cl;
}

// Reach test of a mean (reading s21): can a Gaussian of scale <= smax at this mean touch the image at all?  smax < 0:
// no bound is known, every Gaussian goes through the full test.
__device__ __forceinline__ bool reaches(const float* m, const CamDev& cam, float smax) {
  if (!(smax >= 0.f)) return true;
  const float x = cam.R[0] * m[0] + cam.R[1] * m[1] + cam.R[2] * m[2] + cam.t[0];
  const float y = cam.R[3] * m[0] + cam.R[4] * m[1] + cam.R[5] * m[2] + cam.t[1];
  const float z = cam.R[6] * m[0] + cam.R[7] * m[1] + cam.R[8] * m[2] + cam.t[2];
  const float h = 3.0f * cam.reach_c * smax, fxx = cam.fx * x, fyy = cam.fy * y;
  return z > cam.near_z * 0.999f && fxx <= cam.reach_r * z + h && -fxx <= cam.reach_l * z + h &&
         fyy <= cam.reach_b * z + h && -fyy <= cam.reach_t * z + h;
}

// The geometry half of Gaussian i (its mean already in gin.m): covariance, footprint, tile count; a visible one gets its
// parity outputs and the first two quarters of its blend record.  Returns the visibility; writes nothing for a culled one.
__device__ __forceinline__ bool project_one(const splx_gaussians& g, int64_t i, GeoIn& gin, const CamDev& cam,
                                            const splx_config& cfg, const splx_projected& out) {
  Geo G;
#pragma unroll
  for (int k = 0; k < 3; ++k) gin.ls[k] = g.log_scale[3 * i + k];
  gin.q = *reinterpret_cast<const float4*>(g.quat + 4 * i);
  const float logit = g.opacity_logit[i];       // requested with the others: one memory latency, not a second one behind the chain
  if (!geometry(gin, cam, cfg.dilation, G)) return false;
  const float mid = 0.5f * (G.a + G.c);
  const float hd = 0.5f * (G.a - G.c);
  const float lam = mid + sqrtf(fmaxf(cfg.radius_floor, hd * hd + G.b * G.b));  // mid^2 - det
  const int rad = (int)ceilf(3.0f * sqrtf(lam));
  const float iz = 1.0f / G.p[2];
  const float u = cam.fx * G.p[0] * iz + cam.cx;
  const float v = cam.fy * G.p[1] * iz + cam.cy;
  int x0, y0, x1, y1;
  tile_rect(u, v, rad, cam.TX, cam.TY, x0, y0, x1, y1);
  const int tt = (x1 - x0) * (y1 - y0);
  if (tt <= 0) return false;
  float4* bl = reinterpret_cast<float4*>(out.blend + SPLX_BLEND_STRIDE * i);
  const float idet = 1.0f / G.det;
  const float op = 1.0f / (1.0f + expf(-logit));
  *reinterpret_cast<float2*>(out.means2d + 2 * i) = make_float2(u, v);
  out.depth[i] = G.p[2];
  const float cA = G.c * idet, cB = -G.b * idet, cC = G.a * idet;
  *reinterpret_cast<float4*>(out.conic_opacity + 4 * i) = make_float4(cA, cB, cC, op);
  out.radius[i] = rad; out.tiles_touched[i] = (uint32_t)tt;
  constexpr float kLog2e = 1.4426950408889634f;
  bl[0] = make_float4(u, v, op, G.p[2]);
  bl[1] = make_float4(cA * (-0.5f * kLog2e), cB * (-kLog2e), cC * (-0.5f * kLog2e), __uint_as_float((uint32_t)i));
  return true;
}

// SH rows: a thread-per-Gaussian read of its 192-byte row is a 192-byte stride across the warp -- every 16-byte load
// instruction touches 32 different lines (32 L1 wavefronts instead of 4) and the kernel ran at half the HBM roof,
// bound by the L1's wavefront rate (ncu: lg_throttle + long_scoreboard stalls).  The 32 rows of a warp are 6 KB of
// CONTIGUOUS memory, so when at least SH_STAGE_MIN of them are visible the warp copies the block with coalesced
// 16-byte cp.async into shared memory (chunk index XOR-swizzled by the row so that the row-wise LDS.128 of a quarter
// warp hits eight different bank groups) and reads its rows from there; with fewer visible rows (the culled
// partitions of a city view) the direct loads touch less memory and are kept.
constexpr int SH_STAGE_MIN = 12;
// COLOUR = false (splx_project_geometry_plan): everything but the colour, which k_colour_list then computes for the
// VISIBLE Gaussians only.  On a city view ~13 % of the participating Gaussians are visible, scattered over the warps:
// nearly every warp ran the whole colour path (a third of the kernel's instructions) for 4 of its 32 lanes.
template <int DEG, bool COLOUR>
__global__ void __launch_bounds__(PROJ_THREADS)
k_project_fwd(splx_gaussians g, const __grid_constant__ PlanDev plan, const __grid_constant__ RunTable rt,
              splx_config cfg, splx_projected out) {
  constexpr int NSH = (DEG + 1) * (DEG + 1);
  constexpr int NV = (NSH * 3 + 3) / 4;
  constexpr bool STAGE = COLOUR && DEG > 0;
  __shared__ __align__(16) float4 s_sh[STAGE ? PROJ_THREADS * NV : 1];
  const int r = find_run(rt, (int)blockIdx.x);
  const int64_t i = rt.begin[r] + (int64_t)((int)blockIdx.x - rt.block_prefix[r]) * PROJ_THREADS + threadIdx.x;
  const bool active = i < rt.end[r];
  const CamDev& cam = plan.cam[rt.view[r]];   // the view this partition renders (indexed constant-bank loads)
  float m[3] = {0.f, 0.f, 0.f};
  bool vis = false;
  if (active) {
    GeoIn gin;
#pragma unroll
    for (int k = 0; k < 3; ++k) gin.m[k] = g.mean[3 * i + k];
    // reach test on the mean alone (splx_plan.max_scale, reading s21): most Gaussians of a city view fail it, and their
    // scale and rotation (28 of the 40 bytes a culled Gaussian costs) are never read
    const bool reach = reaches(gin.m, cam, plan.max_scale[rt.part[r]]);
    vis = reach && project_one(g, i, gin, cam, cfg, out);
    if (!vis) {   // a culled Gaussian: radius = tiles_touched = 0 say so; nothing downstream reads its other attributes, and
      out.radius[i] = 0; out.tiles_touched[i] = 0;     // writing 129 bytes of zeros for it was most of this kernel's traffic
    } else {
      m[0] = gin.m[0]; m[1] = gin.m[1]; m[2] = gin.m[2];
    }
  }
  if (!COLOUR) return;
  float4* bl = reinterpret_cast<float4*>(out.blend + SPLX_BLEND_STRIDE * i);
  const int lane = threadIdx.x & 31;
  const unsigned vmask = __ballot_sync(0xffffffffu, vis);
  if (vmask == 0) return;
  if (STAGE && __popc(vmask) >= SH_STAGE_MIN) {
    float4* ws = s_sh + (threadIdx.x & ~31) * NV;                 // this warp's 32 rows
    const int64_t i0 = i - lane;                                   // first Gaussian of the warp
    const int64_t left = rt.end[r] - i0;
    const int rows = (int)(left < 32 ? left : 32);
    const float4* src = reinterpret_cast<const float4*>(g.sh + 48 * i0);
    for (int c = lane; c < rows * NV; c += 32) {
      const int row = c / NV, q = c - row * NV;
      const unsigned dst = (unsigned)__cvta_generic_to_shared(ws + row * NV + sh_swz<NV>(q, row));
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + (size_t)row * 12 + q));
    }
    asm volatile("cp.async.commit_group;");
    asm volatile("cp.async.wait_group 0;");
    __syncwarp();
    if (vis) colour<DEG, true>(ws, lane, cam, m, i, out, bl);
    return;
  }
  if (vis) colour<DEG, false>(reinterpret_cast<const float4*>(g.sh + 48 * i), lane, cam, m, i, out, bl);
}

// The geometry half alone (splx_project_geometry_plan), in two phases per block of PG_TILE consecutive Gaussians.  On a
// city view ~85 % of the participating Gaussians fail the reach test on their mean and the few that pass are scattered
// over the warps: in the thread-per-Gaussian kernel above nearly every warp then ran the whole covariance chain (~300
// instructions) for 4 of its 32 lanes, and a thread had ONE mean in flight.  Phase 1: every thread tests PG_ITEMS means
// (their loads issued together), marks the ones that fail and appends the others to a list in shared memory; phase 2:
// the block walks the list with full warps.  Same arithmetic per Gaussian (project_one): bit-equal outputs.
constexpr int PG_ITEMS = 4;
constexpr int PG_TILE = PROJ_THREADS * PG_ITEMS;
__global__ void __launch_bounds__(PROJ_THREADS)
k_project_geo(splx_gaussians g, const __grid_constant__ PlanDev plan, const __grid_constant__ RunTable rt, splx_config cfg,
              splx_projected out) {
  __shared__ uint32_t s_list[PG_TILE];
  __shared__ uint32_t s_n;
  const int r = find_run(rt, (int)blockIdx.x);
  const int64_t base = rt.begin[r] + (int64_t)((int)blockIdx.x - rt.block_prefix[r]) * PG_TILE;
  const int64_t end = rt.end[r];
  const CamDev& cam = plan.cam[rt.view[r]];
  const float smax = plan.max_scale[rt.part[r]];
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  float m[PG_ITEMS][3];
#pragma unroll
  for (int it = 0; it < PG_ITEMS; ++it) {
    const int64_t i = base + it * PROJ_THREADS + threadIdx.x;
#pragma unroll
    for (int k = 0; k < 3; ++k) m[it][k] = i < end ? g.mean[3 * i + k] : 0.f;
  }
#pragma unroll
  for (int it = 0; it < PG_ITEMS; ++it) {
    const int64_t i = base + it * PROJ_THREADS + threadIdx.x;
    const bool reach = i < end && reaches(m[it], cam, smax);
    if (i < end && !reach) { out.radius[i] = 0; out.tiles_touched[i] = 0; }
    const unsigned bal = __ballot_sync(0xffffffffu, reach);
    uint32_t pos = 0;
    if (lane == 0 && bal) pos = atomicAdd(&s_n, (uint32_t)__popc(bal));
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if (reach) s_list[pos + __popc(bal & ((1u << lane) - 1u))] = (uint32_t)(it * PROJ_THREADS + threadIdx.x);
  }
  __syncthreads();
  const uint32_t cnt = s_n;
  for (uint32_t j = threadIdx.x; j < cnt; j += PROJ_THREADS) {
    const int64_t i = base + s_list[j];
    GeoIn gin;
#pragma unroll
    for (int k = 0; k < 3; ++k) gin.m[k] = g.mean[3 * i + k];
    if (!project_one(g, i, gin, cam, cfg, out)) { out.radius[i] = 0; out.tiles_touched[i] = 0; }
  }
}

// The colour of the visible Gaussians (the binning's list, index order): one thread per entry, persistent grid because
// the count lives on the device.  Same arithmetic as the colour half of k_project_fwd (bit-equal rgb, clamp, blend[2]).
// The 32 rows of a warp are scattered (192 contiguous bytes each): the warp copies them chunk by chunk -- lane c of
// round r takes chunk (32 r + c) % NV of row (32 r + c) / NV, so that 12 consecutive lanes cover one row's 192 bytes --
// into its swizzled shared-memory block with 16-byte cp.async, instead of every lane walking its own row with a
// 192-byte stride (32 L1 wavefronts per load instruction).
template <int DEG>
__global__ void __launch_bounds__(PROJ_THREADS)
k_colour_list(splx_gaussians g, const __grid_constant__ PlanDev plan, const __grid_constant__ RunTable rt, splx_projected out,
              const uint32_t* __restrict__ vlist, const uint64_t* __restrict__ nvis_ptr) {
  constexpr int NSH = (DEG + 1) * (DEG + 1);
  constexpr int NV = (NSH * 3 + 3) / 4;
  constexpr bool STAGE = DEG > 0;
  __shared__ __align__(16) float4 s_sh[STAGE ? PROJ_THREADS * NV : 1];
  const uint64_t nvis = *nvis_ptr;
  const int lane = threadIdx.x & 31;
  float4* ws = s_sh + (threadIdx.x & ~31) * NV;                 // this warp's 32 rows
  // whole warps stay in the loop together (j0 is warp uniform): the staging below is warp cooperative
  for (uint64_t j0 = (uint64_t)blockIdx.x * PROJ_THREADS + (threadIdx.x & ~31); j0 < nvis; j0 += (uint64_t)gridDim.x * PROJ_THREADS) {
    const uint64_t j = j0 + lane;
    const bool have = j < nvis;
    const int64_t i = have ? (int64_t)vlist[j] : 0;
    if (STAGE) {
      const int rows = (int)(nvis - j0 < 32 ? nvis - j0 : 32);
      __syncwarp();                                              // the previous round's reads of ws are done
      for (int c = lane; c < 32 * NV; c += 32) {
        const int row = c / NV, q = c - row * NV;
        const int64_t ir = __shfl_sync(0xffffffffu, i, row);
        if (row < rows) {
          const unsigned dst = (unsigned)__cvta_generic_to_shared(ws + row * NV + sh_swz<NV>(q, row));
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(reinterpret_cast<const float4*>(g.sh + 48 * ir) + q));
        }
      }
      asm volatile("cp.async.commit_group;");
    }
    const CamDev* cam = &plan.cam[0];
    float m[3] = {0.f, 0.f, 0.f};
    if (have) {
      int lo = 0, hi = rt.n - 1;                          // the run (partition) of Gaussian i -> its view
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (rt.begin[mid] <= i) lo = mid; else hi = mid - 1;
      }
      cam = &plan.cam[rt.view[lo]];
#pragma unroll
      for (int k = 0; k < 3; ++k) m[k] = g.mean[3 * i + k];
    }
    if (STAGE) {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      __syncwarp();
    }
    if (have) {
      float4* bl = reinterpret_cast<float4*>(out.blend + SPLX_BLEND_STRIDE * i);
      if (STAGE) colour<DEG, true>(ws, lane, *cam, m, i, out, bl);
      else colour<DEG, false>(reinterpret_cast<const float4*>(g.sh + 48 * i), lane, *cam, m, i, out, bl);
    }
  }
}

// Gradients of Y_l with respect to the (unconstrained) direction components.
__device__ __forceinline__ void sh_grad(int deg, float x, float y, float z, float (*dY)[3]) {
  for (int l = 0; l < (deg + 1) * (deg + 1); ++l) dY[l][0] = dY[l][1] = dY[l][2] = 0.f;
  if (deg < 1) return;
  dY[1][1] = -kK1; dY[2][2] = kK1; dY[3][0] = -kK1;
  if (deg < 2) return;
  dY[4][0] = kK2a * y; dY[4][1] = kK2a * x;
  dY[5][1] = -kK2a * z; dY[5][2] = -kK2a * y;
  dY[6][0] = -2.f * kK2b * x; dY[6][1] = -2.f * kK2b * y; dY[6][2] = 4.f * kK2b * z;
  dY[7][0] = -kK2a * z; dY[7][2] = -kK2a * x;
  dY[8][0] = 2.f * kK2c * x; dY[8][1] = -2.f * kK2c * y;
  if (deg < 3) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  dY[9][0] = -6.f * kK3a * x * y; dY[9][1] = -3.f * kK3a * (xx - yy);
  dY[10][0] = kK3b * y * z; dY[10][1] = kK3b * x * z; dY[10][2] = kK3b * x * y;
  dY[11][0] = 2.f * kK3c * x * y; dY[11][1] = -kK3c * (4.f * zz - xx - 3.f * yy); dY[11][2] = -8.f * kK3c * y * z;
  dY[12][0] = -6.f * kK3d * x * z; dY[12][1] = -6.f * kK3d * y * z; dY[12][2] = 3.f * kK3d * (2.f * zz - xx - yy);
  dY[13][0] = -kK3c * (4.f * zz - 3.f * xx - yy); dY[13][1] = 2.f * kK3c * x * y; dY[13][2] = -8.f * kK3c * x * z;
  dY[14][0] = 2.f * kK3e * x * z; dY[14][1] = -2.f * kK3e * y * z; dY[14][2] = kK3e * (xx - yy);
  dY[15][0] = -3.f * kK3a * (xx - yy); dY[15][1] = 6.f * kK3a * x * y;
}

// Backward block = 128 Gaussians.  The 48 SH coefficients of a Gaussian are 192 contiguous bytes, so a
// thread-per-Gaussian access has a 192-byte stride: scattered 4-byte read-modify-writes of the SH
// gradient ran at 9 % of the HBM roof (profiles/r01a_launches_aerial_1M.md).  Here the block's SH tile [128][48] and, when
// accumulating, the tile of the SH gradient travel global -> shared with 16-byte cp.async (LDGSTS)
// issued before the geometry chain, so ~50 KB per block are in flight while the ALU work runs; the
// result leaves with coalesced 128-bit stores.  Row stride 52 floats keeps 16-byte alignment and makes
// both the row-wise LDS.128 of a thread and the cooperative pass conflict-free.  mean / log_scale
// gradients (12-byte stride) are staged the same way.  Culled rows are never read.
constexpr int PB_THREADS = 128;
constexpr int PB_STRIDE = 52;

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

constexpr int PB_MIN_CTAS = 5;   // 96 registers, no spills; 6 spills and is not faster (measured)
// LIST (accumulating launches only): the rows of a block are 128 entries of the binning's list of VISIBLE Gaussians
// (splx_bin_sort_visible) instead of 128 consecutive Gaussians, so the work follows the visible count -- on the
// city scenes ~10 % of the participating Gaussians -- and not the partition sizes; the grid is persistent because
// the count lives on the device.
template <int DEG, bool ACC, int LIST>   // LIST: 0 = every row of the runs, 1 = the visible list, 2 = the list + `touched` flags
__global__ void __launch_bounds__(PB_THREADS, PB_MIN_CTAS)
k_project_bwd(splx_gaussians g, const __grid_constant__ PlanDev plan, const __grid_constant__ RunTable rt,
              splx_config cfg, splx_projected pr, float* __restrict__ g2d, int clear_g2d, splx_gaussian_grads out,
              const uint32_t* __restrict__ vlist, const uint64_t* __restrict__ nvis_ptr, uint8_t* __restrict__ touched) {
  extern __shared__ __align__(16) float s_dyn[];
  float* s_sh = s_dyn;                                   // [128][52] sh in, SH gradient out
  float* s_old = s_dyn + PB_THREADS * PB_STRIDE;         // [128][52] previous SH gradient (ACC only)
  __shared__ __align__(16) float s_m[PB_THREADS * 3];    // mean gradient tile
  __shared__ __align__(16) float s_s[PB_THREADS * 3];    // log_scale gradient tile
  __shared__ uint8_t s_vis[PB_THREADS];
  __shared__ int64_t s_idx[PB_THREADS];                  // Gaussian of each row of the block
  __shared__ uint8_t s_fresh[LIST == 2 ? PB_THREADS : 1];                // LIST + touched: first gradient of this row in the iteration ("=")
  const uint64_t nvis = LIST ? *nvis_ptr : 0;
  for (uint64_t blk = blockIdx.x; LIST ? (blk * PB_THREADS < nvis) : (blk == blockIdx.x); blk += gridDim.x) {
  int64_t base = 0, run_end = 0, i = 0;
  int nrows, view;
  if (LIST) {
    const uint64_t j0 = blk * PB_THREADS;
    nrows = (int)min((uint64_t)PB_THREADS, nvis - j0);
    view = 0;
    if ((int)threadIdx.x < nrows) {
      i = (int64_t)vlist[j0 + threadIdx.x];
      run_end = i + 1;
      int lo = 0, hi = rt.n - 1;                          // the run (partition) of Gaussian i -> its view
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (rt.begin[mid] <= i) lo = mid; else hi = mid - 1;
      }
      view = rt.view[lo];
    }
  } else {
    const int run = find_run(rt, (int)blockIdx.x);
    base = rt.begin[run] + (int64_t)((int)blockIdx.x - rt.block_prefix[run]) * PB_THREADS;
    run_end = rt.end[run];
    i = base + threadIdx.x;
    nrows = (int)min((int64_t)PB_THREADS, run_end - base);
    view = rt.view[run];                                  // < 0: a non-participating partition (OVERWRITE only): zeros
  }
  s_idx[threadIdx.x] = i;
  const CamDev& cam = plan.cam[view < 0 ? 0 : view];
  constexpr int NSH = (DEG + 1) * (DEG + 1);
  constexpr int NV = (NSH * 3 + 3) / 4;        // float4 chunks of a row that hold used coefficients
  // Two dependent rounds of loads: the radius (4 B per row, decides visibility), then -- for visible rows only --
  // every other per-Gaussian input at once (independent loads in flight together).  Requesting them inside the
  // geometry chain stalled the kernel on dependent loads (23 % of DRAM peak); requesting them for culled rows too
  // moved ~100 B per culled row, which is most rows on the city scenes.
  const bool inr = (i < run_end) && (view >= 0);
  const int rad = inr ? pr.radius[i] : 0;
  GeoIn gin;
  float4 g0 = make_float4(0.f, 0.f, 0.f, 0.f), g1 = g0, g2 = g0;
  float op = 0.f;
  uint8_t cl = 0;
  float4* gp = reinterpret_cast<float4*>(g2d + (int64_t)SPLX_G2D_STRIDE * i);
  if (rad > 0) {
    gin = load_geo(g, i);
    g0 = gp[0]; g1 = gp[1]; g2 = gp[2];
    op = pr.conic_opacity[4 * i + 3];
    cl = pr.clamp[i];
  }
  const bool vis = inr && rad > 0;
  s_vis[threadIdx.x] = vis ? 1 : 0;
  // sparse-optimiser mode: a row whose flag is still clear has no gradient yet in this iteration: its old content is
  // garbage, this launch stores instead of accumulating and sets the flag (a list holds a Gaussian once: no race)
  bool fresh = false;
  if (LIST == 2 && vis) {
    fresh = touched[i] == 0;
    touched[i] = 1;
  }
  if (LIST == 2) s_fresh[threadIdx.x] = fresh ? 1 : 0;
  __syncthreads();
#pragma unroll
  for (int c = 0; c < NV; ++c) {
    const int q = c * PB_THREADS + threadIdx.x;
    const int row = q / NV, c4 = q - row * NV;
    if (row < nrows && s_vis[row]) {
      cp_async16(s_sh + row * PB_STRIDE + 4 * c4, g.sh + 48 * s_idx[row] + 4 * c4);
      // (LIST: the previous gradient is never read: the write-back ADDS in memory with vector reductions, see below)
      if (ACC && !LIST) {
        cp_async16(s_old + row * PB_STRIDE + 4 * c4, out.sh + 48 * s_idx[row] + 4 * c4);
      }
    }
  }
  float dmu[3] = {0.f, 0.f, 0.f}, dls[3] = {0.f, 0.f, 0.f};
  float4 dq = make_float4(0.f, 0.f, 0.f, 0.f);
  float dlogit = 0.f;
  float grgb[3] = {0.f, 0.f, 0.f};
  Geo G;
  if (vis && geometry(gin, cam, cfg.dilation, G)) {
    if (clear_g2d) { const float4 zz = make_float4(0.f, 0.f, 0.f, 0.f); gp[0] = zz; gp[1] = zz; gp[2] = zz; }
    const float gu = g0.x, gv = g0.y, gA = g0.z, gB = g0.w, gC = g1.x, gop = g1.y;
    grgb[0] = g1.z; grgb[1] = g1.w; grgb[2] = g2.x;
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) if ((cl >> ch) & 1) grgb[ch] = 0.f;

    // opacity: o = sigmoid(logit)
    dlogit = op * (1.f - op) * gop;

    // conic Q = P^-1 (P = Sigma2D):  dL/dP = -Q Gm Q,  Gm = [[gA, gB/2],[gB/2, gC]]
    const float idet = 1.0f / G.det;
    const float A = G.c * idet, B = -G.b * idet, C = G.a * idet;
    const float hB = 0.5f * gB;
    const float qg00 = A * gA + B * hB, qg01 = A * hB + B * gC;
    const float qg10 = B * gA + C * hB, qg11 = B * hB + C * gC;
    const float p00 = -(qg00 * A + qg01 * B), p01 = -(qg00 * B + qg01 * C);
    const float p11 = -(qg10 * B + qg11 * C);   // symmetric: p10 == p01
    // P = N N^T + dI, N = Tm Mm:  dL/dN = 2 Gc N;   dL/dTm = dL/dN Mm^T;  dL/dMm = Tm^T dL/dN
    float dN[6];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      dN[c] = 2.f * (p00 * G.N[c] + p01 * G.N[3 + c]);
      dN[3 + c] = 2.f * (p01 * G.N[c] + p11 * G.N[3 + c]);
    }
    float dTm[6], dMm[9];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int k = 0; k < 3; ++k)
        dTm[3 * r + k] = dN[3 * r] * G.Mm[3 * k] + dN[3 * r + 1] * G.Mm[3 * k + 1] + dN[3 * r + 2] * G.Mm[3 * k + 2];
#pragma unroll
    for (int k = 0; k < 3; ++k)
#pragma unroll
      for (int c = 0; c < 3; ++c) dMm[3 * k + c] = G.Tm[k] * dN[c] + G.Tm[3 + k] * dN[3 + c];
    // Tm = J W:  dL/dJ = dL/dTm W^T.  J = [[fx/z, 0, -fx Lx/z],[0, fy/z, -fy Ly/z]]
    const float dJ00 = dTm[0] * cam.R[0] + dTm[1] * cam.R[1] + dTm[2] * cam.R[2];
    const float dJ02 = dTm[0] * cam.R[6] + dTm[1] * cam.R[7] + dTm[2] * cam.R[8];
    const float dJ11 = dTm[3] * cam.R[3] + dTm[4] * cam.R[4] + dTm[5] * cam.R[5];
    const float dJ12 = dTm[3] * cam.R[6] + dTm[4] * cam.R[7] + dTm[5] * cam.R[8];
    const float z = G.p[2], iz = 1.f / z, iz2 = iz * iz;
    float dp[3] = {0.f, 0.f, 0.f};
    dp[2] += -cam.fx * iz2 * dJ00 - cam.fy * iz2 * dJ11;
    // J02 = -fx Lx / z with Lx = clamp(x/z): inside the clamp Lx = x/z -> J02 = -fx x / z^2
    if (!G.clx) { dp[0] += -cam.fx * iz2 * dJ02; dp[2] += 2.f * cam.fx * G.p[0] * iz2 * iz * dJ02; }
    else        { dp[2] += cam.fx * G.Lx * iz2 * dJ02; }
    if (!G.cly) { dp[1] += -cam.fy * iz2 * dJ12; dp[2] += 2.f * cam.fy * G.p[1] * iz2 * iz * dJ12; }
    else        { dp[2] += cam.fy * G.Ly * iz2 * dJ12; }
    // 2-D mean
    dp[0] += cam.fx * iz * gu;
    dp[1] += cam.fy * iz * gv;
    dp[2] += -(cam.fx * G.p[0] * gu + cam.fy * G.p[1] * gv) * iz2;
#pragma unroll
    for (int k = 0; k < 3; ++k)
      dmu[k] = cam.R[k] * dp[0] + cam.R[3 + k] * dp[1] + cam.R[6 + k] * dp[2];

    // Mm = Rot diag(s)
    float dRot[9];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      float ds = 0.f;
#pragma unroll
      for (int r = 0; r < 3; ++r) { ds = fmaf(G.Rot[3 * r + c], dMm[3 * r + c], ds); dRot[3 * r + c] = G.s[c] * dMm[3 * r + c]; }
      dls[c] = G.s[c] * ds;
    }
    // Rot(q_hat) then the normalisation q_hat = q/|q|
    const float w = G.qh[0], x = G.qh[1], y = G.qh[2], zq = G.qh[3];
    float gq[4];
    gq[0] = 2.f * (-zq * dRot[1] + y * dRot[2] + zq * dRot[3] - x * dRot[5] - y * dRot[6] + x * dRot[7]);
    gq[1] = 2.f * (y * dRot[1] + zq * dRot[2] + y * dRot[3] - 2.f * x * dRot[4] - w * dRot[5] + zq * dRot[6] + w * dRot[7] - 2.f * x * dRot[8]);
    gq[2] = 2.f * (-2.f * y * dRot[0] + x * dRot[1] + w * dRot[2] + x * dRot[3] + zq * dRot[5] - w * dRot[6] + zq * dRot[7] - 2.f * y * dRot[8]);
    gq[3] = 2.f * (-2.f * zq * dRot[0] - w * dRot[1] + x * dRot[2] + w * dRot[3] - 2.f * zq * dRot[4] + y * dRot[5] + x * dRot[6] + y * dRot[7]);
    const float qd = w * gq[0] + x * gq[1] + y * gq[2] + zq * gq[3];
    const float iqn = 1.f / G.qn;
    dq = make_float4((gq[0] - w * qd) * iqn, (gq[1] - x * qd) * iqn, (gq[2] - y * qd) * iqn, (gq[3] - zq * qd) * iqn);
  }
  cp_async_wait_all();
  __syncthreads();
  if (vis) {
    // colour: rgb = max(0, 0.5 + sum_l Y_l(dir) sh_l), dir = (mu - o)/|mu - o|
    float dv[3] = {gin.m[0] - cam.o[0], gin.m[1] - cam.o[1], gin.m[2] - cam.o[2]};
    const float dinv = rsqrtf(dv[0] * dv[0] + dv[1] * dv[1] + dv[2] * dv[2]);
    const float dir[3] = {dv[0] * dinv, dv[1] * dinv, dv[2] * dinv};
    float Y[NSH];
    sh_eval(DEG, dir[0], dir[1], dir[2], Y);
    float dot[NSH];
#pragma unroll
    for (int l = 0; l < NSH; ++l) dot[l] = 0.f;
    float4* row = reinterpret_cast<float4*>(s_sh + threadIdx.x * PB_STRIDE);
    // the row is read (sh) and overwritten in place with this view's SH gradient Y_l * dL/drgb
#pragma unroll
    for (int q = 0; q < NV; ++q) {
      const float4 f = row[q];
      const float e[4] = {f.x, f.y, f.z, f.w};
      float o4[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) {
        const int idx = 4 * q + t;
        if (idx < NSH * 3) {
          dot[idx / 3] = fmaf(e[t], grgb[idx % 3], dot[idx / 3]);
          o4[t] = Y[idx / 3] * grgb[idx % 3];
        } else {
          o4[t] = 0.f;
        }
      }
      row[q] = make_float4(o4[0], o4[1], o4[2], o4[3]);
    }
    float dY[NSH][3];
    sh_grad(DEG, dir[0], dir[1], dir[2], dY);
    float gdir[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int l = 0; l < NSH; ++l)
#pragma unroll
      for (int k = 0; k < 3; ++k) gdir[k] = fmaf(dY[l][k], dot[l], gdir[k]);
    const float dd = dir[0] * gdir[0] + dir[1] * gdir[1] + dir[2] * gdir[2];
#pragma unroll
    for (int k = 0; k < 3; ++k) dmu[k] += (gdir[k] - dir[k] * dd) * dinv;
  }
#pragma unroll
  for (int k = 0; k < 3; ++k) { s_m[3 * threadIdx.x + k] = dmu[k]; s_s[3 * threadIdx.x + k] = dls[k]; }
  if (i < run_end) {
    float4* oq = reinterpret_cast<float4*>(out.quat + 4 * i);
    if (ACC) {
      if (vis) {
        if (LIST && !fresh) {       // a list holds a Gaussian once: the reduction is the plain sum old + new, without reading old here
          atomicAdd(oq, dq);
          atomicAdd(out.opacity_logit + i, dlogit);
        } else {
          float4 cur = fresh ? make_float4(0.f, 0.f, 0.f, 0.f) : *oq;
          cur.x += dq.x; cur.y += dq.y; cur.z += dq.z; cur.w += dq.w;
          *oq = cur;
          out.opacity_logit[i] = (fresh ? 0.f : out.opacity_logit[i]) + dlogit;
        }
      }
    } else {
      *oq = dq;
      out.opacity_logit[i] = dlogit;
    }
  }
  __syncthreads();
  // coalesced write-back of the SH-gradient tile (+= needs visible rows only; = writes every row)
#pragma unroll
  for (int c = 0; c < 12; ++c) {
    const int q = c * PB_THREADS + threadIdx.x;
    const int row = q / 12, c4 = q - row * 12;
    if (row < nrows) {
      float4* dst = reinterpret_cast<float4*>(out.sh + 48 * s_idx[row]) + c4;
      const bool live = s_vis[row] && c4 < NV;
      if (ACC) {
        if (live) {
          const float4 a = *reinterpret_cast<const float4*>(s_sh + row * PB_STRIDE + 4 * c4);
          if (LIST) {
            // red.global.add.v4.f32 (sm_90+): the sum is formed in L2, nothing waits for the old value and no tile of
            // old gradients is staged -- half the shared memory, 5 resident CTAs instead of 4
            if (LIST == 2 && s_fresh[row]) *dst = make_float4(0.f + a.x, 0.f + a.y, 0.f + a.z, 0.f + a.w);
            else atomicAdd(dst, a);
          } else {
            const float4 o = *reinterpret_cast<const float4*>(s_old + row * PB_STRIDE + 4 * c4);
            *dst = make_float4(o.x + a.x, o.y + a.y, o.z + a.z, o.w + a.w);
          }
        } else if (LIST == 2 && s_fresh[row]) {
          *dst = make_float4(0.f, 0.f, 0.f, 0.f);       // coefficients above sh_degree of a freshly stored row
        }
      } else {
        *dst = live ? *reinterpret_cast<const float4*>(s_sh + row * PB_STRIDE + 4 * c4) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
  }
  // mean / log_scale gradient tiles: 96 float4 each; a partial last block, or a run that does not start
  // on a multiple of 4 Gaussians (12-byte rows: 16-byte alignment needs base % 4 == 0), falls back to scalars
  if (!LIST && nrows == PB_THREADS && (base & 3) == 0) {
    if (threadIdx.x < 96) {
      float4* dm = reinterpret_cast<float4*>(out.mean + 3 * base) + threadIdx.x;
      float4* ds = reinterpret_cast<float4*>(out.log_scale + 3 * base) + threadIdx.x;
      float4 a = reinterpret_cast<const float4*>(s_m)[threadIdx.x], b = reinterpret_cast<const float4*>(s_s)[threadIdx.x];
      if (ACC) {
        const float4 om = *dm, os = *ds;
        a.x += om.x; a.y += om.y; a.z += om.z; a.w += om.w;
        b.x += os.x; b.y += os.y; b.z += os.z; b.w += os.w;
      }
      *dm = a; *ds = b;
    }
  } else if (i < run_end) {
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      if (ACC && LIST && !fresh) {
        if (vis) { atomicAdd(out.mean + 3 * i + k, dmu[k]); atomicAdd(out.log_scale + 3 * i + k, dls[k]); }
      } else if (ACC) {
        out.mean[3 * i + k] = (fresh ? 0.f : out.mean[3 * i + k]) + dmu[k];
        out.log_scale[3 * i + k] = (fresh ? 0.f : out.log_scale[3 * i + k]) + dls[k];
      }
      else     { out.mean[3 * i + k] = dmu[k]; out.log_scale[3 * i + k] = dls[k]; }
    }
  }
  __syncthreads();      // LIST: the next block of rows reuses the shared tiles
  }
}

template <int DEG, bool ACC>
static void launch_pb(splx_ctx* ctx, const splx_gaussians* g, const PlanDev& plan, const RunTable& rt,
                      const splx_projected* pr, float* g2d, int clear_g2d, const splx_gaussian_grads* grads) {
  const size_t smem = (size_t)PB_THREADS * PB_STRIDE * sizeof(float) * (ACC ? 2 : 1);
  cudaFuncSetAttribute(k_project_bwd<DEG, ACC, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaFuncSetAttribute(k_project_bwd<DEG, ACC, 0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  k_project_bwd<DEG, ACC, 0><<<(unsigned)rt.blocks_total, PB_THREADS, smem, ctx->stream>>>(
      *g, plan, rt, ctx->cfg, *pr, g2d, clear_g2d, *grads, nullptr, nullptr, nullptr);
}

// accumulating launch over the list of visible Gaussians (persistent grid: the count lives on the device)
template <int DEG, int LIST>
static void launch_pb_list(splx_ctx* ctx, const splx_gaussians* g, const PlanDev& plan, const RunTable& rt,
                           const splx_projected* pr, float* g2d, int clear_g2d, const splx_gaussian_grads* grads,
                           const uint32_t* vlist, const uint64_t* nvis, uint8_t* touched) {
  const size_t smem = (size_t)PB_THREADS * PB_STRIDE * sizeof(float);     // the SH tile only
  const int64_t need = (rt.jprefix[rt.n] + PB_THREADS - 1) / PB_THREADS;
  const int64_t grid = need < (int64_t)SPLX_SM_COUNT * 5 ? need : (int64_t)SPLX_SM_COUNT * 5;     // 96 registers: 5 resident CTAs
  cudaFuncSetAttribute(k_project_bwd<DEG, true, LIST>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaFuncSetAttribute(k_project_bwd<DEG, true, LIST>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
  k_project_bwd<DEG, true, LIST><<<(unsigned)grid, PB_THREADS, smem, ctx->stream>>>(
      *g, plan, rt, ctx->cfg, *pr, g2d, clear_g2d, *grads, vlist, nvis, touched);
}

template <int DEG>
static void launch_pb_deg(splx_ctx* ctx, bool overwrite, const splx_gaussians* g, const PlanDev& plan, const RunTable& rt,
                          const splx_projected* pr, float* g2d, int clr, const splx_gaussian_grads* grads,
                          const uint32_t* vlist, const uint64_t* nvis, uint8_t* touched) {
  if (vlist && touched) launch_pb_list<DEG, 2>(ctx, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched);
  else if (vlist) launch_pb_list<DEG, 1>(ctx, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched);
  else if (overwrite) launch_pb<DEG, false>(ctx, g, plan, rt, pr, g2d, clr, grads);
  else launch_pb<DEG, true>(ctx, g, plan, rt, pr, g2d, clr, grads);
}

}  // namespace

int launch_project_fwd(splx_ctx* ctx, const splx_gaussians* g, const PlanDev& plan, const int64_t* part_offsets, int deg,
                       const splx_projected* out, bool with_colour) {
  const RunTable rt = make_runs(plan, part_offsets, PROJ_THREADS, false);
  if (rt.blocks_total == 0) return SPLX_OK;
  const unsigned grid = (unsigned)rt.blocks_total;
#define PF(D, C) k_project_fwd<D, C><<<grid, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rt, ctx->cfg, *out)
  if (with_colour) {
    switch (deg) { case 0: PF(0, true); break; case 1: PF(1, true); break; case 2: PF(2, true); break; default: PF(3, true); break; }
  } else {               // the degree only matters to the colour
    const RunTable rg = make_runs(plan, part_offsets, PG_TILE, false);
    k_project_geo<<<(unsigned)rg.blocks_total, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rg, ctx->cfg, *out);
  }
#undef PF
  SPLX_LAUNCH_CHECK(ctx, with_colour ? "k_project_fwd" : "k_project_geo");
  return SPLX_OK;
}

int launch_project_colour_list(splx_ctx* ctx, const splx_gaussians* g, const PlanDev& plan, const int64_t* part_offsets, int deg,
                               const splx_projected* out, const uint32_t* vlist, const uint64_t* nvis) {
  const RunTable rt = make_runs(plan, part_offsets, PROJ_THREADS, false);
  if (rt.blocks_total == 0) return SPLX_OK;
  const unsigned grid = SPLX_SM_COUNT * 8;     // persistent: the count lives on the device
  switch (deg) {
    case 0: k_colour_list<0><<<grid, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rt, *out, vlist, nvis); break;
    case 1: k_colour_list<1><<<grid, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rt, *out, vlist, nvis); break;
    case 2: k_colour_list<2><<<grid, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rt, *out, vlist, nvis); break;
    default: k_colour_list<3><<<grid, PROJ_THREADS, 0, ctx->stream>>>(*g, plan, rt, *out, vlist, nvis); break;
  }
  SPLX_LAUNCH_CHECK(ctx, "k_colour_list");
  return SPLX_OK;
}

int launch_project_bwd(splx_ctx* ctx, const splx_gaussians* g, const PlanDev& plan, const int64_t* part_offsets, int deg,
                       const splx_projected* pr, float* g2d, int flags, const splx_gaussian_grads* grads,
                       const uint32_t* vlist, const uint64_t* nvis, uint8_t* touched) {
  const int clr = (flags & SPLX_PB_CLEAR_G2D) ? 1 : 0;
  const bool overwrite = (flags & SPLX_PB_OVERWRITE) != 0;
  const bool list = vlist && nvis && !overwrite;      // += over the visible Gaussians only
  // "=" must also clear the rows of partitions that do not participate in this launch
  const RunTable rt = make_runs(plan, part_offsets, PB_THREADS, overwrite);
  if (list ? rt.jprefix[rt.n] == 0 : rt.blocks_total == 0) return SPLX_OK;
  if (!list) { vlist = nullptr; nvis = nullptr; touched = nullptr; }
  switch (deg) {
    case 0: launch_pb_deg<0>(ctx, overwrite, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched); break;
    case 1: launch_pb_deg<1>(ctx, overwrite, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched); break;
    case 2: launch_pb_deg<2>(ctx, overwrite, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched); break;
    default: launch_pb_deg<3>(ctx, overwrite, g, plan, rt, pr, g2d, clr, grads, vlist, nvis, touched); break;
  }
  SPLX_LAUNCH_CHECK(ctx, "k_project_bwd");
  return SPLX_OK;
}
