// sort.cu -- steps a2-a4: tile-intersection keys, stable radix sort, per-tile ranges.
// PAPER.md L81 ("3D Gaussians are sorted based on their distance from the camera, i.e., depth
// d"), L165 (each rank blends "in depth order").  Mechanism: 64-bit key =
// (slot << 32) | float_bits(depth), slot = partition * tiles + tile; result = the STABLE sort
// of the (key, Gaussian index) pairs emitted in Gaussian-index order.
//
// B200 design: the full sort is split so that the wide keys are moved as little as possible.
//   1. compact the visible Gaussians in index order: count -> scan -> scatter (8 B read per participating Gaussian,
//      12 B written per visible one)
//   2. stable LSD radix sort of (depth bits, index), 4 x 8 bits (over N_visible, not over M)
//   3. exclusive scan of tiles_touched in that depth order, emit (sort slot, depth-order position) pairs in that order
//   4. stable LSD radix sort on the sort-slot bits only (the slots of the participating partitions, or -- splx_plan.open_slots --
//      of their open slots: 2-3 passes); the last pass writes the 64-bit keys and the values
//   5. tile ranges from the sorted keys, slot order by descending list length
// Step 2 + step 4 give exactly the stable sort on the whole key: within a slot the entries
// keep the order of step 2 = (depth bits, index).  No host synchronisation: the counts
// (N_visible, M) stay on the device and every grid is sized from the caller's capacities.
#include "common.cuh"

namespace {

// 8 items per thread against 16, same session: city_10M 12.50 / 12.62 ms, street_10M 16.46 / 16.56, city_100M 66.8 / 67.2
constexpr int SCAN_THREADS = 512, SCAN_IPT = 8, SCAN_TILE = SCAN_THREADS * SCAN_IPT;   // 4096 elements per tile
constexpr int RS_THREADS = 256, RS_IPT = 8, RS_TILE = RS_THREADS * RS_IPT, RS_WARPS = 8;  // 2048
constexpr int MAX_PASSES = 4;
// Digit values of the slot sort.  512 (9-bit digits: <= 18 compact slot bits in two passes instead of three) is implemented
// (radix_tile<..., 512>: two digits per thread in the per-digit phases) and was MEASURED SLOWER everywhere: bin/sort
// 11.9 -> 12.8 ms on city_100M and 13.3 -> 15.0 ms on city_40M although a pass is saved there, 0.32 -> 0.37 ms on
// aerial_1M and 2.8 -> 3.6 ms on city_10M where none is (twice the look-back chains per thread, 512 status words per
// 2048-key tile, 39 KB of shared memory).  256 stays.
constexpr int SLOT_NB = 256;
constexpr int SLOT_BITS = SLOT_NB == 256 ? 8 : 9;
static_assert(SCAN_TILE % RS_TILE == 0, "the compaction scan clears the radix status words of the tiles it covers");
constexpr int SCAN_RS = SCAN_TILE / RS_TILE;
constexpr uint32_t PERSISTENT_CTAS = SPLX_SM_COUNT * 8;   // grid of the persistent kernels: 8 CTAs per SM

struct Counters {   // device-resident counts, written by kernels, read by later kernels
  uint64_t n_visible;
  uint64_t n_rows;      // entries of the list of Gaussians with a non-zero 2-D gradient (k_gradient_rows)
  uint64_t m_total;     // true number of intersections
  uint64_t m_sorted;    // min(m_total, capacity)
  uint32_t ticket[16];  // dynamic tile counters, one per single-pass kernel of the pipeline
};

// rank[k]: position of partition k among the partitions that take part in this launch (-1: it does not).  The slot sort
// runs on the COMPACT slot rank[k] * ntiles + tile -- monotone in the true slot k * ntiles + tile, so the order is the
// same, with fewer key bits (6-8 of 32 partitions take part in a city view: 16 bits instead of 18, two passes for three).
struct PartOffs { int64_t off[SPLX_MAX_K + 1]; int K; signed char rank[SPLX_MAX_K]; };

// Tile status word of the single-pass ("decoupled look-back") scans: flag in the top two bits,
// running count below.  A tile publishes its own total (AGG) as soon as it knows it and its
// inclusive prefix (PREFIX) once it has walked back to a predecessor that published one.
// Tiles take their index from an atomic ticket, so every predecessor of a running tile has
// started: the spin below cannot wait on a CTA that was never scheduled.
constexpr uint64_t ST_AGG = 1ull << 62, ST_PREFIX = 2ull << 62, ST_MASK = 3ull << 62;

__device__ __forceinline__ uint64_t ld_status(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(uint64_t* p, uint64_t v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// exclusive prefix of tile t (t > 0) given its own total: publish, look back, publish again.
// The walk reads W predecessors per round trip (independent loads), consumes them nearest first
// and stops at the first PREFIX; a predecessor that has published nothing yet ends the round.
template <int W>
__device__ __forceinline__ uint64_t lookback(uint64_t* status, uint32_t t, uint32_t stride, uint64_t total) {
  st_status(status + (uint64_t)t * stride, ST_AGG | total);
  uint64_t excl = 0;
  int64_t p = (int64_t)t - 1;
  while (p >= 0) {
    uint64_t v[W];
#pragma unroll
    for (int i = 0; i < W; ++i) v[i] = (p - i >= 0) ? ld_status(status + (uint64_t)(p - i) * stride) : ST_PREFIX;
    bool done = false;
    int used = 0;
#pragma unroll
    for (int i = 0; i < W; ++i) {
      if (!done && used == i && (v[i] & ST_MASK) != 0) {
        excl += v[i] & ~ST_MASK;
        ++used;
        if ((v[i] & ST_MASK) == ST_PREFIX) done = true;
      }
    }
    if (done) break;
    p -= used;
    if (used == 0) __nanosleep(20);
  }
  st_status(status + (uint64_t)t * stride, ST_PREFIX | (excl + total));
  return excl;
}

// ---------------------------------------------------------------- generic exclusive scan --
// One launch: tiles of SCAN_TILE values, chained by look-back.  Op supplies count(), load(i) and
// store(i, value, exclusive_prefix).  The grand total goes to *total_out (and, clamped, to *clamp_out).

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* smem /*>=33*/, uint32_t& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) smem[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < nw ? smem[lane] : 0, wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += t; }
    smem[lane] = wi - w;           // exclusive warp offsets
    if (lane == 31) smem[32] = wi;  // block total
  }
  __syncthreads();
  const uint32_t res = inc - v + smem[warp];
  total = smem[32];
  __syncthreads();
  return res;
}

// Persistent: a CTA keeps taking tiles from the ticket counter until the (device-side) element count is
// exhausted, so the grid is sized for the machine, not for the caller's capacity.
template <class Op>
__global__ void __launch_bounds__(SCAN_THREADS, 2)
k_scan(const __grid_constant__ Op op, const uint64_t* n_ptr, uint64_t* status, uint32_t* ticket, uint64_t* total_out, uint64_t* clamp_out,
       uint64_t clamp_to) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_tile;
  __shared__ uint64_t s_excl;
  const uint64_t n = op.count(n_ptr);
  const uint64_t ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (n == 0) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
      if (total_out) *total_out = 0;
      if (clamp_out) *clamp_out = 0;
    }
    return;
  }
  for (;;) {
    __syncthreads();                       // s_tile / s_excl of the previous round are no longer read
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t t = s_tile;
    if (t >= ntiles) break;
    const uint64_t base = (uint64_t)t * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_IPT;
    uint32_t v[SCAN_IPT], s = 0;
    op.load_all(base, n, v);                 // the thread's SCAN_IPT elements are consecutive
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) s += v[k];
    uint32_t total;
    uint32_t ex = block_exclusive_scan(s, sm, total);
    if (threadIdx.x == 0) {
      uint64_t excl = 0;
      if (t == 0) st_status(status, ST_PREFIX | (uint64_t)total);
      else excl = lookback<16>(status, t, 1, total);
      s_excl = excl;
      if (t + 1 == ntiles) {
        const uint64_t grand = excl + total;
        if (total_out) *total_out = grand;
        if (clamp_out) *clamp_out = grand < clamp_to ? grand : clamp_to;
      }
    }
    __syncthreads();
    ex += (uint32_t)s_excl;
    op.store_all(base, n, v, ex, nullptr);
  }
}

struct RunMap {
  int n;
  int64_t begin[SPLX_MAX_K], jprefix[SPLX_MAX_K + 1];
  __device__ uint64_t operator()(uint64_t j) const {
    int lo = 0, hi = n - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if ((uint64_t)jprefix[mid] <= j) lo = mid; else hi = mid - 1;
    }
    return (uint64_t)begin[lo] + (j - (uint64_t)jprefix[lo]);
  }
};

struct VisibleOp {  // step 1: compaction of the visible Gaussians, index order preserved
  const uint32_t* tiles_touched; const float* depth; uint32_t* ckeys; uint32_t* cvals; uint32_t* vis_list; uint64_t n; RunMap map;
  __device__ uint64_t count(const uint64_t*) const { return n; }
  // A thread's SCAN_IPT elements are consecutive positions j of the concatenated runs: the run of the first one is
  // searched once (a <= 6-step search over the run starts: constant-bank loads), the Gaussian index then advances
  // with j; only a thread that straddles two runs searches again.
  __device__ void span(uint64_t base, uint64_t& gi0, uint32_t& rem) const {
    int lo = 0, hi = map.n - 1;
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if ((uint64_t)map.jprefix[mid] <= base) lo = mid; else hi = mid - 1;
    }
    gi0 = (uint64_t)map.begin[lo] + (base - (uint64_t)map.jprefix[lo]);
    const uint64_t left = (uint64_t)map.jprefix[lo + 1] - base;
    rem = left < (uint64_t)SCAN_IPT ? (uint32_t)left : (uint32_t)SCAN_IPT;
  }
  __device__ void load_all(uint64_t base, uint64_t cnt, uint32_t (&v)[SCAN_IPT]) const {
    uint64_t gi0 = 0; uint32_t rem = 0;
    if (base < cnt) span(base, gi0, rem);
    static_assert(SCAN_IPT == 8, "two 16-byte loads per thread");
    if (rem == SCAN_IPT && base + SCAN_IPT <= cnt && (gi0 & 3) == 0) {     // the common case: eight consecutive, aligned counts
      const uint4 a = *reinterpret_cast<const uint4*>(tiles_touched + gi0), b = *reinterpret_cast<const uint4*>(tiles_touched + gi0 + 4);
      v[0] = a.x > 0; v[1] = a.y > 0; v[2] = a.z > 0; v[3] = a.w > 0; v[4] = b.x > 0; v[5] = b.y > 0; v[6] = b.z > 0; v[7] = b.w > 0;
      return;
    }
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) {
      v[k] = 0;
      if (base + k < cnt) v[k] = tiles_touched[(uint32_t)k < rem ? gi0 + k : map(base + k)] > 0 ? 1u : 0u;
    }
  }
  __device__ void store_all(uint64_t base, uint64_t cnt, const uint32_t (&v)[SCAN_IPT], uint32_t ex, uint32_t* hist) const {
    uint64_t gi0 = 0; uint32_t rem = 0;
    if (base < cnt) span(base, gi0, rem);
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) {
      if (base + k < cnt && v[k]) {
        const uint64_t i = (uint32_t)k < rem ? gi0 + k : map(base + k);
        const uint32_t key = __float_as_uint(depth[i]);
        ckeys[ex] = key; cvals[ex] = (uint32_t)i;
        vis_list[ex] = (uint32_t)i;      // the visible Gaussians in INDEX order (kept: the depth sort permutes cvals)
#pragma unroll
        for (int p = 0; p < 4; ++p) atomicAdd(&hist[p * 256 + ((key >> (8 * p)) & 255u)], 1u);
      }
      ex += v[k];
    }
  }
};
struct TouchedOp {  // step 3: offsets of each visible Gaussian's run of keys, depth order
  const uint32_t* tiles_touched; const uint32_t* cvals; uint32_t* offs;
  __device__ uint64_t count(const uint64_t* n_ptr) const { return *n_ptr; }
  __device__ void load_all(uint64_t base, uint64_t cnt, uint32_t (&v)[SCAN_IPT]) const {
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) v[k] = base + k < cnt ? tiles_touched[cvals[base + k]] : 0u;
  }
  __device__ void store_all(uint64_t base, uint64_t cnt, const uint32_t (&v)[SCAN_IPT], uint32_t ex, uint32_t*) const {
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) { if (base + k < cnt) offs[base + k] = ex; ex += v[k]; }
  }
};

template <class Op>
int scan_exclusive(splx_ctx* ctx, Op op, uint64_t capacity, const uint64_t* n_ptr, uint64_t* status, uint32_t* ticket,
                   uint64_t* total_out, uint64_t* clamp_out, uint64_t clamp_to) {
  uint32_t nb = (uint32_t)((capacity + SCAN_TILE - 1) / SCAN_TILE);
  if (nb == 0) return SPLX_OK;
  if (nb > PERSISTENT_CTAS) nb = PERSISTENT_CTAS;
  k_scan<Op><<<nb, SCAN_THREADS, 0, ctx->stream>>>(op, n_ptr, status, ticket, total_out, clamp_out, clamp_to);
  SPLX_LAUNCH_CHECK(ctx, "k_scan<TouchedOp>");
  return SPLX_OK;
}

// ------------------------------------------------- step 1: compaction of the visible Gaussians --
// Count -> scan -> scatter in three launches.  (It used to be ONE decoupled look-back scan: at city scale -- 40-50 M
// participating Gaussians per bucket, 13 % of them visible -- that kernel ran at 1 TB/s with its warps waiting at the
// barrier behind the one thread that walks back over the predecessors' status words, 0.35-0.42 ms per bucket; and it
// cleared the depth sort's look-back words for as many tiles as there are PARTICIPATING Gaussians, as many bytes as it
// read.)  Nothing here waits on another CTA: k_vis_count streams tiles_touched once (a count per SCAN_TILE elements),
// k_vis_offsets scans the counts in one CTA and publishes N_visible, k_vis_compact reads tiles_touched again, ranks
// inside the tile and scatters (depth bits, index), the index-ordered list, the four digit histograms of the depth sort,
// and clears the status words of the tiles the depth sort will really use.
__global__ void __launch_bounds__(SCAN_THREADS)
k_vis_count(const __grid_constant__ VisibleOp op, uint32_t* __restrict__ tile_counts) {
  __shared__ uint32_t sm[SCAN_THREADS / 32];
  const uint64_t n = op.n, ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  for (uint64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const uint64_t base = t * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_IPT;
    uint32_t v[SCAN_IPT], s = 0;
    op.load_all(base, n, v);
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) s += v[k];
    s = __reduce_add_sync(0xffffffffu, s);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
      uint32_t w = threadIdx.x < SCAN_THREADS / 32 ? sm[threadIdx.x] : 0u;
      w = __reduce_add_sync(0xffffffffu, w);
      if (threadIdx.x == 0) tile_counts[t] = w;
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(1024)
k_vis_offsets(uint32_t* __restrict__ tile_counts, uint64_t ntiles, uint64_t* __restrict__ n_visible) {
  __shared__ uint32_t sm[33];
  uint32_t running = 0;
  for (uint64_t b = 0; b < ntiles; b += 1024) {
    const uint64_t t = b + threadIdx.x;
    const uint32_t c = t < ntiles ? tile_counts[t] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(c, sm, total);
    if (t < ntiles) tile_counts[t] = running + ex;
    running += total;
  }
  if (threadIdx.x == 0) *n_visible = running;
}

__global__ void __launch_bounds__(SCAN_THREADS, 2)
k_vis_compact(const __grid_constant__ VisibleOp op, const uint32_t* __restrict__ tile_offsets, const uint64_t* __restrict__ n_visible,
              uint32_t* __restrict__ ghist, uint64_t* __restrict__ rstatus, size_t rstride) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_hist[4 * 256];
  for (int x = threadIdx.x; x < 4 * 256; x += SCAN_THREADS) s_hist[x] = 0;
  // look-back status words of the four passes of the depth sort: 256 per tile of RS_TILE visible Gaussians
  const uint64_t words = ((*n_visible + RS_TILE - 1) / RS_TILE) * 256;
  for (uint64_t x = (uint64_t)blockIdx.x * SCAN_THREADS + threadIdx.x; x < words; x += (uint64_t)gridDim.x * SCAN_THREADS) {
#pragma unroll
    for (int pass = 0; pass < 4; ++pass) rstatus[(size_t)pass * rstride + x] = 0;
  }
  __syncthreads();
  const uint64_t n = op.n, ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  for (uint64_t t = blockIdx.x; t < ntiles; t += gridDim.x) {
    const uint64_t base = t * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_IPT;
    uint32_t v[SCAN_IPT], s = 0;
    op.load_all(base, n, v);
#pragma unroll
    for (int k = 0; k < SCAN_IPT; ++k) s += v[k];
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(s, sm, total) + tile_offsets[t];
    if (total) op.store_all(base, n, v, ex, s_hist);
  }
  __syncthreads();
  for (int x = threadIdx.x; x < 4 * 256; x += SCAN_THREADS) { const uint32_t c = s_hist[x]; if (c) atomicAdd(&ghist[x], c); }
}

static int compact_visible(splx_ctx* ctx, const VisibleOp& op, uint32_t* tile_counts, uint64_t* n_visible, uint32_t* ghist,
                           uint64_t* rstatus, size_t rstride) {
  const uint64_t ntiles = (op.n + SCAN_TILE - 1) / SCAN_TILE;
  if (ntiles == 0) return SPLX_OK;
  const unsigned nb = (unsigned)(ntiles < 4 * SPLX_SM_COUNT ? ntiles : 4 * SPLX_SM_COUNT);
  k_vis_count<<<nb, SCAN_THREADS, 0, ctx->stream>>>(op, tile_counts);
  SPLX_LAUNCH_CHECK(ctx, "k_vis_count");
  k_vis_offsets<<<1, 1024, 0, ctx->stream>>>(tile_counts, ntiles, n_visible);
  SPLX_LAUNCH_CHECK(ctx, "k_vis_offsets");
  k_vis_compact<<<nb, SCAN_THREADS, 0, ctx->stream>>>(op, tile_counts, n_visible, ghist, rstatus, rstride);
  SPLX_LAUNCH_CHECK(ctx, "k_vis_compact");
  return SPLX_OK;
}

// ---------------------------------------------------------------------- LSD radix sort --
// "Onesweep" organisation: the digit histograms of ALL passes are counted in one read of the
// input (a histogram does not depend on the order), then each pass is ONE kernel: a tile ranks
// its 2048 keys (stable; digit peers found with MATCH.ANY), chains its per-digit counts to
// its predecessors by look-back (256 independent chains, one per thread) and scatters.
// Per item and pass: key+value read once and written once (24 B for 64-bit keys, 16 B for 32-bit).

struct PassPlan { int npass; int shift[MAX_PASSES]; int bits[MAX_PASSES]; };

static PassPlan plan_passes(int begin_bit, int end_bit, int max_bits = 8) {
  PassPlan p;
  const int total = end_bit - begin_bit;
  p.npass = (total + max_bits - 1) / max_bits;
  int shift = begin_bit;
  for (int i = 0; i < p.npass; ++i) {
    p.bits[i] = (total + p.npass - 1 - i) / p.npass;   // spread the bits evenly over the passes
    p.shift[i] = shift;
    shift += p.bits[i];
  }
  return p;
}

// The LAST pass of the slot sort writes the binning itself: its 32-bit items are (compact slot, position j in the
// depth-sorted list of visible Gaussians); the 64-bit key (true slot << 32 | depth bits of j) and the value (Gaussian
// index of j) are formed on the way out, from two arrays of N_visible entries that sit in L2.  The passes before it
// move 8 bytes per intersection instead of 12.
struct FinalOut {
  uint64_t* keys; uint32_t* vals;               // splx_binning.keys / vals
  const uint32_t* ckeys; const uint32_t* cvals; // depth bits / Gaussian index of the j-th visible Gaussian in depth order
  uint32_t ntiles;
  uint32_t skip[SPLX_MAX_K + 1];                // true slot = compact slot + skip[compact slot / ntiles]
  const uint32_t* inv;                          // or (renumbered open slots, k_slot_map): true slot = inv[sort slot]
};

// One tile of a radix pass (RS_TILE keys of one CTA): stable ranks by warp multisplit, the tile's keys reordered in
// shared memory, the per-digit prefix over the tiles by look-back, the scatter.  FULL: every one of the RS_TILE
// positions holds a key.  NB = number of digit values (256: 8-bit digits; 512: 9-bit digits, two per thread in the
// per-digit phases -- 17 or 18 slot bits then take two passes instead of three).
template <typename KeyT, bool FINAL, bool FULL, int NB>
__device__ __forceinline__ void radix_tile(const KeyT* __restrict__ kin, const uint32_t* __restrict__ vin, KeyT* __restrict__ kout,
                                           uint32_t* __restrict__ vout, uint64_t start, uint32_t nv, uint32_t t, int shift,
                                           int bits, uint32_t mask, uint64_t* status, const FinalOut& fin, uint32_t (*whist)[NB],
                                           uint32_t* dbase, const uint32_t* gbase, uint32_t* lbase, KeyT* skey, uint32_t* sval,
                                           uint32_t* sm) {
  constexpr int DPT = NB / RS_THREADS;      // digits per thread: thread x owns digits DPT x .. DPT x + DPT - 1
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned lt = (1u << lane) - 1u;
  // warp w owns the contiguous segment [w*256, +256) of the tile; iteration `it` covers 32 consecutive
  // positions, so (it, lane) is the input order and the ranks below are stable.
  const uint32_t seg = (uint32_t)warp * (32 * RS_IPT) + (uint32_t)lane;
  KeyT key[RS_IPT];
  uint32_t val[RS_IPT], dg[RS_IPT], rank[RS_IPT];
#pragma unroll
  for (int it = 0; it < RS_IPT; ++it) {
    const uint32_t o = seg + (uint32_t)it * 32;
    const bool valid = FULL || o < nv;
    key[it] = valid ? kin[start + o] : (KeyT)0;
    val[it] = valid ? vin[start + o] : 0u;
  }
#pragma unroll
  for (int it = 0; it < RS_IPT; ++it) {
    const bool valid = FULL || seg + (uint32_t)it * 32 < nv;
    const uint32_t d = (uint32_t)(key[it] >> shift) & mask;
    dg[it] = d;
    // lanes of the warp with this lane's digit (the invalid lanes of a ragged tile form a group of their own).  MATCH.ANY
    // against one vote per digit bit (6 instructions each): neutral while the slot passes had 5-6 bit digits, -7 % of
    // bin/sort at city scale once the renumbered slots made them 8-bit passes (sort, end of round 2)
    const unsigned peers = __match_any_sync(0xffffffffu, (FULL || valid) ? d : 0xffffffffu);
    uint32_t old = 0;
    const int leader = __ffs(peers) - 1;               // (an invalid lane: its own digit-0 group among the invalid ones; unused)
    if (valid && lane == leader) { old = whist[warp][d]; whist[warp][d] = old + __popc(peers); }
    old = __shfl_sync(0xffffffffu, old, leader & 31);
    rank[it] = old + __popc(peers & lt);
    __syncwarp();
  }
  __syncthreads();
  uint32_t run[DPT];   // per digit: exclusive prefix over the warps (left in whist), tile total
  uint32_t rsum = 0;
#pragma unroll
  for (int q = 0; q < DPT; ++q) {
    const int d = DPT * threadIdx.x + q;
    run[q] = 0;
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w) { const uint32_t c = whist[w][d]; whist[w][d] = run[q]; run[q] += c; }
    rsum += run[q];
  }
  {  // position of digit d's first key inside the tile, in digit order
    uint32_t tot;
    uint32_t ex = block_exclusive_scan(rsum, sm, tot);
#pragma unroll
    for (int q = 0; q < DPT; ++q) { lbase[DPT * threadIdx.x + q] = ex; ex += run[q]; }
  }
  __syncthreads();
  // the tile's keys go to shared memory in digit order, so that the scatter below writes runs of consecutive
  // addresses (one run per digit) instead of 2048 isolated items
#pragma unroll
  for (int it = 0; it < RS_IPT; ++it) {
    if (FULL || seg + (uint32_t)it * 32 < nv) {
      const uint32_t lp = lbase[dg[it]] + whist[warp][dg[it]] + rank[it];
      skey[lp] = key[it];
      sval[lp] = val[it];
    }
  }
  // chained prefix over the tiles (look-back), one chain per digit
#pragma unroll
  for (int q = 0; q < DPT; ++q) {
    const int d = DPT * threadIdx.x + q;
    uint64_t excl = 0;
    uint64_t* st = status + d;
    if (t == 0) st_status(st, ST_PREFIX | (uint64_t)run[q]);
    else excl = lookback<8>(st, t, NB, run[q]);
    dbase[d] = gbase[d] + (uint32_t)excl - lbase[d];      // global position = dbase[d] + position in the tile
  }
  __syncthreads();
#pragma unroll
  for (int it = 0; it < RS_IPT; ++it) {
    const uint32_t j = (uint32_t)it * RS_THREADS + threadIdx.x;
    if (FULL || j < nv) {
      const KeyT k = skey[j];
      const uint32_t d = (uint32_t)(k >> shift) & mask;
      const uint32_t pos = dbase[d] + j;
      if (FINAL) {
        const uint32_t cs = (uint32_t)k, jj = sval[j];
        const uint32_t slot = fin.inv ? __ldg(fin.inv + cs) : cs + fin.skip[cs / fin.ntiles];
        fin.keys[pos] = ((uint64_t)slot << 32) | __ldg(fin.ckeys + jj);
        fin.vals[pos] = __ldg(fin.cvals + jj);
      } else {
        kout[pos] = k;
        vout[pos] = sval[j];
      }
    }
  }
}

// Persistent: tiles are taken from the ticket counter in order, so every predecessor of a running tile has
// started and the look-back spin cannot wait on a CTA that was never scheduled.
template <typename KeyT, bool FINAL, int NB>
__global__ void __launch_bounds__(RS_THREADS, 4)
k_radix_pass(const KeyT* __restrict__ kin, const uint32_t* __restrict__ vin, KeyT* __restrict__ kout,
             uint32_t* __restrict__ vout, const uint64_t* n_ptr, const uint32_t* __restrict__ ghist /*[NB] of this pass*/,
             uint64_t* status /*[tiles][NB]*/, uint32_t* ticket, int shift, int bits, const __grid_constant__ FinalOut fin) {
  constexpr int DPT = NB / RS_THREADS;
  __shared__ uint32_t whist[RS_WARPS][NB];
  __shared__ uint32_t dbase[NB];
  __shared__ uint32_t gbase[NB];
  __shared__ uint32_t lbase[NB];
  __shared__ KeyT skey[RS_TILE];
  __shared__ uint32_t sval[RS_TILE];
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_tile;
  const uint64_t n = *n_ptr;
  const uint64_t ntiles = (n + RS_TILE - 1) / RS_TILE;
  if (blockIdx.x >= ntiles) return;
  const uint32_t mask = (1u << bits) - 1u;
  {  // exclusive scan of the global digit histogram = first output position of each digit (once per CTA)
    uint32_t g[DPT], gs = 0, tot;
#pragma unroll
    for (int q = 0; q < DPT; ++q) { g[q] = ghist[DPT * threadIdx.x + q]; gs += g[q]; }
    uint32_t ex = block_exclusive_scan(gs, sm, tot);
#pragma unroll
    for (int q = 0; q < DPT; ++q) { gbase[DPT * threadIdx.x + q] = ex; ex += g[q]; }
  }
  for (;;) {
    __syncthreads();                       // the previous round no longer reads whist / dbase / s_tile
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < RS_WARPS; ++w)
#pragma unroll
      for (int q = 0; q < DPT; ++q) whist[w][DPT * threadIdx.x + q] = 0;
    __syncthreads();
    const uint32_t t = s_tile;
    if (t >= ntiles) return;
    const uint64_t start = (uint64_t)t * RS_TILE;
    const uint32_t nv = (uint32_t)((n - start) < (uint64_t)RS_TILE ? (n - start) : (uint64_t)RS_TILE);
    // the kernel is bound by instruction issue (ncu, city_100M: 62 % issue slots, DRAM 13 %): a full tile -- all but the
    // last one -- takes the copy of the body without the per-item range checks
    if (nv == RS_TILE)
      radix_tile<KeyT, FINAL, true, NB>(kin, vin, kout, vout, start, nv, t, shift, bits, mask, status, fin, whist, dbase, gbase, lbase, skey, sval, sm);
    else
      radix_tile<KeyT, FINAL, false, NB>(kin, vin, kout, vout, start, nv, t, shift, bits, mask, status, fin, whist, dbase, gbase, lbase, skey, sval, sm);
  }
}

// Sorts bits [begin_bit, end_bit) in passes of <= log2(NB) bits.  Input in (ka, va); buffers alternate
// (result in (ka, va) after an even number of passes, (kb, vb) after an odd number).
// ghist: [MAX_PASSES][NB] u32 counted by the producer of the keys, which also cleared status: [npass][tiles][NB] u64.
template <typename KeyT, int NB>
int radix_sort(splx_ctx* ctx, KeyT* ka, uint32_t* va, KeyT* kb, uint32_t* vb, uint64_t capacity,
               const uint64_t* n_ptr, int begin_bit, int end_bit, uint32_t* ghist, uint64_t* status, uint32_t* tickets,
               size_t stride_words = 0 /* status words per pass; 0 = tiles(capacity) * NB */,
               const FinalOut* fin = nullptr /* the last pass writes the binning (see FinalOut) */) {
  const uint32_t ntiles_cap = (uint32_t)((capacity + RS_TILE - 1) / RS_TILE);
  if (ntiles_cap == 0) return SPLX_OK;
  const uint32_t nblocks = ntiles_cap < PERSISTENT_CTAS ? ntiles_cap : PERSISTENT_CTAS;
  const size_t stride = stride_words ? stride_words : (size_t)ntiles_cap * NB;     // status words per pass
  const PassPlan plan = plan_passes(begin_bit, end_bit, NB == 256 ? 8 : 9);
  FinalOut none;
  memset(&none, 0, sizeof none);
  for (int p = 0; p < plan.npass; ++p) {
#define PASS_ARGS(F) ka, va, kb, vb, n_ptr, ghist + NB * p, status + (size_t)p * stride, tickets + p, plan.shift[p], plan.bits[p], F
    if (fin && p + 1 == plan.npass) k_radix_pass<KeyT, true, NB><<<nblocks, RS_THREADS, 0, ctx->stream>>>(PASS_ARGS(*fin));
    else k_radix_pass<KeyT, false, NB><<<nblocks, RS_THREADS, 0, ctx->stream>>>(PASS_ARGS(none));
#undef PASS_ARGS
    SPLX_LAUNCH_CHECK(ctx, "k_radix_pass");
    KeyT* tk = ka; ka = kb; kb = tk;
    uint32_t* tv = va; va = vb; vb = tv;
  }
  return SPLX_OK;
}

// ------------------------------------------------------------------------- key emission --
// Two kernels hand out the work in two ways; both are launched and the device-side counts decide which one works
// (the other returns at once -- the host does not know M):
//  * k_emit_keys, by Gaussian (a warp writes the 32 adjacent runs of its 32 Gaussians): cheapest when footprints are
//    small and alike (aerial views: 3-12 tiles per Gaussian);
//  * k_emit_keys_lb, by output position: when the mean footprint is large the sizes are very unequal as well
//    (street-level views: a few Gaussians next to each other at the head of the depth order cover thousands of tiles
//    each) and the first scheme leaves a handful of CTAs with all the work (1.5 ms on street_10M against 0.2 ms).
__device__ __forceinline__ bool emit_by_output(const Counters* cnt) { return cnt->m_total > 16 * cnt->n_visible; }

// Cross-boundary per-ray filtering (L474-L476): a removed (Gaussian, tile) pair is emitted under the slot number
// `nslots` (one past the last real slot), so the slot sort carries it behind every list and k_tile_ranges never
// gives it a range; the rectangle arithmetic of the emission stays as it is.
struct CrossEmit {
  const uint64_t* mask;          // nullptr = no filtering
  const uint8_t* tile_state;
  const uint32_t* cmap;          // nullptr, or the renumbering of the OPEN slots (k_slot_map): sort slot = cmap[true slot]
  uint32_t ntiles, nslots;
  float zlo[SPLX_MAX_K], zhi[SPLX_MAX_K];
  signed char view[SPLX_MAX_K];
};

// F_i: the partitions s whose visible tiles lose Gaussian i (partition k, depth d): i in Q_cross(k, s), same view,
// d in D^k ^ D^s.
__device__ __forceinline__ uint64_t cross_filter(const CrossEmit& cx, uint32_t i, int k, float d) {
  uint64_t m = cx.mask[i], F = 0;
  while (m) {
    const int s = __ffsll((long long)m) - 1;
    m &= m - 1;
    if (cx.view[s] == cx.view[k] && d >= fmaxf(cx.zlo[k], cx.zlo[s]) && d <= fminf(cx.zhi[k], cx.zhi[s])) F |= 1ull << s;
  }
  return F;
}

// p in Omega^s for some s of F
__device__ __forceinline__ bool cross_removed(const CrossEmit& cx, uint64_t F, uint32_t tile) {
  while (F) {
    const int s = __ffsll((long long)F) - 1;
    F &= F - 1;
    if (!cx.tile_state || !(cx.tile_state[(size_t)s * cx.ntiles + tile] & SPLX_TILE_INVISIBLE)) return true;
  }
  return false;
}

template <bool FILTER>     // FILTER: cross-boundary per-ray filtering on (cx.mask != nullptr)
__global__ void __launch_bounds__(256)
k_emit_keys(const float* __restrict__ means2d, const int32_t* __restrict__ radius,
            const uint32_t* __restrict__ ckeys, const uint32_t* __restrict__ cvals,
            const uint32_t* __restrict__ offs, const Counters* cnt, PartOffs parts, int TX, int TY,
            uint64_t capacity, uint32_t* __restrict__ skeys, uint32_t* __restrict__ spay, PassPlan plan,
            uint32_t* __restrict__ ghist, uint64_t* __restrict__ rstatus, size_t rstride,
            const __grid_constant__ CrossEmit cx) {
  if (emit_by_output(cnt) || (cnt->m_total >> 32)) return;   // M >= 2^32: the 32-bit offsets have wrapped, nothing is emitted
  // The producer of the keys also counts the digit histograms of the slot sort (shared atomics, one flush per
  // CTA) and clears the look-back status words of the tiles the M keys will occupy: no histogram kernel.
  __shared__ uint32_t s_hist[MAX_PASSES * SLOT_NB];
  for (int x = threadIdx.x; x < MAX_PASSES * SLOT_NB; x += blockDim.x) s_hist[x] = 0;
  {
    const uint64_t words = ((cnt->m_sorted + RS_TILE - 1) / RS_TILE) * SLOT_NB;
    for (int p = 0; p < plan.npass; ++p)
      for (uint64_t x = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; x < words; x += (uint64_t)gridDim.x * blockDim.x)
        rstatus[(size_t)p * rstride + x] = 0;
  }
  __syncthreads();
  const uint64_t nvis = cnt->n_visible;
  const int lane = threadIdx.x & 31;
  // grid-stride over blocks of 256 visible Gaussians (the grid is sized for the machine; nvis lives on the device)
  for (uint64_t base = (uint64_t)blockIdx.x * blockDim.x; base < nvis; base += (uint64_t)gridDim.x * blockDim.x) {
  const uint64_t j = base + threadIdx.x;
  int x0 = 0, y0 = 0, w = 0, tt = 0;
  uint32_t i = 0, o = 0, slot0 = 0;
  uint64_t F = 0;
  if (j < nvis) {
    i = cvals[j]; o = offs[j];
    const float2 m = *reinterpret_cast<const float2*>(means2d + 2 * (uint64_t)i);
    int x1, y1;
    tile_rect(m.x, m.y, radius[i], TX, TY, x0, y0, x1, y1);
    w = x1 - x0; tt = w * (y1 - y0);
    int lo = 0, hi = parts.K - 1;  // partition of Gaussian i: last k with off[k] <= i
    while (lo < hi) {
      const int mid = (lo + hi + 1) >> 1;
      if (parts.off[mid] <= (int64_t)i) lo = mid; else hi = mid - 1;
    }
    slot0 = (uint32_t)(cx.cmap ? lo : (int)parts.rank[lo]) * (uint32_t)(TX * TY);      // compact slot (see PartOffs), or the true one
    if (FILTER) F = cross_filter(cx, i, lo, __uint_as_float(ckeys[j]));
  }
  // The 32 runs of a warp are adjacent in the output (offs is the running sum of tiles_touched in this very
  // order), so the warp writes its whole range [o_0, o_0 + T) cooperatively: lane l produces output slot
  // s0 + l, finds the owning Gaussian by a binary search over the lanes' run starts (5 shuffles) and fetches its
  // rectangle (6 shuffles).  Every store instruction covers 32 consecutive keys / values.
  uint32_t pre = (uint32_t)tt;                      // exclusive prefix of tt over the warp
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, pre, d); if (lane >= d) pre += v; }
  const uint32_t T = __shfl_sync(0xffffffffu, pre, 31);
  pre -= (uint32_t)tt;
  const uint32_t o0 = __shfl_sync(0xffffffffu, o, 0);
  for (uint32_t s0 = 0; s0 < T; s0 += 32) {
    const uint32_t sidx = s0 + lane;
    int own = 0;
#pragma unroll
    for (int step = 16; step >= 1; step >>= 1) {
      const int cand = own + step;
      const uint32_t pc = __shfl_sync(0xffffffffu, pre, cand & 31);
      if (cand < 32 && pc <= sidx) own = cand;
    }
    const uint32_t t = sidx - __shfl_sync(0xffffffffu, pre, own);
    const int sx0 = __shfl_sync(0xffffffffu, x0, own), sy0 = __shfl_sync(0xffffffffu, y0, own);
    const int sw = __shfl_sync(0xffffffffu, w, own);
    const uint32_t sj = (uint32_t)base + (uint32_t)(threadIdx.x & ~31) + (uint32_t)own;     // position in the depth-sorted list
    const uint32_t ss = __shfl_sync(0xffffffffu, slot0, own);
    const uint64_t pos = (uint64_t)o0 + sidx;
    uint64_t sF = 0;
    if (FILTER) sF = __shfl_sync(0xffffffffu, F, own);
    if (sidx < T && pos < capacity) {
      const uint32_t ty = t / (uint32_t)sw;
      const uint32_t tile = (uint32_t)((sy0 + (int)ty) * TX + sx0 + (int)(t - ty * (uint32_t)sw));
      uint32_t slot = ss + tile;
      if (cx.cmap) slot = __ldg(cx.cmap + slot);
      if (FILTER && sF && cross_removed(cx, sF, tile)) slot = cx.nslots;
      skeys[pos] = slot;
      spay[pos] = sj;
      for (int p = 0; p < plan.npass; ++p)
        atomicAdd(&s_hist[p * SLOT_NB + ((slot >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u))], 1u);
    }
  }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < plan.npass * SLOT_NB; x += blockDim.x) { const uint32_t c = s_hist[x]; if (c) atomicAdd(&ghist[x], c); }
}

template <bool FILTER>
__global__ void __launch_bounds__(256)
k_emit_keys_lb(const float* __restrict__ means2d, const int32_t* __restrict__ radius,
            const uint32_t* __restrict__ ckeys, const uint32_t* __restrict__ cvals,
            const uint32_t* __restrict__ offs, const Counters* cnt, PartOffs parts, int TX, int TY,
            uint64_t capacity, uint32_t* __restrict__ skeys, uint32_t* __restrict__ spay, PassPlan plan,
            uint32_t* __restrict__ ghist, uint64_t* __restrict__ rstatus, size_t rstride,
            const __grid_constant__ CrossEmit cx) {
  if (!emit_by_output(cnt) || (cnt->m_total >> 32)) return;
  // The producer of the keys also counts the digit histograms of the slot sort (shared atomics, one flush per
  // CTA) and clears the look-back status words of the tiles the M keys will occupy: no histogram kernel.
  __shared__ uint32_t s_hist[MAX_PASSES * SLOT_NB];
  for (int x = threadIdx.x; x < MAX_PASSES * SLOT_NB; x += blockDim.x) s_hist[x] = 0;
  {
    const uint64_t words = ((cnt->m_sorted + RS_TILE - 1) / RS_TILE) * SLOT_NB;
    for (int p = 0; p < plan.npass; ++p)
      for (uint64_t x = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; x < words; x += (uint64_t)gridDim.x * blockDim.x)
        rstatus[(size_t)p * rstride + x] = 0;
  }
  __syncthreads();
  // Load-balanced by OUTPUT position: a CTA produces tiles of EK_TILE consecutive keys, whatever the sizes of the
  // footprints they belong to (street-level views put a few Gaussians that cover thousands of tiles next to each
  // other at the head of the depth order: partitioning by Gaussian left a handful of CTAs with all the work,
  // 1.5 ms on street_10M).  Per tile: a 256-ary search over offs finds the first owner, the owners' run starts and
  // rectangles are staged in shared memory, every thread places EK_IPT keys by a binary search over the staged starts.
  constexpr int EK_TILE = 1024, EK_IPT = EK_TILE / 256;
  __shared__ uint32_t s_off[EK_TILE + 1], s_xy[EK_TILE + 1], s_w[EK_TILE + 1], s_slot0[EK_TILE + 1];
  __shared__ uint64_t s_F[FILTER ? EK_TILE + 1 : 1];
  __shared__ uint32_t s_nown;
  const uint64_t nvis = cnt->n_visible;
  const uint64_t m = cnt->m_sorted;                       // min(M, capacity): positions beyond the capacity are dropped
  for (uint64_t begin = (uint64_t)blockIdx.x * EK_TILE; begin < m; begin += (uint64_t)gridDim.x * EK_TILE) {
    const uint64_t end = begin + EK_TILE < m ? begin + EK_TILE : m;
    // last j with offs[j] <= begin (offs is strictly increasing, offs[0] == 0)
    uint64_t lo = 0, hi = nvis;
    while (hi - lo > 1) {
      const uint64_t step = (hi - lo + 255) / 256;
      const uint64_t pidx = lo + (uint64_t)threadIdx.x * step;
      const bool ok = pidx < hi && (uint64_t)offs[pidx] <= begin;
      const int c = __syncthreads_count(ok);             // the trues are a prefix; thread 0 is always true
      lo = lo + (uint64_t)(c - 1) * step;
      hi = lo + step < hi ? lo + step : hi;
    }
    const uint64_t j0 = lo;
    if (threadIdx.x == 0) s_nown = 0;
    __syncthreads();
    // stage the owners j0, j0 + 1, ... whose runs start before `end` (at most EK_TILE + 1 of them)
    for (int q = threadIdx.x; q <= EK_TILE; q += 256) {
      const uint64_t j = j0 + q;
      uint32_t o = 0xffffffffu;
      if (j < nvis) o = offs[j];
      if (j < nvis && (uint64_t)o < end) {
        const uint32_t i = cvals[j];
        const float2 mm = *reinterpret_cast<const float2*>(means2d + 2 * (uint64_t)i);
        int x0, y0, x1, y1;
        tile_rect(mm.x, mm.y, radius[i], TX, TY, x0, y0, x1, y1);
        int plo = 0, phi = parts.K - 1;                   // partition of Gaussian i: last k with off[k] <= i
        while (plo < phi) {
          const int mid = (plo + phi + 1) >> 1;
          if (parts.off[mid] <= (int64_t)i) plo = mid; else phi = mid - 1;
        }
        s_off[q] = o; s_xy[q] = ((uint32_t)y0 << 16) | (uint32_t)x0; s_w[q] = (uint32_t)(x1 - x0);
        s_slot0[q] = (uint32_t)(cx.cmap ? plo : (int)parts.rank[plo]) * (uint32_t)(TX * TY);
        if (FILTER) s_F[q] = cross_filter(cx, i, plo, __uint_as_float(ckeys[j]));
        atomicMax(&s_nown, (uint32_t)q + 1);
      }
    }
    __syncthreads();
    const uint32_t nown = s_nown;
#pragma unroll
    for (int k = 0; k < EK_IPT; ++k) {
      const uint64_t pos = begin + (uint64_t)k * 256 + threadIdx.x;
      if (pos < end) {
        uint32_t ql = 0, qh = nown - 1;                   // last staged owner whose run starts at or before pos
        while (ql < qh) {
          const uint32_t mid = (ql + qh + 1) >> 1;
          if ((uint64_t)s_off[mid] <= pos) ql = mid; else qh = mid - 1;
        }
        const uint32_t t = (uint32_t)(pos - s_off[ql]), w = s_w[ql], xy = s_xy[ql];
        const uint32_t ty = t / w;
        const uint32_t tile = ((xy >> 16) + ty) * (uint32_t)TX + (xy & 0xffffu) + (t - ty * w);
        uint32_t slot = s_slot0[ql] + tile;
        if (cx.cmap) slot = __ldg(cx.cmap + slot);
        if (FILTER) { const uint64_t F = s_F[ql]; if (F && cross_removed(cx, F, tile)) slot = cx.nslots; }
        skeys[pos] = slot;
        spay[pos] = (uint32_t)j0 + ql;                    // position of the owner in the depth-sorted list
        for (int p = 0; p < plan.npass; ++p)
          atomicAdd(&s_hist[p * SLOT_NB + ((slot >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u))], 1u);
      }
    }
    __syncthreads();
  }
  __syncthreads();
  for (int x = threadIdx.x; x < plan.npass * SLOT_NB; x += blockDim.x) { const uint32_t c = s_hist[x]; if (c) atomicAdd(&ghist[x], c); }
}

// Renumbering of the OPEN slots (splx_plan.open_slots > 0: the caller vouches that a slot whose state has
// SPLX_TILE_INVISIBLE holds no key -- the conservative regions of reading s21).  A city view leaves 85-90 % of the
// (partition, tile) slots invisible, so the open ones need 16 bits where all slots of the participating partitions need
// 17 or 18: two radix passes over the intersections instead of three.  cmap[s] = number of open slot s in slot order
// (monotone: the sort order is unchanged); every other slot -> cap + 1, carried behind every list and counted by
// k_tile_ranges (num_intersections[1]); cap itself = the pairs removed by the cross-boundary filter.  inv = the way back.
// One CTA: 32 slots per thread and round, K * tiles <= 2 M slots.
__global__ void __launch_bounds__(1024)
k_slot_map(const uint8_t* __restrict__ state, const __grid_constant__ PartView pv, uint32_t ntiles, uint32_t nslots, uint32_t cap,
           uint32_t* __restrict__ cmap, uint32_t* __restrict__ inv) {
  __shared__ uint32_t sm[33];
  uint32_t running = 0;
  for (uint32_t b = 0; b < nslots; b += 1024 * 32) {
    const uint32_t s0 = b + threadIdx.x * 32;
    uint32_t open = 0;
    if (s0 < nslots) {
      uint32_t w[8];
      if (s0 + 32 <= nslots) {
        const uint4 a = *reinterpret_cast<const uint4*>(state + s0), c = *reinterpret_cast<const uint4*>(state + s0 + 16);
        w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w; w[4] = c.x; w[5] = c.y; w[6] = c.z; w[7] = c.w;
      } else {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          w[q] = 0xffffffffu;
          for (int c = 0; c < 4; ++c) if (s0 + 4 * q + c < nslots) w[q] = (w[q] & ~(0xffu << (8 * c))) | ((uint32_t)state[s0 + 4 * q + c] << (8 * c));
        }
      }
#pragma unroll
      for (int k = 0; k < 32; ++k) {
        const uint32_t s = s0 + k;
        const bool inv_bit = (w[k >> 2] >> (8 * (k & 3))) & SPLX_TILE_INVISIBLE;
        if (s < nslots && !inv_bit && pv.v[s / ntiles] >= 0) open |= 1u << k;
      }
    }
    uint32_t total;
    uint32_t ex = block_exclusive_scan((uint32_t)__popc(open), sm, total) + running;
    if (s0 < nslots) {
#pragma unroll
      for (int k = 0; k < 32; ++k) {
        const uint32_t s = s0 + k;
        if (s >= nslots) break;
        uint32_t c = cap + 1;
        if ((open >> k) & 1u) { if (ex < cap) { c = ex; inv[ex] = s; } ++ex; }
        cmap[s] = c;
      }
    }
    running += total;
  }
  if (threadIdx.x == 0) { inv[cap] = nslots; inv[cap + 1] = nslots + 1; }
}

// Four consecutive keys per thread (two 16-byte loads; the neighbours of the group's ends come from the adjacent lanes,
// from memory at the warp's ends); only a key that opens or closes a list looks at the tile state and writes -- the
// one-key-per-thread version read three keys and a state byte for every intersection and sat on their latency
// (ncu r02c, city_10M: 28 warps waiting on the long scoreboard per issued instruction).
__global__ void __launch_bounds__(256)
k_tile_ranges(const uint64_t* __restrict__ keys, const Counters* cnt, const uint8_t* __restrict__ tile_state,
              uint32_t* __restrict__ ranges, uint64_t* __restrict__ m_out, uint32_t nslots, bool filtered) {
  const uint64_t m = cnt->m_sorted;
  // M as published: the unfiltered count (it is what the capacity must hold) unless the filter ran and everything
  // fitted -- then the number of pairs kept, written by the thread that sees the first removed pair (or the last
  // key, when nothing was removed).
  const bool count_kept = filtered && cnt->m_total == m && m > 0;
  if (blockIdx.x == 0 && threadIdx.x == 0 && !count_kept) *m_out = cnt->m_total;
  const int lane = threadIdx.x & 31;
  const uint64_t groups = (m + 3) / 4;
  // whole warps stay in the loop together (the shuffles below): the bound is rounded up to a multiple of 32 groups
  for (uint64_t g0 = (uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); g0 < groups; g0 += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t j0 = 4 * (g0 + lane);
    uint32_t s[4];
    if (j0 + 4 <= m) {
      const ulonglong2 a = *reinterpret_cast<const ulonglong2*>(keys + j0), c = *reinterpret_cast<const ulonglong2*>(keys + j0 + 2);
      s[0] = (uint32_t)(a.x >> 32); s[1] = (uint32_t)(a.y >> 32); s[2] = (uint32_t)(c.x >> 32); s[3] = (uint32_t)(c.y >> 32);
    } else {
#pragma unroll
      for (int q = 0; q < 4; ++q) s[q] = j0 + q < m ? (uint32_t)(keys[j0 + q] >> 32) : 0xffffffffu;
    }
    uint32_t prev = __shfl_up_sync(0xffffffffu, s[3], 1), next = __shfl_down_sync(0xffffffffu, s[0], 1);
    if (lane == 0) prev = (j0 > 0 && j0 <= m) ? (uint32_t)(keys[j0 - 1] >> 32) : 0xffffffffu;
    if (lane == 31) next = j0 + 4 < m ? (uint32_t)(keys[j0 + 4] >> 32) : 0xffffffffu;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint64_t j = j0 + q;
      if (j >= m) break;
      const uint32_t sj = s[q], sp = q ? s[q - 1] : prev, sn = q < 3 ? s[q + 1] : next;
      const bool first = j == 0 || sp != sj, last = j + 1 == m || sn != sj;
      if (sj >= nslots) {           // removed pairs: behind every list
        if (count_kept && (j == 0 || sp < nslots)) *m_out = j;
        // renumbered open slots (splx_plan.open_slots): a key that landed in a slot the caller declared INVISIBLE
        if (sj == nslots + 1) atomicAdd((unsigned long long*)(m_out + 1), 1ull);
        continue;
      }
      if (count_kept && j + 1 == m) *m_out = m;
      if (!first && !last) continue;
      if (tile_state && tile_state[sj]) {           // a skipped (partition, tile) slot keeps the empty range (0,0)
        // a NON-EMPTY list dropped on geometric grounds: the caller's regions were not conservative (splx_footprint_margin)
        if ((tile_state[sj] & SPLX_TILE_INVISIBLE) && first) atomicAdd((unsigned long long*)(m_out + 1), 1ull);
        continue;
      }
      if (first) ranges[2 * (uint64_t)sj] = (uint32_t)j;
      if (last) ranges[2 * (uint64_t)sj + 1] = (uint32_t)(j + 1);
    }
  }
}

// ---- slots by descending list length (splx_binning.slot_order) ----------------------------------------------
// The blend kernels' CTAs differ in work by two orders of magnitude (list lengths); handed out in tile order, a long
// list that starts late is the tail of the launch.  Longest-first needs no exact sort: 1024 log-linear length classes
// (5 mantissa bits: 3 % resolution), a histogram, a descending scan and a scatter with atomic cursors.
constexpr int ORD_CLASSES = 1024;
__device__ __forceinline__ uint32_t length_class(uint32_t len) {   // len >= 1; monotonic in len
  const int e = 31 - __clz(len);
  const uint32_t m = e >= 5 ? (len >> (e - 5)) & 31u : (len << (5 - e)) & 31u;
  return (uint32_t)e * 32u + m;
}

__global__ void __launch_bounds__(256)
k_order_hist(const uint32_t* __restrict__ ranges, uint32_t nslots, uint32_t* __restrict__ hist) {
  __shared__ uint32_t s_h[ORD_CLASSES];
  for (int x = threadIdx.x; x < ORD_CLASSES; x += 256) s_h[x] = 0;
  __syncthreads();
  for (uint32_t s = blockIdx.x * 256 + threadIdx.x; s < nslots; s += gridDim.x * 256) {
    const uint2 r = reinterpret_cast<const uint2*>(ranges)[s];
    if (r.y > r.x) atomicAdd(&s_h[length_class(r.y - r.x)], 1u);
  }
  __syncthreads();
  for (int x = threadIdx.x; x < ORD_CLASSES; x += 256) if (s_h[x]) atomicAdd(&hist[x], s_h[x]);
}

// One CTA: class c (thread t = 1023 - c, so that the scan runs from the longest class down) gets the first output
// position of its slots; the total is the number of live slots.
__global__ void __launch_bounds__(ORD_CLASSES)
k_order_scan(uint32_t* __restrict__ hist, uint32_t* __restrict__ n_live) {
  __shared__ uint32_t s_w[32];
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  const uint32_t c = hist[ORD_CLASSES - 1 - t];
  uint32_t inc = c;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
  if (lane == 31) s_w[w] = inc;
  __syncthreads();
  if (w == 0) {
    uint32_t x = s_w[lane];
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += v; }
    s_w[lane] = x;
  }
  __syncthreads();
  const uint32_t before = (w ? s_w[w - 1] : 0u) + inc - c;
  hist[ORD_CLASSES - 1 - t] = before;
  if (t == ORD_CLASSES - 1) *n_live = before + c;
}

__global__ void __launch_bounds__(256)
k_order_scatter(const uint32_t* __restrict__ ranges, uint32_t nslots, uint32_t* __restrict__ cursor, uint32_t* __restrict__ order) {
  for (uint32_t s = blockIdx.x * 256 + threadIdx.x; s < nslots; s += gridDim.x * 256) {
    const uint2 r = reinterpret_cast<const uint2*>(ranges)[s];
    if (r.y > r.x) order[atomicAdd(&cursor[length_class(r.y - r.x)], 1u)] = s;
  }
}

__global__ void k_publish_m(const Counters* cnt, uint64_t* out) { *out = cnt->m_total; }

// Workspace: a small zero-initialised control region (counters, tickets, digit histograms, the scans' status
// words: one memset per call), the radix passes' status words (cleared on the device, only as far as the
// actual counts reach) and the sort buffers.
struct Layout {
  size_t counters, ghist_d, ghist_s, st_scan_v, st_scan_t, st_depth, st_slot, zero_bytes;
  size_t ckeys_a, cvals_a, ckeys_b, cvals_b, offs, vis_list, pairs_tmp, total;
};

static int slot_bits(int K, int TX, int TY) {
  const uint64_t slots = (uint64_t)K * TX * TY;
  int b = 1;
  while (((uint64_t)1 << b) <= slots) ++b;   // the values 0..slots: `slots` itself marks a filtered pair
  return b;
}

static Layout make_layout(int64_t n, uint64_t capacity, int sbits) {
  Layout L;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  const size_t tiles_m = ((size_t)capacity + RS_TILE - 1) / RS_TILE;
  const size_t scan_n = ((size_t)n + SCAN_TILE - 1) / SCAN_TILE;
  L.counters = take(sizeof(Counters));
  L.ghist_d = take(MAX_PASSES * 256 * 4);
  L.ghist_s = take(MAX_PASSES * SLOT_NB * 4);
  L.st_scan_v = take(scan_n * 8);
  L.st_scan_t = take(scan_n * 8);
  L.zero_bytes = off;
  L.st_depth = take(4 * scan_n * SCAN_RS * 256 * 8);                          // cleared by the compaction scan, whole scan tiles
  L.st_slot = take((size_t)((sbits + SLOT_BITS - 1) / SLOT_BITS) * tiles_m * SLOT_NB * 8);
  L.ckeys_a = take((size_t)n * 4); L.cvals_a = take((size_t)n * 4);
  L.ckeys_b = take((size_t)n * 4); L.cvals_b = take((size_t)n * 4);
  L.offs = take((size_t)n * 4);
  L.vis_list = take((size_t)n * 4);
  L.pairs_tmp = take((size_t)capacity * 8);      // (compact slot, depth-order position) pairs: two uint32[capacity]
  L.total = off;
  return L;
}

}  // namespace

size_t bin_sort_ws_bytes(int64_t n, uint64_t capacity, int K, int TX, int TY) {
  return make_layout(n, capacity, slot_bits(K, TX, TY)).total;
}

int bin_sort_visible(const void* ws, int64_t n, uint64_t capacity, int K, int TX, int TY, const uint32_t** list,
                     const uint64_t** count) {
  const Layout L = make_layout(n, capacity, slot_bits(K, TX, TY));
  const char* base = (const char*)ws;
  *list = (const uint32_t*)(base + L.vis_list);       // index order: consecutive rows of the list are close in memory
  *count = &((const Counters*)(base + L.counters))->n_visible;
  return SPLX_OK;
}

// The Gaussians of the visible list that received a 2-D gradient: a visible Gaussian that no pixel blended (hidden
// behind opaque surfaces: about half of the visible ones on a city view) has an all-zero g2d row and therefore -- the
// projection backward is linear in that row -- a zero gradient.  Compacted here (a vote and one atomic per warp; the
// order inside the list does not matter to its consumer) so that the projection backward runs on full blocks of rows
// that have work: skipping them INSIDE that kernel left its blocks as slow as before (the block's time is the
// latency of its phases, not the number of live rows: 4.53 -> 4.40 ms at city_100M).
__global__ void __launch_bounds__(256)
k_gradient_rows(const float* __restrict__ g2d, const uint32_t* __restrict__ vlist, const uint64_t* __restrict__ nvis_ptr,
                uint32_t* __restrict__ rows, unsigned long long* __restrict__ n_rows) {
  constexpr int U = 4;      // list entries per thread and trip: their dependent loads (entry -> row) overlap
  const uint64_t nvis = *nvis_ptr;
  const int lane = threadIdx.x & 31;
  const uint64_t warp0 = ((uint64_t)blockIdx.x * blockDim.x + (threadIdx.x & ~31u)) * U;
  for (uint64_t j0 = warp0; j0 < nvis; j0 += (uint64_t)gridDim.x * blockDim.x * U) {
    uint32_t i[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { const uint64_t j = j0 + 32 * u + lane; i[u] = j < nvis ? vlist[j] : 0xffffffffu; }
    bool nz[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      nz[u] = false;
      if (i[u] != 0xffffffffu) {
        const float* gp = g2d + (int64_t)SPLX_G2D_STRIDE * i[u];
        const float4 a = *reinterpret_cast<const float4*>(gp), b = *reinterpret_cast<const float4*>(gp + 4);
        const float c = gp[8];
        nz[u] = a.x != 0.f || a.y != 0.f || a.z != 0.f || a.w != 0.f || b.x != 0.f || b.y != 0.f || b.z != 0.f || b.w != 0.f ||
                c != 0.f;
      }
    }
    unsigned bal[U];
    int total = 0;
#pragma unroll
    for (int u = 0; u < U; ++u) { bal[u] = __ballot_sync(0xffffffffu, nz[u]); total += __popc(bal[u]); }
    unsigned long long base = 0;
    if (lane == 0 && total) base = atomicAdd(n_rows, (unsigned long long)total);
    base = __shfl_sync(0xffffffffu, base, 0);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (nz[u]) rows[base + __popc(bal[u] & ((1u << lane) - 1u))] = i[u];
      base += __popc(bal[u]);
    }
  }
}

int launch_gradient_rows(splx_ctx* ctx, void* ws, int64_t n, uint64_t capacity, int K, int TX, int TY, const float* g2d,
                         const uint32_t** rows, const uint64_t** num_rows) {
  const Layout L = make_layout(n, capacity, slot_bits(K, TX, TY));
  char* base = (char*)ws;
  Counters* cnt = (Counters*)(base + L.counters);
  uint32_t* out = (uint32_t*)(base + L.cvals_b);      // scratch of the depth sort, free once the binning is built
  SPLX_CUDA_OK(ctx, cudaMemsetAsync(&cnt->n_rows, 0, sizeof(uint64_t), ctx->stream));
  k_gradient_rows<<<SPLX_SM_COUNT * 8, 256, 0, ctx->stream>>>(g2d, (const uint32_t*)(base + L.vis_list), &cnt->n_visible, out,
                                                             (unsigned long long*)&cnt->n_rows);
  SPLX_LAUNCH_CHECK(ctx, "k_gradient_rows");
  *rows = out;
  *num_rows = &cnt->n_rows;
  return SPLX_OK;
}

int launch_slot_map(splx_ctx* ctx, const PlanDev& plan, uint32_t* slot_map_out) {
  const uint32_t nslots = (uint32_t)plan.K * (uint32_t)plan.ntiles;
  k_slot_map<<<1, 1024, 0, ctx->stream>>>(plan.tile_state, plan.pv, (uint32_t)plan.ntiles, nslots, plan.open_slots, slot_map_out,
                                          slot_map_out + nslots);
  SPLX_LAUNCH_CHECK(ctx, "k_slot_map");
  return SPLX_OK;
}

int launch_bin_sort(splx_ctx* ctx, const splx_projected* pr, int64_t n, const PlanDev& plan, const int64_t* part_offsets,
                    const splx_binning* out, void* ws, size_t ws_bytes, const CrossDev* cross) {
  const int K = plan.K;
  const PlanDev& cam = plan;   // TX, TY
  const int sbits = slot_bits(K, cam.TX, cam.TY);
  if (sbits > SLOT_BITS * MAX_PASSES) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_bin_sort: K*tiles needs %d key bits (max 32)", sbits);
  const Layout L = make_layout(n, out->capacity, sbits);
  if (ws_bytes < L.total)
    SPLX_FAIL(ctx, SPLX_ERR_WORKSPACE, "splx_bin_sort: workspace %zu B < required %zu B", ws_bytes, L.total);
  char* base = (char*)ws;
  Counters* cnt = (Counters*)(base + L.counters);
  uint32_t* ckeys_a = (uint32_t*)(base + L.ckeys_a); uint32_t* cvals_a = (uint32_t*)(base + L.cvals_a);
  uint32_t* ckeys_b = (uint32_t*)(base + L.ckeys_b); uint32_t* cvals_b = (uint32_t*)(base + L.cvals_b);
  uint32_t* offs = (uint32_t*)(base + L.offs);
  const int ntiles = cam.TX * cam.TY;

  SPLX_CUDA_OK(ctx, cudaMemsetAsync(base, 0, L.zero_bytes, ctx->stream));
  SPLX_CUDA_OK(ctx, cudaMemsetAsync(out->tile_ranges, 0, (size_t)K * ntiles * 2 * sizeof(uint32_t), ctx->stream));
  SPLX_CUDA_OK(ctx, cudaMemsetAsync(out->num_intersections + 1, 0, sizeof(uint64_t), ctx->stream));
  const RunTable rt = make_runs(plan, part_offsets, 1, false);
  const int64_t n_act = rt.jprefix[rt.n];    // Gaussians of the participating partitions
  if (out->slot_order)   // count of live slots and the class cursors
    SPLX_CUDA_OK(ctx, cudaMemsetAsync(out->slot_order + (size_t)K * ntiles, 0, SPLX_ORDER_EXTRA * sizeof(uint32_t), ctx->stream));
  if (n_act == 0 || out->capacity == 0) {
    k_publish_m<<<1, 1, 0, ctx->stream>>>(cnt, out->num_intersections);
    SPLX_LAUNCH_CHECK(ctx, "k_publish_m");
    return SPLX_OK;
  }
  int rc;
  // 1. visible Gaussians, index order
  VisibleOp vop{pr->tiles_touched, pr->depth, ckeys_a, cvals_a, (uint32_t*)(base + L.vis_list), (uint64_t)n_act, {}};
  vop.map.n = rt.n;
  for (int r = 0; r < rt.n; ++r) { vop.map.begin[r] = rt.begin[r]; vop.map.jprefix[r] = rt.jprefix[r]; }
  vop.map.jprefix[rt.n] = rt.jprefix[rt.n];
  // status words per pass of the depth sort (room for every participating Gaussian being visible)
  const size_t stride_d = (((size_t)n_act + SCAN_TILE - 1) / SCAN_TILE) * SCAN_RS * 256;
  if ((rc = compact_visible(ctx, vop, (uint32_t*)(base + L.st_scan_v), &cnt->n_visible, (uint32_t*)(base + L.ghist_d),
                            (uint64_t*)(base + L.st_depth), stride_d))) return rc;
  // 2. stable sort by depth bits (4 passes of 8 bits: result back in the a-buffers); histograms came with step 1
  if ((rc = radix_sort<uint32_t, 256>(ctx, ckeys_a, cvals_a, ckeys_b, cvals_b, (uint64_t)n_act, &cnt->n_visible, 0, 32,
                                      (uint32_t*)(base + L.ghist_d), (uint64_t*)(base + L.st_depth), &cnt->ticket[2],
                                      stride_d))) return rc;
  // 3. offsets of every visible Gaussian's run, M, and the keys in depth order
  TouchedOp top{pr->tiles_touched, cvals_a, offs};
  if ((rc = scan_exclusive<TouchedOp>(ctx, top, (uint64_t)n_act, &cnt->n_visible, (uint64_t*)(base + L.st_scan_t), &cnt->ticket[1],
                           &cnt->m_total, &cnt->m_sorted, out->capacity))) return rc;
  // 4. the (compact slot, depth-order position) pairs and their stable sort on the compact slot bits.  Two pair buffers:
  // A in the workspace, B in the memory of out->keys (dead until the last pass writes the 64-bit keys there, reading A).
  PartOffs parts;
  parts.K = K;
  for (int k = 0; k <= K; ++k) parts.off[k] = part_offsets[k];
  FinalOut fin;
  memset(&fin, 0, sizeof fin);
  int nact = 0;
  for (int k = 0; k < K; ++k) {
    const bool act = plan.pv.v[k] >= 0 && part_offsets[k + 1] > part_offsets[k];
    parts.rank[k] = act ? (signed char)nact : (signed char)-1;
    if (act) { fin.skip[nact] = (uint32_t)(k - nact) * (uint32_t)ntiles; ++nact; }
  }
  fin.skip[nact] = (uint32_t)(K - nact) * (uint32_t)ntiles;       // the slot of filtered pairs: one past the last real slot
  fin.keys = out->keys; fin.vals = out->vals; fin.ckeys = ckeys_a; fin.cvals = cvals_a; fin.ntiles = (uint32_t)ntiles;
  const uint32_t cslots = (uint32_t)nact * (uint32_t)ntiles;      // compact slots 0 .. cslots (cslots itself = filtered)
  int cbits = 1;
  while (((uint64_t)1 << cbits) <= cslots) ++cbits;
  // renumbered open slots (splx_plan.open_slots), where that saves a pass over the intersections
  CrossEmit cx;
  memset(&cx, 0, sizeof cx);
  cx.ntiles = (uint32_t)ntiles; cx.nslots = cslots;
  if (plan.open_slots > 0 && plan.slot_map) {
    const uint32_t cap = plan.open_slots;       // the bound the caller built the map with (splx_slot_map)
    int obits = 1;
    while (((uint64_t)1 << obits) <= (uint64_t)cap + 1) ++obits;       // the values 0 .. cap + 1
    if (plan.open_forced || (obits + SLOT_BITS - 1) / SLOT_BITS < (cbits + SLOT_BITS - 1) / SLOT_BITS) {
      cx.cmap = plan.slot_map; cx.nslots = cap; fin.inv = plan.slot_map + (size_t)K * ntiles; cbits = obits;
    }
  }
  const PassPlan spl = plan_passes(0, cbits, SLOT_BITS);
  uint32_t* A_k = (uint32_t*)(base + L.pairs_tmp); uint32_t* A_p = A_k + out->capacity;
  uint32_t* B_k = (uint32_t*)out->keys; uint32_t* B_p = B_k + out->capacity;
  const bool startA = (spl.npass & 1) != 0;                       // so that the LAST pass reads A (and may overwrite B's memory)
  uint32_t* k0 = startA ? A_k : B_k; uint32_t* p0 = startA ? A_p : B_p;
  uint32_t* k1 = startA ? B_k : A_k; uint32_t* p1 = startA ? B_p : A_p;
  if (cross && cross->mask) {
    cx.mask = cross->mask; cx.tile_state = plan.tile_state;
    for (int k = 0; k < K; ++k) { cx.zlo[k] = cross->zlo[k]; cx.zhi[k] = cross->zhi[k]; cx.view[k] = plan.pv.v[k]; }
  }
  const uint64_t emit_blocks = ((uint64_t)n_act + 255) / 256, range_blocks = (out->capacity / 4 + 255) / 256 + 1;
  const unsigned g_emit = (unsigned)(emit_blocks < 2 * PERSISTENT_CTAS ? emit_blocks : 2 * PERSISTENT_CTAS);
  const uint64_t emit_tiles = (out->capacity + 1023) / 1024;     // output tiles of 1024 keys
  const unsigned g_lb = (unsigned)(emit_tiles < PERSISTENT_CTAS ? emit_tiles : PERSISTENT_CTAS);
  uint32_t* gh = (uint32_t*)(base + L.ghist_s);
  uint64_t* sst = (uint64_t*)(base + L.st_slot);
  const size_t sstride = (((size_t)out->capacity + RS_TILE - 1) / RS_TILE) * SLOT_NB;
  if (cx.mask) {
    k_emit_keys<true><<<g_emit, 256, 0, ctx->stream>>>(pr->means2d, pr->radius, ckeys_a, cvals_a, offs, cnt, parts, cam.TX, cam.TY,
                                                       out->capacity, k0, p0, spl, gh, sst, sstride, cx);
    SPLX_LAUNCH_CHECK(ctx, "k_emit_keys");
    k_emit_keys_lb<true><<<g_lb, 256, 0, ctx->stream>>>(pr->means2d, pr->radius, ckeys_a, cvals_a, offs, cnt, parts, cam.TX, cam.TY,
                                                        out->capacity, k0, p0, spl, gh, sst, sstride, cx);
    SPLX_LAUNCH_CHECK(ctx, "k_emit_keys_lb");
  } else {
    k_emit_keys<false><<<g_emit, 256, 0, ctx->stream>>>(pr->means2d, pr->radius, ckeys_a, cvals_a, offs, cnt, parts, cam.TX, cam.TY,
                                                        out->capacity, k0, p0, spl, gh, sst, sstride, cx);
    SPLX_LAUNCH_CHECK(ctx, "k_emit_keys");
    k_emit_keys_lb<false><<<g_lb, 256, 0, ctx->stream>>>(pr->means2d, pr->radius, ckeys_a, cvals_a, offs, cnt, parts, cam.TX, cam.TY,
                                                         out->capacity, k0, p0, spl, gh, sst, sstride, cx);
    SPLX_LAUNCH_CHECK(ctx, "k_emit_keys_lb");
  }
  if ((rc = radix_sort<uint32_t, SLOT_NB>(ctx, k0, p0, k1, p1, out->capacity, &cnt->m_sorted, 0, cbits, gh, sst, &cnt->ticket[6], 0,
                                          &fin))) return rc;
  // 5. ranges
  k_tile_ranges<<<(unsigned)(range_blocks < 4 * PERSISTENT_CTAS ? range_blocks : 4 * PERSISTENT_CTAS), 256, 0, ctx->stream>>>(
      out->keys, cnt, plan.tile_state, out->tile_ranges, out->num_intersections, (uint32_t)K * (uint32_t)ntiles, cx.mask != nullptr);
  SPLX_LAUNCH_CHECK(ctx, "k_tile_ranges");
  if (out->slot_order && slot_order_pays(plan)) {
    const uint32_t nslots = (uint32_t)K * (uint32_t)ntiles;
    uint32_t* n_live = out->slot_order + nslots;
    uint32_t* cursor = n_live + 1;
    const unsigned ob = (nslots + 255) / 256 < 2 * PERSISTENT_CTAS ? (nslots + 255) / 256 : 2 * PERSISTENT_CTAS;
    k_order_hist<<<ob, 256, 0, ctx->stream>>>(out->tile_ranges, nslots, cursor);
    SPLX_LAUNCH_CHECK(ctx, "k_order_hist");
    k_order_scan<<<1, ORD_CLASSES, 0, ctx->stream>>>(cursor, n_live);
    SPLX_LAUNCH_CHECK(ctx, "k_order_scan");
    k_order_scatter<<<ob, 256, 0, ctx->stream>>>(out->tile_ranges, nslots, cursor, out->slot_order);
    SPLX_LAUNCH_CHECK(ctx, "k_order_scatter");
  }
  return SPLX_OK;
}
