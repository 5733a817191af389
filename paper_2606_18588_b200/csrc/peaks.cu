// peaks.cu -- the two micro-benchmarks behind the "alu" rooflines of the blend kernels ("the bench
// must first measure an FMA-loop and an ex2-loop micro-peak on the box ... and use those as denominators").  Not part
// of the method: measurement helpers, timed by the caller with CUDA events.
//   kind 0: FP32 FMA issue peak   -- 8 independent FFMA chains per thread (ILP hides the 4-cycle dependent latency)
//   kind 1: MUFU ex2 issue peak   -- 8 independent ex2.approx chains per thread (x <- 2^-x stays in (0.5, 1))
#include "common.cuh"

namespace {

constexpr int PK_THREADS = 256, PK_CTAS_PER_SM = 8, PK_ILP = 8;

__global__ void __launch_bounds__(PK_THREADS)
k_peak_fma(long long iters, float a, float b, float* sink) {
  float x[PK_ILP];
#pragma unroll
  for (int i = 0; i < PK_ILP; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) x[i] = fmaf(x[i], a, b);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PK_ILP; ++i) s += x[i];
  if (s == 123.456f) *sink = s;      // never true for the a, b passed: keeps the chains alive without a store
}

__global__ void __launch_bounds__(PK_THREADS)
k_peak_ex2(long long iters, float* sink) {
  float x[PK_ILP];
#pragma unroll
  for (int i = 0; i < PK_ILP; ++i) x[i] = 0.5f + (float)(threadIdx.x + i) * 1e-3f;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < PK_ILP; ++i) asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(x[i]) : "f"(-x[i]));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PK_ILP; ++i) s += x[i];
  if (s == 123.456f) *sink = s;
}

}  // namespace

extern "C" int splx_microbench(splx_ctx* ctx, int kind, int64_t iters, float* sink, double* work) {
  if (!ctx) return SPLX_ERR_INVALID_ARG;
  if ((kind != 0 && kind != 1) || iters < 1 || !sink || !work) SPLX_FAIL(ctx, SPLX_ERR_INVALID_ARG, "splx_microbench: bad argument");
  const int grid = SPLX_SM_COUNT * PK_CTAS_PER_SM;
  const double ops = (double)grid * PK_THREADS * (double)iters * PK_ILP;
  if (kind == 0) {
    k_peak_fma<<<grid, PK_THREADS, 0, ctx->stream>>>((long long)iters, 0.999f, 1e-3f, sink);
    *work = 2.0 * ops;      // one FMA = 2 flops
  } else {
    k_peak_ex2<<<grid, PK_THREADS, 0, ctx->stream>>>((long long)iters, sink);
    *work = ops;            // ex2 evaluations
  }
  SPLX_LAUNCH_CHECK(ctx, "k_peak");
  return SPLX_OK;
}
