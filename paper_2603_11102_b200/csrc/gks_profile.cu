/*
 * gks_profile.cu — measurement helpers of the C ABI: per-kernel-class CUDA-event timing on the
 * context's stream and, in the GKS_DEBUG library only, an fp64 FMA throughput calibration kernel (context
 * for the "alu" roofline bench.py reports).
 */
#include <cstdlib>

#include "gks_internal.h"

void gks_prof_begin(gks_ctx *ctx, int cat) {
  if (!ctx->prof_on || ctx->prof_n >= GKS_PROF_MAX) return;
  ctx->prof_cat[ctx->prof_n] = cat;
  cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n], ctx->stream);
}

void gks_prof_end(gks_ctx *ctx) {
  if (!ctx->prof_on || ctx->prof_n >= GKS_PROF_MAX) return;
  cudaEventRecord(ctx->prof_ev[2 * ctx->prof_n + 1], ctx->stream);
  ctx->prof_n += 1;
}

void gks_prof_free(gks_ctx *ctx) {
  if (ctx->prof_ev) {
    for (int i = 0; i < 2 * GKS_PROF_MAX; ++i) cudaEventDestroy(ctx->prof_ev[i]);
    free(ctx->prof_ev);
    free(ctx->prof_cat);
    ctx->prof_ev = nullptr;
    ctx->prof_cat = nullptr;
  }
}

#ifdef GKS_DEBUG
namespace {

/* 8 independent DFMA chains per thread, all in registers */
__global__ void __launch_bounds__(256) k_dfma(double *out, int iters, double a, double b) {
  gks_pdl_enter();
  double x0 = threadIdx.x * 1e-9, x1 = x0 + 1e-3, x2 = x0 + 2e-3, x3 = x0 + 3e-3, x4 = x0 + 4e-3, x5 = x0 + 5e-3,
         x6 = x0 + 6e-3, x7 = x0 + 7e-3;
#pragma unroll 4
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 12345.678) out[0] = s; /* never true: keeps the chains alive */
}

/* Issue-rate probe: per round KF DFMA on 8 independent register chains plus KI integer multiply-adds on 8 more, per
 * warp; 512 threads per CTA, one CTA per SM (4 warps per scheduler, as the fused sweep runs).  Answers: does an
 * instruction of another pipe cost the fp64 pipe an issue slot?  (DESIGN.md section 7.) */
template <int KF, int KI, int CHAINS>
__global__ void __launch_bounds__(512, 1) k_probe(double *out, int iters, double a, double b, int ia) {
  double x[8];
  int y[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    x[i] = threadIdx.x * 1e-9 + i;
    y[i] = threadIdx.x + i;
  }
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int j = 0; j < KF; ++j) x[(r + j) % CHAINS] = fma(x[(r + j) % CHAINS], a, b);
#pragma unroll
      for (int j = 0; j < KI; ++j) y[(r + j) & 7] = y[(r + j) & 7] * ia + 7;
    }
  }
  const long long t1 = clock64();
  double s = 0;
  int q = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    s += x[i];
    q += y[i];
  }
  if (ia == 0x7fffffff) out[2 + threadIdx.x] = s + q; /* never true at run time: keeps the chains alive */
  if (threadIdx.x == 0 && blockIdx.x == 0) out[1] = (double)(t1 - t0) / iters / 8;
}

template <int KF, int KI, int CHAINS>
double run_probe(gks_ctx *ctx, int nsm) {
  k_probe<KF, KI, CHAINS><<<nsm, 512, 0, ctx->stream>>>(ctx->red, 2000, 0.999999, 1e-7, 3);
  double h[2] = {0, 0};
  cudaMemcpyAsync(h, ctx->red, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream);
  cudaStreamSynchronize(ctx->stream);
  ctx->launches += 1;
  return h[1];
}

} /* namespace */
#endif

extern "C" {

gks_status gks_profile_enable(gks_ctx *ctx, int on) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (on && !ctx->prof_ev) {
    ctx->prof_ev = (cudaEvent_t *)calloc(2 * GKS_PROF_MAX, sizeof(cudaEvent_t));
    ctx->prof_cat = (int *)calloc(GKS_PROF_MAX, sizeof(int));
    if (!ctx->prof_ev || !ctx->prof_cat) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "out of host memory");
    for (int i = 0; i < 2 * GKS_PROF_MAX; ++i)
      if (cudaEventCreate(&ctx->prof_ev[i]) != cudaSuccess)
        return gks_set_err(ctx, GKS_ERR_CUDA, "cudaEventCreate failed");
  }
  ctx->prof_on = on ? 1 : 0;
  ctx->prof_n = 0;
  return GKS_OK;
}

gks_status gks_profile_read(gks_ctx *ctx, double *ms, long long *count) {
  if (!ctx || !ms || !count) return GKS_ERR_INVALID_ARG;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "sync: %s", cudaGetErrorString(e));
  for (int i = 0; i < ctx->prof_n; ++i) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, ctx->prof_ev[2 * i], ctx->prof_ev[2 * i + 1]) == cudaSuccess) {
      ms[ctx->prof_cat[i]] += t;
      count[ctx->prof_cat[i]] += 1;
    }
  }
  ctx->prof_n = 0;
  return GKS_OK;
}

#ifdef GKS_DEBUG
gks_status gks_debug_fp64_peak(gks_ctx *ctx, double *tflops) {
  if (!ctx || !tflops) return GKS_ERR_INVALID_ARG;
  cudaDeviceProp prop;
  int dev = 0;
  cudaGetDevice(&dev);
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "device properties");
  const int blocks = prop.multiProcessorCount * 8, iters = 1 << 15;
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(a, ctx->stream);
    k_dfma<<<blocks, 256, 0, ctx->stream>>>(ctx->red, iters, 0.999999, 1e-7);
    cudaEventRecord(b, ctx->stream);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    const double fl = 2.0 * 8.0 * (double)iters * 256.0 * blocks;
    if (rep > 0 && ms > 0) best = fmax(best, fl / (ms * 1e-3) * 1e-12);
    ctx->launches += 1;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "fp64 peak: %s", cudaGetErrorString(e));
  *tflops = best;
  return GKS_OK;
}

gks_status gks_debug_issue_probe(gks_ctx *ctx, double *cycles, int n) {
  if (!ctx || !cycles || n < GKS_DEBUG_PROBE_N) return GKS_ERR_INVALID_ARG;
  int dev = 0, nsm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  int k = 0;
  /* (KF, KI, chains): see include/gks_debug.h for the order */
  cycles[k++] = run_probe<8, 0, 8>(ctx, nsm);
  cycles[k++] = run_probe<8, 4, 8>(ctx, nsm);
  cycles[k++] = run_probe<8, 8, 8>(ctx, nsm);
  cycles[k++] = run_probe<8, 12, 8>(ctx, nsm);
  cycles[k++] = run_probe<8, 16, 8>(ctx, nsm);
  cycles[k++] = run_probe<4, 8, 8>(ctx, nsm);
  cycles[k++] = run_probe<8, 0, 1>(ctx, nsm);
  cycles[k++] = run_probe<8, 0, 2>(ctx, nsm);
  cycles[k++] = run_probe<8, 0, 4>(ctx, nsm);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "issue probe: %s", cudaGetErrorString(e));
  return GKS_OK;
}
#endif

} /* extern "C" */
