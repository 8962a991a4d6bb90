/*
 * gks_noalloc.cu — gks_cfl_dt_noalloc: the CFL time step of PAPER.md:91 for callers that cannot allocate
 * (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): no context, no caller workspace.
 *
 * It is a variant of the reduction behind gks_cfl_dt (gks_forcing.cu: k_umax / k_cfl_final, whose scratch is carved
 * from the caller's workspace).  Here the scratch - one partial maximum per block - lives in the file-scope
 * __device__ array g_noalloc_scratch below: GKS_NOALLOC_MAX_BLOCKS doubles = 512 KB that every GPU which loads the
 * library holds until the process exits.  A block reduces GKS_NOALLOC_CELLS_PER_BLOCK cells, so the largest state
 * is GKS_NOALLOC_MAX_CELLS = 2^28 cells; larger ones are refused.
 *
 * In host code the NAME of a __device__ array is a host-side stand-in, not a device address, so the host never hands
 * the name to a kernel: noalloc_scratch() asks cudaGetSymbolAddress once per device, with that device current, and the
 * launches take the pointer it returned.
 *
 * Nothing in the scratch has to start at zero: slot b is WRITTEN by block b of the first kernel (a plain store, not an
 * accumulation) before the second kernel of the same call reads slots 0 .. blocks-1; what an earlier call left in the
 * array is never read.  All calls on a device share the array: two calls whose kernels may overlap on the GPU (different
 * streams without an ordering between them) race.
 *
 * This file calls no cudaMalloc / cudaFree and no allocating library routine, and no existing code path uses it.
 */
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "../../include/gks.h"

namespace {

constexpr int NOALLOC_THREADS = 256;
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_scratch[GKS_NOALLOC_MAX_BLOCKS];

thread_local char g_noalloc_err[256] = "";

gks_status noalloc_fail(gks_status st, const char *msg) {
  snprintf(g_noalloc_err, sizeof(g_noalloc_err), "%s", msg);
  return st;
}

/* device address of g_noalloc_scratch on the CURRENT device; looked up once per device */
cudaError_t noalloc_scratch(double **out) {
  static std::mutex mu;
  static double *ptr[NOALLOC_MAX_DEVICES] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!ptr[dev]) {
    double *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return cudaSuccess;
}

/* partial[b] = max over the cells of block b of |m| / rho; W is the plain state W[c][cell], c = rho, m_x, m_y, m_z */
__global__ void __launch_bounds__(NOALLOC_THREADS)
    k_umax_noalloc(const double *__restrict__ W, long long ncells, double *__restrict__ partial) {
  __shared__ double sh[NOALLOC_THREADS];
  const long long lo = (long long)blockIdx.x * GKS_NOALLOC_CELLS_PER_BLOCK;
  const long long hi = lo + GKS_NOALLOC_CELLS_PER_BLOCK < ncells ? lo + GKS_NOALLOC_CELLS_PER_BLOCK : ncells;
  double acc = 0.0;
  for (long long t = lo + threadIdx.x; t < hi; t += NOALLOC_THREADS) {
    const double mx = W[ncells + t], my = W[2 * ncells + t], mz = W[3 * ncells + t];
    acc = fmax(acc, sqrt(mx * mx + my * my + mz * mz) / W[t]);
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = NOALLOC_THREADS / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}

/* dt = cfl dmin / (max_b partial[b] + c_s) */
__global__ void __launch_bounds__(NOALLOC_THREADS)
    k_cfl_final_noalloc(const double *__restrict__ partial, int blocks, double cfl, double dmin, double cs,
                        double *__restrict__ dt) {
  __shared__ double sh[NOALLOC_THREADS];
  double acc = 0.0;
  for (int b = threadIdx.x; b < blocks; b += NOALLOC_THREADS) acc = fmax(acc, partial[b]);
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = NOALLOC_THREADS / 2; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
    __syncthreads();
  }
  if (threadIdx.x == 0) *dt = cfl * dmin / (sh[0] + cs);
}

} /* namespace */

extern "C" {

gks_status gks_cfl_dt_noalloc(const double *W, int nx, int ny, int nz, double dmin, double RT, double cfl, double *dt,
                              void *cuda_stream) {
  if (!W || !dt) return noalloc_fail(GKS_ERR_INVALID_ARG, "gks_cfl_dt_noalloc: W or dt is NULL");
  if (nx < 1 || ny < 1 || nz < 1) return noalloc_fail(GKS_ERR_INVALID_ARG, "gks_cfl_dt_noalloc: nx, ny, nz must be >= 1");
  if (!(dmin > 0) || !std::isfinite(dmin) || !(RT > 0) || !std::isfinite(RT) || !(cfl > 0) || !std::isfinite(cfl))
    return noalloc_fail(GKS_ERR_INVALID_ARG, "gks_cfl_dt_noalloc: dmin, RT and cfl must be finite and > 0");
  const long long ncells = (long long)nx * ny * nz;
  if (ncells > (long long)GKS_NOALLOC_MAX_CELLS) {
    snprintf(g_noalloc_err, sizeof(g_noalloc_err),
             "gks_cfl_dt_noalloc: %lld cells exceed GKS_NOALLOC_MAX_CELLS = %lld (static scratch of %d block partials); "
             "use gks_cfl_dt with a workspace",
             ncells, (long long)GKS_NOALLOC_MAX_CELLS, GKS_NOALLOC_MAX_BLOCKS);
    return GKS_ERR_INVALID_ARG;
  }
  cudaPointerAttributes pa;
  if (cudaPointerGetAttributes(&pa, W) != cudaSuccess || pa.type != cudaMemoryTypeDevice ||
      cudaPointerGetAttributes(&pa, dt) != cudaSuccess || pa.type != cudaMemoryTypeDevice) {
    cudaGetLastError();
    return noalloc_fail(GKS_ERR_INVALID_ARG, "gks_cfl_dt_noalloc: W and dt must be DEVICE pointers");
  }
  double *scratch = nullptr;
  cudaError_t e = noalloc_scratch(&scratch);
  if (e != cudaSuccess) {
    snprintf(g_noalloc_err, sizeof(g_noalloc_err), "gks_cfl_dt_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    return GKS_ERR_CUDA;
  }
  const int blocks = (int)((ncells + GKS_NOALLOC_CELLS_PER_BLOCK - 1) / GKS_NOALLOC_CELLS_PER_BLOCK);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  k_umax_noalloc<<<blocks, NOALLOC_THREADS, 0, s>>>(W, ncells, scratch);
  k_cfl_final_noalloc<<<1, NOALLOC_THREADS, 0, s>>>(scratch, blocks, cfl, dmin, sqrt(RT), dt);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    snprintf(g_noalloc_err, sizeof(g_noalloc_err), "gks_cfl_dt_noalloc: launch: %s", cudaGetErrorString(e));
    return GKS_ERR_CUDA;
  }
  return GKS_OK;
}

const char *gks_noalloc_last_error(void) { return g_noalloc_err; }

} /* extern "C" */
