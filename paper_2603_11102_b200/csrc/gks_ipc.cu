/*
 * gks_ipc.cu — a sub-domain's halo windows offered to ANOTHER PROCESS (one process per GPU: the
 * x-slab decomposition over several GPUs).  gks_halo_push writes a sub-domain's boundary planes straight into the ghost
 * layers of its neighbour's padded state; inside one process the neighbour's window is a plain device pointer
 * (gks_halo_window_get), between processes the allocation that holds the neighbour's workspace is mapped with CUDA IPC:
 *
 *   owner:      gks_halo_export_get(ctx, &e)      e = { cudaIpcMemHandle_t of the allocation, byte offsets of W^n and W*
 *                                                       inside it, extents and pitches }: plain bytes, sent to the neighbour
 *   neighbour:  gks_halo_export_open(&e, win, &m) maps the allocation (peer-to-peer over NVLink when the owner's GPU is
 *                                                 another one) and fills win[0] (W^n) and win[1] (W*) for gks_halo_push
 *               gks_halo_export_close(m)          unmaps it
 *
 * The workspace must come from cudaMalloc (torch's caching allocator does, unless expandable segments are on): only
 * such allocations have IPC handles.  One allocation can be opened once per process: the driver opens it once per
 * neighbour RANK (two slabs on a periodic axis are each other's neighbour on both sides).
 * Ordering between the processes (the push must not land before the neighbour has finished reading its ghosts, the
 * neighbour must not sweep before the push has landed) is the driver's: paper_2603_11102_b200/slab.py IpcPushTransport.
 */
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstring>

#include "gks_internal.h"

static_assert(sizeof(cudaIpcMemHandle_t) == 64, "gks_halo_export::mem carries a cudaIpcMemHandle_t");

extern "C" {

gks_status gks_halo_export_get(gks_ctx *ctx, gks_halo_export *out) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!out) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "out is NULL");
  if (gks_status st = gks_check_device(ctx)) return st;
  /* base of the allocation that holds the workspace (a caching allocator hands out pieces of larger blocks) */
  typedef CUresult (*range_fn_t)(CUdeviceptr *, size_t *, CUdeviceptr);
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn ||
      q != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return gks_set_err(ctx, GKS_ERR_CUDA, "cuMemGetAddressRange is not available");
  }
  CUdeviceptr base = 0;
  size_t size = 0;
  if (((range_fn_t)fn)(&base, &size, (CUdeviceptr)ctx->Wn) != CUDA_SUCCESS || !base)
    return gks_set_err(ctx, GKS_ERR_CUDA, "cuMemGetAddressRange failed on the workspace");
  const unsigned long long b = (unsigned long long)base, n0 = (unsigned long long)(uintptr_t)ctx->Wn,
                           n1 = (unsigned long long)(uintptr_t)ctx->Ws;
  if (n1 < b || n1 + 4ull * ctx->g.FS * sizeof(double) > b + size || n0 + 4ull * ctx->g.FS * sizeof(double) > b + size)
    return gks_set_err(ctx, GKS_ERR_WORKSPACE, "the workspace spans more than one device allocation");
  cudaIpcMemHandle_t h;
  const cudaError_t e = cudaIpcGetMemHandle(&h, (void *)(uintptr_t)base);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return gks_set_err(ctx, GKS_ERR_CUDA, "cudaIpcGetMemHandle: %s (the workspace must be a cudaMalloc allocation)",
                       cudaGetErrorString(e));
  }
  memset(out, 0, sizeof(*out));
  memcpy(out->mem, &h, sizeof(h));
  out->offset[0] = n0 - b;
  out->offset[1] = n1 - b;
  out->nx = ctx->g.n[0];
  out->ny = ctx->g.n[1];
  out->nz = ctx->g.n[2];
  out->pitch_x = ctx->g.P[0];
  out->pitch_y = ctx->g.P[1];
  out->field_stride = ctx->g.FS;
  return GKS_OK;
}

gks_status gks_halo_export_open(const gks_halo_export *in, gks_halo_window win[2], void **mapping) {
  if (!in || !win || !mapping) return gks_set_err(nullptr, GKS_ERR_INVALID_ARG, "gks_halo_export_open: NULL argument");
  if (in->nx < 6 || in->ny < 6 || in->nz < 6 || in->pitch_x < in->nx + 2 * GKS_NG || in->pitch_y != in->ny + 2 * GKS_NG ||
      in->field_stride < (long long)in->pitch_x * in->pitch_y * (in->nz + 2 * GKS_NG) || (in->offset[0] & 7) || (in->offset[1] & 7))
    return gks_set_err(nullptr, GKS_ERR_INVALID_ARG, "gks_halo_export_open: not a description written by gks_halo_export_get");
  cudaIpcMemHandle_t h;
  memcpy(&h, in->mem, sizeof(h));
  void *base = nullptr;
  const cudaError_t e = cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess);
  if (e != cudaSuccess || !base) {
    cudaGetLastError();
    return gks_set_err(nullptr, GKS_ERR_CUDA, "cudaIpcOpenMemHandle: %s (an allocation opens once per process, and not in "
                       "the process that owns it)", cudaGetErrorString(e));
  }
  for (int w = 0; w < 2; ++w) {
    win[w].W = reinterpret_cast<double *>(static_cast<char *>(base) + in->offset[w]);
    win[w].nx = in->nx;
    win[w].ny = in->ny;
    win[w].nz = in->nz;
    win[w].pitch_x = in->pitch_x;
    win[w].pitch_y = in->pitch_y;
    win[w].field_stride = in->field_stride;
  }
  *mapping = base;
  return GKS_OK;
}

gks_status gks_halo_export_close(void *mapping) {
  if (!mapping) return GKS_OK;
  const cudaError_t e = cudaIpcCloseMemHandle(mapping);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return gks_set_err(nullptr, GKS_ERR_CUDA, "cudaIpcCloseMemHandle: %s", cudaGetErrorString(e));
  }
  return GKS_OK;
}

} /* extern "C" */
