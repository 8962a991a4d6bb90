/*
 * gks_debug.h — additions of the DEBUG build of the library (libgks_b200_debug.so, compiled with -DGKS_DEBUG from the
 * same sources).  Not part of the product: libgks_b200.so exports include/gks.h and nothing of this file, and its
 * workspace does not carry the buffers these hooks need.  Used by tests/ (cross-check of the fused sweep) and by
 * bench.py (context figure for the fp64 roofline).
 */
#ifndef GKS_B200_DEBUG_H
#define GKS_B200_DEBUG_H

#include "gks.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Test hook: choose the sweep implementation.  0 (default) = fused production kernels (reconstruction + flux in one
 * kernel per direction, slabs staged through shared memory by TMA; the only one the product library has);
 * 1 = unfused cross-check kernels (three kernels per direction, 32 padded fields of intermediates in HBM, which
 * gks_workspace_bytes of the debug library adds to the workspace).  Both implement PAPER.md:68-89 (Eq. 6-8) under the
 * same readings and are compared with the oracle.  GKS_ERR_STATE inside a split step. */
gks_status gks_debug_set_sweep(gks_ctx *ctx, int mode);

/* Calibration: sustained fp64 FMA throughput of this GPU in TFLOP/s (2 flop per DFMA), measured with a
 * register-resident DFMA kernel on the context's stream (about 50 ms).  Synchronises. */
gks_status gks_debug_fp64_peak(gks_ctx *ctx, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* GKS_B200_DEBUG_H */
