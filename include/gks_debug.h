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

/* Issue-rate probe (profiles/r2_microbench.md): clock cycles per round and warp of a loop that issues, per round and
 * warp, KF DFMA on `chains` independent register chains and KI integer multiply-adds on 8 independent ones, with 512
 * threads per CTA and one CTA per SM (4 warps per scheduler, as the fused sweep runs).  cycles[] receives
 * GKS_DEBUG_PROBE_N numbers, for (KF, KI, chains) = (8,0,8) (8,4,8) (8,8,8) (8,12,8) (8,16,8) (4,8,8) (8,0,1) (8,0,2)
 * (8,0,4).  Synchronises. */
#define GKS_DEBUG_PROBE_N 9
gks_status gks_debug_issue_probe(gks_ctx *ctx, double *cycles, int n);

/* Phase timeline of the fused sweep: ticks[32][8] = for every warp of CTA 0 of the LAST sweep launch the clock64 ticks
 * spent in the phases 0 loop bookkeeping, 1 hand-over wait, 2 TMA issue + cursor, 3 stage A, 4 stages BC + D + arrival,
 * 5 pass 2 (E), 6 transposes + flux + store (F).  Only a library built with -DGKS_TRACE records them
 * (`python -m paper_2603_11102_b200.trace`); any other returns GKS_ERR_STATE.  Synchronises. */
gks_status gks_debug_trace(gks_ctx *ctx, unsigned long long *ticks);

#ifdef __cplusplus
}
#endif
#endif /* GKS_B200_DEBUG_H */
