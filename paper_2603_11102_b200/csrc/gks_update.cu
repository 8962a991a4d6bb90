/*
 * gks_update.cu — flux divergence (Eq. 5) fused with the two S2O4 stage updates
 * (formulas DESIGN.md S11):
 *   stage 1:  L = -sum_d (F_d+ - F_d-)/Delta_d, dL likewise from dF/dt, kept in registers;
 *             W* = W^n + dt/2 L + dt^2/8 dL,   P = W^n + dt L + dt^2/6 dL
 *   stage 2:  W^{n+1} = P + dt^2/3 dL(W*)
 * HBM-bound: per cell and component stage 1 reads 12 face values (6 distinct lines, neighbours hit
 * L1/L2) + W and writes 2; stage 2 reads 6 + P and writes 1.
 *
 * Update + halo transfer in one kernel (x-slab decomposition): given the windows of the neighbouring
 * sub-domains (GksPush), stage 1 stores the 3 planes of W* next to a cut face ALSO into the ghost planes of the neighbour
 * beyond it - the mapping of k_halo_push (gks_ghost.cu) - as it computes them; with the neighbour on another GPU the
 * stores travel peer to peer while the rest of the update runs.  gks_step_begin_push.
 */
#include "gks_internal.h"

namespace {

template <bool STAGE1, bool PUSH>
__global__ void __launch_bounds__(256) k_update(GksGrid g, const double *__restrict__ Win,
                                                const double *__restrict__ fx, const double *__restrict__ fy,
                                                const double *__restrict__ fz, double dt,
                                                double *__restrict__ out1, double *__restrict__ out2, int x0, int x1,
                                                GksPush push) {
  gks_pdl_enter();
  const int i = x0 + blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= x1 || j >= g.n[1]) return;
  const long long id = g.idx(i, j, k);
  const double iwx = g.inv_w[0][i + GKS_NG], iwy = g.inv_w[1][j + GKS_NG], iwz = g.inv_w[2][k + GKS_NG];
  /* upper face of the cell along each axis; where face n of an axis is face 0 (g.wrapf: periodic axis) the sweep
     does not store it and the last cell reads face 0 */
  const long long sx = (g.wrapf[0] && i == g.n[0] - 1) ? -(long long)(g.n[0] - 1) : 1;
  const long long sy = (g.wrapf[1] && j == g.n[1] - 1) ? -(long long)(g.n[1] - 1) * g.st[1] : g.st[1];
  const long long sz = (g.wrapf[2] && k == g.n[2] - 1) ? -(long long)(g.n[2] - 1) * g.st[2] : g.st[2];
  double wsv[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const long long o = c * g.FS + id, od = (4 + c) * g.FS + id;
    const double dL = -((fx[od + sx] - fx[od]) * iwx + (fy[od + sy] - fy[od]) * iwy + (fz[od + sz] - fz[od]) * iwz);
    if (STAGE1) {
      const double L = -((fx[o + sx] - fx[o]) * iwx + (fy[o + sy] - fy[o]) * iwy + (fz[o + sz] - fz[o]) * iwz);
      const double w = Win[o];
      const double ws = w + 0.5 * dt * L + (dt * dt / 8.0) * dL;
      out1[o] = ws;
      out2[o] = w + dt * L + (dt * dt / 6.0) * dL;
      wsv[c] = ws;
    } else {
      out1[o] = Win[o] + (dt * dt / 3.0) * dL;
    }
  }
  /* after all loads (the compiler batches them): my low planes are the neighbour's HIGH ghosts (cells nx_nb .. nx_nb+2),
     my high planes its low ghosts (-3 .. -1) */
  if (STAGE1 && PUSH) {
    if (push.W[0] != nullptr && i < GKS_NG) {
      const long long d = ((long long)(k + GKS_NG) * push.PY[0] + (j + GKS_NG)) * push.PX[0] + (push.nx[0] + i + GKS_NG);
#pragma unroll
      for (int c = 0; c < 4; ++c) push.W[0][c * push.FS[0] + d] = wsv[c];
    }
    if (push.W[1] != nullptr && i >= g.n[0] - GKS_NG) {
      const long long d = ((long long)(k + GKS_NG) * push.PY[1] + (j + GKS_NG)) * push.PX[1] + (i - g.n[0] + GKS_NG);
#pragma unroll
      for (int c = 0; c < 4; ++c) push.W[1][c * push.FS[1] + d] = wsv[c];
    }
  }
}

/* 256 threads; 64 along x unless the (sub-)domain is narrower (an x-slab of 32 cells would idle half of them) */
dim3 update_block(int nx) { return nx > 32 ? dim3(64, 4) : dim3(32, 8); }

} /* namespace */

int gks_launch_stage1(const GksGrid &g, const double *Wn, double *const flux[3], double dt, double *Ws,
                      double *Pbuf, cudaStream_t s, int x0, int x1, const GksPush *push) {
  if (x1 < 0) x1 = g.n[0];
  if (x1 <= x0) return 0;
  const dim3 blk = update_block(x1 - x0), grid((x1 - x0 + blk.x - 1) / blk.x, (g.n[1] + blk.y - 1) / blk.y, g.n[2]);
  GksPush none;
  memset(&none, 0, sizeof(none));
  /* the variant with the extra stores is a kernel of its own: in the plain one the compiler batches the loads of the
     four components, which stores through a pointer it cannot prove distinct would forbid (measured 1.27 -> 1.52 ms) */
  if (push && (push->W[0] || push->W[1]))
    gks_launch(k_update<true, true>, grid, blk, 0, s, g, Wn, flux[0], flux[1], flux[2], dt, Ws, Pbuf, x0, x1, *push);
  else
    gks_launch(k_update<true, false>, grid, blk, 0, s, g, Wn, flux[0], flux[1], flux[2], dt, Ws, Pbuf, x0, x1, none);
  return 1;
}

int gks_launch_stage2(const GksGrid &g, const double *Pbuf, double *const flux[3], double dt, double *Wn,
                      cudaStream_t s, int x0, int x1) {
  if (x1 < 0) x1 = g.n[0];
  if (x1 <= x0) return 0;
  const dim3 blk = update_block(x1 - x0), grid((x1 - x0 + blk.x - 1) / blk.x, (g.n[1] + blk.y - 1) / blk.y, g.n[2]);
  GksPush none;
  memset(&none, 0, sizeof(none));
  gks_launch(k_update<false, false>, grid, blk, 0, s, g, Pbuf, flux[0], flux[1], flux[2], dt, Wn, (double *)nullptr, x0, x1, none);
  return 1;
}
