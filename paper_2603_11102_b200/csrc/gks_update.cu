/*
 * gks_update.cu — flux divergence (Eq. 5) fused with the two S2O4 stage updates
 * (formulas DESIGN.md S11):
 *   stage 1:  L = -sum_d (F_d+ - F_d-)/Delta_d, dL likewise from dF/dt, kept in registers;
 *             W* = W^n + dt/2 L + dt^2/8 dL,   P = W^n + dt L + dt^2/6 dL
 *   stage 2:  W^{n+1} = P + dt^2/3 dL(W*)
 * HBM-bound: per cell and component stage 1 reads 12 face values (6 distinct lines, neighbours hit
 * L1/L2) + W and writes 2; stage 2 reads 6 + P and writes 1.
 */
#include "gks_internal.h"

namespace {

template <bool STAGE1>
__global__ void __launch_bounds__(256) k_update(GksGrid g, const double *__restrict__ Win,
                                                const double *__restrict__ fx, const double *__restrict__ fy,
                                                const double *__restrict__ fz, double dt,
                                                double *__restrict__ out1, double *__restrict__ out2, int x0, int x1) {
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
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const long long o = c * g.FS + id, od = (4 + c) * g.FS + id;
    const double dL = -((fx[od + sx] - fx[od]) * iwx + (fy[od + sy] - fy[od]) * iwy + (fz[od + sz] - fz[od]) * iwz);
    if (STAGE1) {
      const double L = -((fx[o + sx] - fx[o]) * iwx + (fy[o + sy] - fy[o]) * iwy + (fz[o + sz] - fz[o]) * iwz);
      const double w = Win[o];
      out1[o] = w + 0.5 * dt * L + (dt * dt / 8.0) * dL;
      out2[o] = w + dt * L + (dt * dt / 6.0) * dL;
    } else {
      out1[o] = Win[o] + (dt * dt / 3.0) * dL;
    }
  }
}

/* 256 threads; 64 along x unless the (sub-)domain is narrower (an x-slab of 32 cells would idle half of them) */
dim3 update_block(int nx) { return nx > 32 ? dim3(64, 4) : dim3(32, 8); }

} /* namespace */

int gks_launch_stage1(const GksGrid &g, const double *Wn, double *const flux[3], double dt, double *Ws,
                      double *Pbuf, cudaStream_t s, int x0, int x1) {
  if (x1 < 0) x1 = g.n[0];
  if (x1 <= x0) return 0;
  const dim3 blk = update_block(x1 - x0), grid((x1 - x0 + blk.x - 1) / blk.x, (g.n[1] + blk.y - 1) / blk.y, g.n[2]);
  gks_launch(k_update<true>, grid, blk, 0, s, g, Wn, flux[0], flux[1], flux[2], dt, Ws, Pbuf, x0, x1);
  return 1;
}

int gks_launch_stage2(const GksGrid &g, const double *Pbuf, double *const flux[3], double dt, double *Wn,
                      cudaStream_t s, int x0, int x1) {
  if (x1 < 0) x1 = g.n[0];
  if (x1 <= x0) return 0;
  const dim3 blk = update_block(x1 - x0), grid((x1 - x0 + blk.x - 1) / blk.x, (g.n[1] + blk.y - 1) / blk.y, g.n[2]);
  gks_launch(k_update<false>, grid, blk, 0, s, g, Pbuf, flux[0], flux[1], flux[2], dt, Wn, (double *)nullptr, x0, x1);
  return 1;
}
