/*
 * gks_sweep_unfused.cu — straightforward three-kernel sweep of one direction (debug / cross-check
 * path; the production path is the fused kernel in gks_sweep_fused.cu).
 *   K_normal : WENO5 left/right states, normal slope, collision -> Q0[4], Dn[4] per face   (steps 2a-2c)
 *   K_pass1  : tangential pass along t1 -> per Gauss point g1: Q0, Dn, Dt1 (24 doubles)    (step 2d)
 *   K_pass2  : tangential pass along t2, Gauss-point fluxes, face average (F, dF/dt)       (steps 2e-2g)
 * Intermediates live in HBM in the padded cell index space (gks_internal.h).
 * PAPER.md:68-89 (Eq. 6-8), Appendix :501-558; readings S1-S11.
 */
#ifdef GKS_DEBUG   /* cross-check path: compiled into libgks_b200_debug.so only (include/gks_debug.h) */
#include "gks_internal.h"
#include "gks_math.cuh"

namespace {

template <int DIR> struct Axes {
  static constexpr int A = DIR;
  static constexpr int T1 = DIR == 0 ? 1 : 0;
  static constexpr int T2 = DIR == 2 ? 1 : 2;
};

struct Box3 { int lo[3], cnt[3]; };

__device__ __forceinline__ bool thread_cell(const Box3 &b, int p[3]) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  const int y = blockIdx.y * blockDim.y + threadIdx.y;
  const int z = blockIdx.z * blockDim.z + threadIdx.z;
  if (x >= b.cnt[0] || y >= b.cnt[1] || z >= b.cnt[2]) return false;
  p[0] = b.lo[0] + x;
  p[1] = b.lo[1] + y;
  p[2] = b.lo[2] + z;
  return true;
}

template <int DIR>
__global__ void __launch_bounds__(256) k_normal(GksGrid g, GksPhys ph, Box3 box, const double *__restrict__ W,
                                                double *__restrict__ N) {
  gks_pdl_enter();
  int p[3];
  if (!thread_cell(box, p)) return;
  const long long id = g.idx(p[0], p[1], p[2]);
  const long long sn = g.st[DIR];
  const double ihn = g.inv_12hn[DIR][p[DIR] + GKS_NG];
  double Ql[4], Qr[4], Dn[4], Q0[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const double *w = W + c * g.FS + id;
    const double q0 = w[-3 * sn], q1 = w[-2 * sn], q2 = w[-sn], q3 = w[0], q4 = w[sn], q5 = w[2 * sn];
    double dummy;
    gksd::weno5_edges(q0, q1, q2, q3, q4, ph.weno_eps4, dummy, Ql[c]); /* right edge of cell f-1 */
    gksd::weno5_edges(q1, q2, q3, q4, q5, ph.weno_eps4, Qr[c], dummy); /* left edge of cell f */
    Dn[c] = gksd::normal_slope12(q1, q2, q3, q4) * ihn;
  }
  gksd::collision<DIR>(Ql, Qr, ph.lambda, Q0);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    N[c * g.FS + id] = Q0[c];
    N[(4 + c) * g.FS + id] = Dn[c];
  }
}

template <int DIR>
__global__ void __launch_bounds__(256) k_pass1(GksGrid g, GksPhys ph, Box3 box, const double *__restrict__ N,
                                               double *__restrict__ T) {
  gks_pdl_enter();
  int p[3];
  if (!thread_cell(box, p)) return;
  constexpr int T1 = Axes<DIR>::T1;
  const long long id = g.idx(p[0], p[1], p[2]);
  const long long s1 = g.st[T1];
  const double iw = g.inv_w[T1][p[T1] + GKS_NG];
#pragma unroll
  for (int f = 0; f < 8; ++f) {
    const double *q = N + f * g.FS + id;
    const double q0 = q[-2 * s1], q1 = q[-s1], q2 = q[0], q3 = q[s1], q4 = q[2 * s1];
    double vm, vp;
    gksd::weno5_gauss(q0, q1, q2, q3, q4, ph.weno_eps4, vm, vp, ph.tang_linear != 0);
    T[(0 * 12 + f) * g.FS + id] = vm;
    T[(1 * 12 + f) * g.FS + id] = vp;
    if (f < 4) {
      double sm, sp;
      gksd::quartic_slope_gauss(q0, q1, q2, q3, q4, sm, sp);
      T[(0 * 12 + 8 + f) * g.FS + id] = sm * iw;
      T[(1 * 12 + 8 + f) * g.FS + id] = sp * iw;
    }
  }
}

template <int DIR, bool NEED_F>
__global__ void __launch_bounds__(256) k_pass2(GksGrid g, GksPhys ph, Box3 box, const double *__restrict__ T,
                                               double *__restrict__ flux) {
  gks_pdl_enter();
  int p[3];
  if (!thread_cell(box, p)) return;
  constexpr int A = Axes<DIR>::A, T1 = Axes<DIR>::T1, T2 = Axes<DIR>::T2;
  const long long id = g.idx(p[0], p[1], p[2]);
  const long long s2 = g.st[T2];
  const double iw = g.inv_w[T2][p[T2] + GKS_NG];
  double Fs[4] = {0, 0, 0, 0}, dFs[4] = {0, 0, 0, 0};
#pragma unroll 1
  for (int g1 = 0; g1 < 2; ++g1) {
    double v[12][2], d2[4][2];
#pragma unroll
    for (int f = 0; f < 12; ++f) {
      const double *q = T + (g1 * 12 + f) * g.FS + id;
      const double q0 = q[-2 * s2], q1 = q[-s2], q2 = q[0], q3 = q[s2], q4 = q[2 * s2];
      gksd::weno5_gauss(q0, q1, q2, q3, q4, ph.weno_eps4, v[f][0], v[f][1], ph.tang_linear != 0);
      if (f < 4) {
        gksd::quartic_slope_gauss(q0, q1, q2, q3, q4, d2[f][0], d2[f][1]);
        d2[f][0] *= iw;
        d2[f][1] *= iw;
      }
    }
#pragma unroll
    for (int g2 = 0; g2 < 2; ++g2) {
      double Q0[4], dQ[3][4], F[4], dF[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        Q0[c] = v[c][g2];
        dQ[A][c] = v[4 + c][g2];
        dQ[T1][c] = v[8 + c][g2];
        dQ[T2][c] = d2[c][g2];
      }
      gksd::gauss_point_flux<DIR, NEED_F>(Q0, dQ, ph.RT, ph.mu, F, dF);
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        if (NEED_F) Fs[c] += F[c];
        dFs[c] += dF[c];
      }
    }
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (NEED_F) flux[c * g.FS + id] = 0.25 * Fs[c];
    flux[(4 + c) * g.FS + id] = 0.25 * dFs[c];
  }
}

inline dim3 grid_for(const Box3 &b, dim3 blk) {
  return dim3((b.cnt[0] + blk.x - 1) / blk.x, (b.cnt[1] + blk.y - 1) / blk.y, (b.cnt[2] + blk.z - 1) / blk.z);
}

template <int DIR>
int sweep_dir(const GksGrid &g, const GksPhys &ph, const double *W, double *tmpN, double *tmpT, double *flux,
              bool need_F, cudaStream_t s) {
  constexpr int A = Axes<DIR>::A, T1 = Axes<DIR>::T1, T2 = Axes<DIR>::T2;
  const dim3 blk(32, 4, 2);
  Box3 b;
  b.lo[A] = 0; b.cnt[A] = g.n[A] + 1;
  b.lo[T1] = -2; b.cnt[T1] = g.n[T1] + 4;
  b.lo[T2] = -2; b.cnt[T2] = g.n[T2] + 4;
  k_normal<DIR><<<grid_for(b, blk), blk, 0, s>>>(g, ph, b, W, tmpN);
  b.lo[T1] = 0; b.cnt[T1] = g.n[T1];
  k_pass1<DIR><<<grid_for(b, blk), blk, 0, s>>>(g, ph, b, tmpN, tmpT);
  b.lo[T2] = 0; b.cnt[T2] = g.n[T2];
  if (need_F) k_pass2<DIR, true><<<grid_for(b, blk), blk, 0, s>>>(g, ph, b, tmpT, flux);
  else k_pass2<DIR, false><<<grid_for(b, blk), blk, 0, s>>>(g, ph, b, tmpT, flux);
  return 3;
}

} /* namespace */

int gks_launch_sweep_unfused(const GksGrid &g, const GksPhys &ph, int dir, const double *W, double *tmpN,
                             double *tmpT, double *flux, bool need_F, cudaStream_t s) {
  switch (dir) {
    case 0: return sweep_dir<0>(g, ph, W, tmpN, tmpT, flux, need_F, s);
    case 1: return sweep_dir<1>(g, ph, W, tmpN, tmpT, flux, need_F, s);
    default: return sweep_dir<2>(g, ph, W, tmpN, tmpT, flux, need_F, s);
  }
}

#endif /* GKS_DEBUG */
