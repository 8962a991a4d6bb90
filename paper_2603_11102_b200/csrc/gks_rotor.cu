/*
 * gks_rotor.cu — actuator-line front half on the device (Eq. 9, Eq. 14; S26-S27):
 * rotating actuator points, trilinear flow sampling, blade-element forces from a tabulated polar, free-stream
 * and tip corrections.  One thread per actuator point; the points and their forces ON THE FLUID land in the
 * same device arrays that alm_set_points fills, and the Gaussian spreading (k_alm, Eq. 10) takes them from
 * there: no host round trip per step.  Written from the paper, independently of oracle/.
 */
#include <cmath>

#include "gks_internal.h"

namespace {

constexpr double PI_D = 3.14159265358979323846;

/* interior cell containing x on axis a, clamped to the domain */
__device__ __forceinline__ int rotor_find_cell(const GksGrid &g, int a, double x) {
  const int n = g.n[a];
  if (g.uniform[a]) {
    const int c = (int)floor((x - g.x0[a]) / g.dx[a]);
    return max(0, min(n - 1, c));
  }
  const double *xf = g.xf[a] + GKS_NG;
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (x >= xf[mid]) lo = mid; else hi = mid;
  }
  return lo;
}

/* (rho, U, V, W) at X by trilinear interpolation between the 8 surrounding cell centres;
 * velocities are interpolated, not momenta; periodic axes wrap, beyond the outermost centres of a
 * non-periodic axis the outermost cell is used (S26) */
__device__ void sample_trilinear(const GksGrid &g, const double *__restrict__ W, const double X[3], double out[4]) {
  int i0[3], i1[3];
  double t[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double *xf = g.xf[a] + GKS_NG, *xc = g.xc[a] + GKS_NG;
    const int n = g.n[a];
    double x = X[a];
    if (g.periodic[a]) {
      const double L = xf[n] - xf[0];
      x -= floor((x - xf[0]) / L) * L;
    }
    const int c = rotor_find_cell(g, a, x);
    const int lo = x < xc[c] ? c - 1 : c;
    t[a] = (x - xc[lo]) / (xc[lo + 1] - xc[lo]);
    if (g.periodic[a]) {
      i0[a] = (lo + n) % n;
      i1[a] = (lo + 1) % n;
    } else { /* the first ghost layer of a HALO face holds the neighbouring sub-domain's cell */
      i0[a] = min(max(lo, g.halo[2 * a] ? -1 : 0), n - 1);
      i1[a] = min(max(lo + 1, 0), g.halo[2 * a + 1] ? n : n - 1);
    }
  }
  out[0] = out[1] = out[2] = out[3] = 0.0;
#pragma unroll
  for (int dk = 0; dk < 2; ++dk)
#pragma unroll
    for (int dj = 0; dj < 2; ++dj)
#pragma unroll
      for (int di = 0; di < 2; ++di) {
        const long long id = g.idx(di ? i1[0] : i0[0], dj ? i1[1] : i0[1], dk ? i1[2] : i0[2]);
        const double wgt = (di ? t[0] : 1.0 - t[0]) * (dj ? t[1] : 1.0 - t[1]) * (dk ? t[2] : 1.0 - t[2]);
        const double rho = W[id], ir = 1.0 / rho;
        out[0] += wgt * rho;
        out[1] += wgt * (W[g.FS + id] * ir);
        out[2] += wgt * (W[2 * g.FS + id] * ir);
        out[3] += wgt * (W[3 * g.FS + id] * ir);
      }
}

/* tabulated 2-D airfoil data of one airfoil section: linear in alpha, end values beyond the table (binary search) */
__device__ void polar_lookup_section(const GksRotor &r, int sec, double alpha, double &cl, double &cd) {
  const int n = r.npolar;
  const double *tcl = r.cl + (size_t)sec * n, *tcd = r.cd + (size_t)sec * n;
  if (alpha <= r.alpha[0]) { cl = tcl[0]; cd = tcd[0]; return; }
  if (alpha >= r.alpha[n - 1]) { cl = tcl[n - 1]; cd = tcd[n - 1]; return; }
  int lo = 0, hi = n - 1;                 /* alpha[lo] < alpha <= alpha[hi] */
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (r.alpha[mid] < alpha) lo = mid; else hi = mid;
  }
  const double t = (alpha - r.alpha[lo]) / (r.alpha[lo + 1] - r.alpha[lo]);
  cl = tcl[lo] + t * (tcl[lo + 1] - tcl[lo]);
  cd = tcd[lo] + t * (tcd[lo + 1] - tcd[lo]);
}

/* C_L, C_D of the station at radius rad (S28): linear in r between the two nearby airfoil
 * sections, the first / last section's inside / outside of them; one section: its table */
__device__ void polar_lookup(const GksRotor &r, double rad, double alpha, double &cl, double &cd) {
  const int ns = r.nsec;
  if (ns <= 1 || rad <= r.sec_r[0]) { polar_lookup_section(r, 0, alpha, cl, cd); return; }
  if (rad >= r.sec_r[ns - 1]) { polar_lookup_section(r, ns - 1, alpha, cl, cd); return; }
  int lo = 0, hi = ns - 1;                /* sec_r[lo] < rad <= sec_r[hi] */
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (r.sec_r[mid] < rad) lo = mid; else hi = mid;
  }
  const double t = (rad - r.sec_r[lo]) / (r.sec_r[lo + 1] - r.sec_r[lo]);
  double cl0, cd0, cl1, cd1;
  polar_lookup_section(r, lo, alpha, cl0, cd0);
  polar_lookup_section(r, lo + 1, alpha, cl1, cd1);
  cl = cl0 + t * (cl1 - cl0);
  cd = cd0 + t * (cd1 - cd0);
}

/* Eq. 14 */
__device__ double tip_factor(int N, double R, double r, double sinphi, double tsr, double c1, double c2) {
  if (!(sinphi > 0.0)) return 1.0;
  const double g1 = exp(-c1 * (N * tsr - c2)) + 0.1;
  return 2.0 / PI_D * acos(exp(-g1 * N * (R - r) / (2.0 * r * sinphi)));
}

__global__ void __launch_bounds__(128) k_rotor_forces(GksGrid g, const double *__restrict__ W, GksRotor R, double time,
                                                      double eps, double *__restrict__ pos,
                                                      double *__restrict__ force) {
  gks_pdl_enter();
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= R.nb * R.np) return;
  const int b = p / R.np, k = p - b * R.np;
  const double r = R.radius[k], w = R.width[k], c = R.chord[k];   /* station radius and element width (S28) */
  const double psi = R.theta0 + R.omega * time + 2.0 * PI_D * b / R.nb;
  double sp, cp;
  sincos(psi, &sp, &cp);
  const double er[3] = {0.0, cp, sp}, et[3] = {0.0, -sp, cp};
  double X[3], q[4];
#pragma unroll
  for (int a = 0; a < 3; ++a) X[a] = R.hub[a] + r * er[a];
  sample_trilinear(g, W, X, q);
  double Ux = q[1], Ut = q[2] * et[1] + q[3] * et[2];
  double phi = atan2(Ux, R.omega * r - Ut);
  double cl, cd;
  polar_lookup(R, r, phi - R.twist[k], cl, cd);
  if (R.fs_corr) {
    const double f = 1.0 / (1.0 - cd * c / (4.0 * sqrt(PI_D) * eps));
    Ux *= f;
    Ut *= f;
    phi = atan2(Ux, R.omega * r - Ut);
    polar_lookup(R, r, phi - R.twist[k], cl, cd);
  }
  const double urel2 = Ux * Ux + (Ut - R.omega * r) * (Ut - R.omega * r);
  const double L = 0.5 * q[0] * c * w * cl * urel2, D = 0.5 * q[0] * c * w * cd * urel2;
  double sphi, cphi;
  sincos(phi, &sphi, &cphi);
  double Fx = L * cphi + D * sphi, Ft = L * sphi - D * cphi;
  if (R.tip_corr) {
    const double tsr = R.omega * R.R / R.uref;
    Fx *= tip_factor(R.nb, R.R, r, sphi, tsr, 0.1219, 21.52);
    Ft *= tip_factor(R.nb, R.R, r, sphi, tsr, 0.0984, 13.026);
  }
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    pos[3 * p + a] = X[a];
    force[3 * p + a] = -(a == 0 ? Fx : Ft * et[a]);
  }
}

} /* namespace */

namespace {
/* x -> x + shift for n points (pos[3 p]): the image of a rotor beyond the seam of a periodic x axis */
__global__ void k_shift_x(double *pos, int n, double shift) {
  gks_pdl_enter();
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) pos[3 * p] += shift;
}
} /* namespace */

int gks_launch_shift_x(double *pos, int n, double shift, cudaStream_t s) {
  gks_launch(k_shift_x, dim3((n + 127) / 128), dim3(128), 0, s, pos, n, shift);
  return 1;
}

int gks_launch_rotor_forces(const GksGrid &g, const double *W, const GksRotor &r, double time, double eps,
                            double *pos, double *force, cudaStream_t s) {
  const int n = r.nb * r.np;
  gks_launch(k_rotor_forces, dim3((n + 127) / 128), dim3(128), 0, s, g, W, r, time, eps, pos, force);
  return 1;
}
