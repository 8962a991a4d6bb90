/*
 * gks_math.cuh — device arithmetic of the CUDA path (fp64).  Written from PAPER.md and DESIGN.md,
 * independently of oracle/ (no shared code, tables or constants).
 *
 *  - WENO5-JS (ref [30]) at the cell edge and at the two Gauss points +-sqrt(3)/6.
 *    The nonlinear weights w_k = alpha_k / sum(alpha), alpha_k = d_k/(eps+beta_k)^2, are evaluated
 *    over the common denominator: with s_k = (eps+beta_k)^2 and t_0 = s_1 s_2, t_1 = s_0 s_2,
 *    t_2 = s_0 s_1,   sum_k w_k p_k = (sum_k d_k t_k p_k)/(sum_k d_k t_k):  one division instead of
 *    four, algebraically identical.
 *  - Collision: half-Maxwellian moments (S4).
 *  - Gauss-point flux (Eq. 6-8 + Appendix) in closed form: the moments of
 *    Eq. 7 with A from the compatibility condition are exactly the isothermal Navier-Stokes flux
 *    F = F_Euler(Q0) - mu (d_i U_j + d_j U_i), mu = tau p = rho_ref nu, and
 *    dF/dt = (dF_Euler/dQ) Q_t with Q_t = -div F_Euler(Q0) by the chain rule through the slopes
 *    (P5; tests/test_oracle_blocks.py pins the identity to 2e-15 on the oracle's literal
 *    moment algebra).
 */
#ifndef GKS_MATH_CUH
#define GKS_MATH_CUH

namespace gksd {

#define GKS_SQRT3 1.7320508075688772935

/* common-denominator Jiang-Shu factors t_k from the 5 averages */
__device__ __forceinline__ void js_t(double q0, double q1, double q2, double q3, double q4, double eps,
                                     double &t0, double &t1, double &t2) {
  const double a0 = q0 - 2.0 * q1 + q2, b0 = q0 - 4.0 * q1 + 3.0 * q2;
  const double a1 = q1 - 2.0 * q2 + q3, b1 = q1 - q3;
  const double a2 = q2 - 2.0 * q3 + q4, b2 = 3.0 * q2 - 4.0 * q3 + q4;
  const double k13 = 13.0 / 12.0;
  double s0 = eps + (k13 * a0 * a0 + 0.25 * b0 * b0);
  double s1 = eps + (k13 * a1 * a1 + 0.25 * b1 * b1);
  double s2 = eps + (k13 * a2 * a2 + 0.25 * b2 * b2);
  s0 *= s0;
  s1 *= s1;
  s2 *= s2;
  t0 = s1 * s2;
  t1 = s0 * s2;
  t2 = s0 * s1;
}

/* WENO5-JS values at BOTH edges of the middle cell: vl at x = -1/2, vr at x = +1/2 */
__device__ __forceinline__ void weno5_edges(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vl, double &vr) {
  double t0, t1, t2;
  js_t(q0, q1, q2, q3, q4, eps, t0, t1, t2);
  /* right edge: candidates (2,-7,11)/6, (-1,5,2)/6, (2,5,-1)/6 with linear weights .1,.6,.3 */
  const double r0 = 2.0 * q0 - 7.0 * q1 + 11.0 * q2;
  const double r1 = -q1 + 5.0 * q2 + 2.0 * q3;
  const double r2 = 2.0 * q2 + 5.0 * q3 - q4;
  /* left edge (mirror): candidates (-1,5,2)/6 on (q0,q1,q2), (2,5,-1)/6 on (q1,q2,q3), (11,-7,2)/6 on (q2,q3,q4);
     linear weights .3,.6,.1 */
  const double l0 = -q0 + 5.0 * q1 + 2.0 * q2;
  const double l1 = 2.0 * q1 + 5.0 * q2 - q3;
  const double l2 = 11.0 * q2 - 7.0 * q3 + 2.0 * q4;
  const double ar0 = 0.1 * t0, ar1 = 0.6 * t1, ar2 = 0.3 * t2;
  const double al0 = 0.3 * t0, al1 = 0.6 * t1, al2 = 0.1 * t2;
  const double numr = ar0 * r0 + ar1 * r1 + ar2 * r2, denr = ar0 + ar1 + ar2;
  const double numl = al0 * l0 + al1 * l1 + al2 * l2, denl = al0 + al1 + al2;
  const double inv = 1.0 / (6.0 * denr * denl);
  vr = numr * denl * inv;
  vl = numl * denr * inv;
}

/* WENO5-JS values at the Gauss points: vm at x = -sqrt(3)/6, vp at x = +sqrt(3)/6 (S7) */
__device__ __forceinline__ void weno5_gauss(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vm, double &vp) {
  double t0, t1, t2;
  js_t(q0, q1, q2, q3, q4, eps, t0, t1, t2);
  const double c12 = GKS_SQRT3 / 12.0, c3 = GKS_SQRT3 / 3.0, c4 = GKS_SQRT3 / 4.0;
  const double dA = (210.0 - GKS_SQRT3) / 1080.0, dB = 11.0 / 18.0, dC = (210.0 + GKS_SQRT3) / 1080.0;
  const double e01 = c12 * (q3 - q1); /* shared by the two middle candidates */
  const double pp0 = c12 * q0 - c3 * q1 + (1.0 + c4) * q2;
  const double pp1 = q2 + e01;
  const double pp2 = (1.0 - c4) * q2 + c3 * q3 - c12 * q4;
  const double pm0 = -c12 * q0 + c3 * q1 + (1.0 - c4) * q2;
  const double pm1 = q2 - e01;
  const double pm2 = (1.0 + c4) * q2 - c3 * q3 + c12 * q4;
  const double bt1 = dB * t1;
  const double ap0 = dA * t0, ap2 = dC * t2;
  const double am0 = dC * t0, am2 = dA * t2;
  const double nump = ap0 * pp0 + bt1 * pp1 + ap2 * pp2, denp = ap0 + bt1 + ap2;
  const double numm = am0 * pm0 + bt1 * pm1 + am2 * pm2, denm = am0 + bt1 + am2;
  const double inv = 1.0 / (denp * denm);
  vp = nump * denm * inv;
  vm = numm * denp * inv;
}

/* derivative of the quartic through the 5 averages at the Gauss points, per unit cell width (S8) */
__device__ __forceinline__ void quartic_slope_gauss(double q0, double q1, double q2, double q3, double q4,
                                                    double &sm, double &sp) {
  const double k0 = 1.0 / 12.0 - GKS_SQRT3 / 54.0, k1 = -2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0;
  const double k2 = -4.0 * GKS_SQRT3 / 9.0, k3 = 2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0;
  const double k4 = -1.0 / 12.0 - GKS_SQRT3 / 54.0;
  sp = k0 * q0 + k1 * q1 + k2 * q2 + k3 * q3 + k4 * q4;
  sm = -(k0 * q4 + k1 * q3 + k2 * q2 + k3 * q1 + k4 * q0);
}

/* index-space slope at the face between qb and qc from 4 averages qa,qb,qc,qd (S5) */
__device__ __forceinline__ double normal_slope(double qa, double qb, double qc, double qd) {
  return (15.0 * (qc - qb) - (qd - qa)) * (1.0 / 12.0);
}

/* collision factors from the normal velocities of the left / right states (S4):
 * el = <u^0>_{>0}(Ul), xl = exp(-lam Ul^2)/(2 sqrt(pi lam)); er = <u^0>_{<0}(Ur), xr likewise (positive) */
__device__ __forceinline__ void collision_factors(double Ul, double Ur, double lambda, double &el,
                                                  double &xl, double &er, double &xr) {
  const double theta = sqrt(lambda);
  const double c = 0.5 / sqrt(3.14159265358979323846 * lambda);
  el = 0.5 * erfc(-theta * Ul);
  er = 0.5 * erfc(theta * Ur);
  xl = c * exp(-lambda * Ul * Ul);
  xr = c * exp(-lambda * Ur * Ur);
}

/* Q0 from Ql, Qr; NRM = 1 + dir is the index of the normal momentum */
template <int DIR>
__device__ __forceinline__ void collision(const double Ql[4], const double Qr[4], double lambda, double Q0[4]) {
  const double Ul = Ql[1 + DIR] / Ql[0], Ur = Qr[1 + DIR] / Qr[0];
  double el, xl, er, xr;
  collision_factors(Ul, Ur, lambda, el, xl, er, xr);
#pragma unroll
  for (int c = 0; c < 4; ++c) Q0[c] = Ql[c] * el + Qr[c] * er;
  Q0[1 + DIR] += Ql[0] * xl - Qr[0] * xr; /* rho_l (Ul el + xl) + rho_r (Ur er - xr) */
}

/* Gauss-point flux in closed form.  dQ[s][c] = d_s Q0_c, s = x,y,z.  F and dF/dt of direction DIR. */
template <int DIR, bool NEED_F>
__device__ __forceinline__ void gauss_point_flux(const double Q0[4], const double dQ[3][4], double RT,
                                                 double mu, double F[4], double dF[4]) {
  const double rho = Q0[0];
  const double ir = 1.0 / rho;
  const double u[3] = {Q0[1] * ir, Q0[2] * ir, Q0[3] * ir};
  /* Q_t = -sum_s d_s F_Euler^s:  rho_t = -sum_s d_s m_s ;
     m_i,t = -sum_s (U_s d_s m_i + m_i d_s U_s) - RT d_i rho,  d_s U_s = (d_s m_s - U_s d_s rho)/rho */
  double du[3][3]; /* du[s][i] = d_s U_i */
#pragma unroll
  for (int s = 0; s < 3; ++s)
#pragma unroll
    for (int i = 0; i < 3; ++i) du[s][i] = (dQ[s][1 + i] - u[i] * dQ[s][0]) * ir;
  const double divm = dQ[0][1] + dQ[1][2] + dQ[2][3];
  const double divu = du[0][0] + du[1][1] + du[2][2];
  const double rho_t = -divm;
  double m_t[3];
#pragma unroll
  for (int i = 0; i < 3; ++i)
    m_t[i] = -(u[0] * dQ[0][1 + i] + u[1] * dQ[1][1 + i] + u[2] * dQ[2][1 + i]) - Q0[1 + i] * divu -
             RT * dQ[i][0];
  const double ud = u[DIR];
  dF[0] = m_t[DIR];
#pragma unroll
  for (int i = 0; i < 3; ++i) dF[1 + i] = ud * m_t[i] + u[i] * m_t[DIR] - u[i] * ud * rho_t;
  dF[1 + DIR] += RT * rho_t;
  if (NEED_F) {
    F[0] = Q0[1 + DIR];
#pragma unroll
    for (int i = 0; i < 3; ++i) F[1 + i] = Q0[1 + i] * ud - mu * (du[DIR][i] + du[i][DIR]);
    F[1 + DIR] += rho * RT;
  }
}

/* 3-point discrete delta (S13) */
__device__ __forceinline__ double delta3(double r) {
  const double x = fabs(r);
  if (x <= 0.5) return (1.0 + sqrt(1.0 - 3.0 * x * x)) * (1.0 / 3.0);
  if (x <= 1.5) {
    const double y = 1.0 - x;
    return (5.0 - 3.0 * x - sqrt(1.0 - 3.0 * y * y)) * (1.0 / 6.0);
  }
  return 0.0;
}

} /* namespace gksd */
#endif
