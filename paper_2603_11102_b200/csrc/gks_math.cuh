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

/* Full-width fp64 constants live in constant memory so that DFMA/DMUL take them as c[bank][offset]
 * operands (no per-use UMOV pairs).  Values with an all-zero low word (0.25, 0.5, 3.0, ...) are
 * written as literals: they encode as instruction immediates. */
static __constant__ double GKC[16] = {
    13.0 / 12.0,                                        /* 0  smoothness: (13/12) a^2 */
    ((210.0 - GKS_SQRT3) / 1080.0) / (11.0 / 18.0),     /* 1  Gauss-point linear weight dA / dB */
    ((210.0 + GKS_SQRT3) / 1080.0) / (11.0 / 18.0),     /* 2  Gauss-point linear weight dC / dB */
    GKS_SQRT3 / 12.0,                                   /* 3  h = x_G / 2, x_G = sqrt(3)/6 */
    1.0 / 6.0,                                          /* 4  edge linear weight .1/.6 */
    1.0 / 12.0,                                         /* 5 */
    -(1.0 / 12.0 - GKS_SQRT3 / 54.0),                                     /* 6  e1 = -k0 */
    -((1.0 / 12.0 - GKS_SQRT3 / 54.0) + (-2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0)), /* 7  e2 = -(k0+k1) */
    (2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0) + (-1.0 / 12.0 - GKS_SQRT3 / 54.0),    /* 8  e3 = k3+k4 */
    -1.0 / 12.0 - GKS_SQRT3 / 54.0,                                       /* 9  e4 = k4 */
    0, 0, 0, 0, 0, 0};

/* reciprocal to fp64 round-off: hardware seed (2^-23) + two Newton steps, no slow path */
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

/* Shared front end of every WENO5-JS evaluation, in difference form.  With D_m = q_m - q_{m-1}:
 *   second differences a_k (sub-stencil curvature), centred slopes g_k (twice the slope of sub-stencil k's
 *   quadratic at the centre of the middle cell; g0 = q0-4q1+3q2, g1 = q3-q1, g2 = -(3q2-4q3+q4)),
 *   Jiang-Shu beta_k = 13/12 a_k^2 + 1/4 g_k^2, and the common-denominator factors
 *   t0 = s1 s2, t1 = s0 s2, t2 = s0 s1 with s_k = (eps + beta_k)^2. */
struct JsFront {
  double a0, a1, a2, g0, g1, g2, t0, t1, t2;
};
__device__ __forceinline__ void js_front(double D1, double D2, double D3, double D4, double eps, JsFront &f) {
  f.a0 = D2 - D1;
  f.a1 = D3 - D2;
  f.a2 = D4 - D3;
  f.g0 = fma(3.0, D2, -D1);
  f.g1 = D2 + D3;
  f.g2 = fma(3.0, D3, -D4);
  const double k13 = GKC[0];
  double s0 = fma(0.25 * f.g0, f.g0, fma(k13 * f.a0, f.a0, eps));
  double s1 = fma(0.25 * f.g1, f.g1, fma(k13 * f.a1, f.a1, eps));
  double s2 = fma(0.25 * f.g2, f.g2, fma(k13 * f.a2, f.a2, eps));
  s0 *= s0;
  s1 *= s1;
  s2 *= s2;
  f.t0 = s1 * s2;
  f.t1 = s0 * s2;
  f.t2 = s0 * s1;
}

/* WENO5-JS values at BOTH edges of the middle cell: vl at x = -1/2, vr at x = +1/2.
 * Candidate k at x = +-1/2 is q2 +- g_k/4 + a_k/12; linear weights (.1,.6,.3) right, mirrored left;
 * nonlinear weights over the common denominator (one reciprocal for both edges). */
__device__ __forceinline__ void weno5_edges(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vl, double &vr) {
  JsFront f;
  js_front(q1 - q0, q2 - q1, q3 - q2, q4 - q3, eps, f);
  const double w6 = GKC[4];
  const double ar0 = w6 * f.t0, ar2 = 0.5 * f.t2; /* (.1,.6,.3)/.6 */
  const double al0 = 0.5 * f.t0, al2 = w6 * f.t2; /* (.3,.6,.1)/.6 */
  const double P0 = fma(3.0, f.g0, f.a0), P1 = fma(3.0, f.g1, f.a1), P2 = fma(3.0, f.g2, f.a2);
  const double M0 = fma(-3.0, f.g0, f.a0), M1 = fma(-3.0, f.g1, f.a1), M2 = fma(-3.0, f.g2, f.a2);
  const double numr = fma(ar2, P2, fma(f.t1, P1, ar0 * P0)), denr = ar0 + f.t1 + ar2;
  const double numl = fma(al2, M2, fma(f.t1, M1, al0 * M0)), denl = al0 + f.t1 + al2;
  const double inv = fast_rcp(denr * denl) * GKC[5];
  vr = fma(numr * denl, inv, q2);
  vl = fma(numl * denr, inv, q2);
}

/* WENO5-JS values at the Gauss points (vm at -sqrt(3)/6, vp at +sqrt(3)/6; S7) and, if SLOPE,
 * the derivative of the quartic through the 5 averages there (S8; per unit cell width).
 * At x^2 = 1/12 the quadratic term of every candidate vanishes: candidate k is q2 +- (x_G/2) g_k. */
template <bool SLOPE>
__device__ __forceinline__ void weno5_gauss_slope(double q0, double q1, double q2, double q3, double q4, double eps,
                                                  double &vm, double &vp, double &sm, double &sp) {
  const double D1 = q1 - q0, D2 = q2 - q1, D3 = q3 - q2, D4 = q4 - q3;
  JsFront f;
  js_front(D1, D2, D3, D4, eps, f);
  const double dA = GKC[1], dC = GKC[2], h = GKC[3];
  const double ap0 = dA * f.t0, ap2 = dC * f.t2;
  const double am0 = dC * f.t0, am2 = dA * f.t2;
  const double c1 = f.t1 * f.g1;
  const double nump = fma(ap2, f.g2, fma(ap0, f.g0, c1)), denp = ap0 + f.t1 + ap2;
  const double numm = fma(am2, f.g2, fma(am0, f.g0, c1)), denm = am0 + f.t1 + am2;
  const double inv = fast_rcp(denp * denm) * h;
  vp = fma(nump * denm, inv, q2);
  vm = fma(-(numm * denp), inv, q2);
  if (SLOPE) {
    const double e1 = GKC[6], e2 = GKC[7], e3 = GKC[8], e4 = GKC[9];
    sp = fma(e4, D4, fma(e3, D3, fma(e2, D2, e1 * D1)));
    sm = fma(e1, D4, fma(e2, D3, fma(e3, D2, e4 * D1)));
  }
}

__device__ __forceinline__ void weno5_gauss(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vm, double &vp) {
  double d0, d1;
  weno5_gauss_slope<false>(q0, q1, q2, q3, q4, eps, vm, vp, d0, d1);
}

/* derivative of the quartic through the 5 averages at the Gauss points, per unit cell width (S8) */
__device__ __forceinline__ void quartic_slope_gauss(double q0, double q1, double q2, double q3, double q4,
                                                    double &sm, double &sp) {
  const double D1 = q1 - q0, D2 = q2 - q1, D3 = q3 - q2, D4 = q4 - q3;
  const double e1 = GKC[6], e2 = GKC[7], e3 = GKC[8], e4 = GKC[9];
  sp = fma(e4, D4, fma(e3, D3, fma(e2, D2, e1 * D1)));
  sm = fma(e1, D4, fma(e2, D3, fma(e3, D2, e4 * D1)));
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
  const double Ul = Ql[1 + DIR] * fast_rcp(Ql[0]), Ur = Qr[1 + DIR] * fast_rcp(Qr[0]);
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
  const double ir = fast_rcp(rho);
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
