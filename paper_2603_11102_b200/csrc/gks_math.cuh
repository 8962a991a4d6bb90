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
    13.0 / 3.0,                                         /* 0  smoothness, scaled by 4: (13/3) a^2 + g^2 */
    ((210.0 - GKS_SQRT3) / 1080.0) / (11.0 / 18.0),     /* 1  Gauss-point linear weight dA / dB */
    ((210.0 + GKS_SQRT3) / 1080.0) / (11.0 / 18.0),     /* 2  Gauss-point linear weight dC / dB */
    GKS_SQRT3 / 12.0,                                   /* 3  h = x_G / 2, x_G = sqrt(3)/6 */
    1.0 / 6.0,                                          /* 4  edge linear weight .1/.6 */
    1.0 / 12.0,                                         /* 5 */
    -(1.0 / 12.0 - GKS_SQRT3 / 54.0),                                     /* 6  e1 = -k0 */
    -((1.0 / 12.0 - GKS_SQRT3 / 54.0) + (-2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0)), /* 7  e2 = -(k0+k1) */
    (2.0 / 3.0 + 13.0 * GKS_SQRT3 / 54.0) + (-1.0 / 12.0 - GKS_SQRT3 / 54.0),    /* 8  e3 = k3+k4 */
    -1.0 / 12.0 - GKS_SQRT3 / 54.0,                                       /* 9  e4 = k4 */
    (GKS_SQRT3 / 12.0) * (11.0 / 18.0),                 /* 10 h dB: linear-weight variant */
    0, 0, 0, 0, 0};

/* reciprocal to fp64 round-off: hardware seed (2^-23) + two Newton steps, no slow path */
__device__ __forceinline__ double fast_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

/* reciprocal from the hardware seed r0 (2^-23) with one cubic correction: 1/x = r0 (1 + e + e^2 + O(e^3)),
 * e = 1 - x r0; truncation below 2^-66, three dependent operations after the seed */
__device__ __forceinline__ double fast_rcp3(double x) {
  double r0;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0) : "d"(x));
  const double e = fma(-x, r0, 1.0);
  return fma(r0, fma(e, e, e), r0);
}

/* Shared front end of every WENO5-JS evaluation, in difference form.  With D_m = q_m - q_{m-1}:
 *   second differences a_k (sub-stencil curvature), centred slopes g_k (twice the slope of sub-stencil k's
 *   quadratic at the centre of the middle cell; g0 = q0-4q1+3q2, g1 = q3-q1, g2 = -(3q2-4q3+q4)),
 *   Jiang-Shu beta_k = 13/12 a_k^2 + 1/4 g_k^2 (carried as 4 beta_k), and the common-denominator factors
 *   t0 = s1 s2, t1 = s0 s2, t2 = s0 s1 with s_k = (eps + beta_k)^2. */
/* N independent stencils at once: every statement is replicated N times back to back so that the
 * instruction stream interleaves N dependency chains (the fp64 pipe needs the ILP at 16 warps/SM). */
template <int N>
struct JsFrontV {
  double a0[N], a1[N], a2[N], g0[N], g1[N], g2[N], t0[N], t1[N], t2[N];
};
template <int N>
__device__ __forceinline__ void js_front_v(const double (&D1)[N], const double (&D2)[N], const double (&D3)[N],
                                           const double (&D4)[N], double eps /* 4 x the WENO epsilon */, JsFrontV<N> &f) {
  /* s_k = 4 (eps + beta_k) = (13/3) a_k^2 + g_k^2 + 4 eps: the common factor 4 (exact in binary) cancels
     in the weight ratios */
  const double k13 = GKC[0];
  const double eps4 = eps;   /* callers pass 4 eps (GksPhys::weno_eps4): a constant-bank operand, no register */
  double s0[N], s1[N], s2[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    f.a0[n] = D2[n] - D1[n];
    f.a1[n] = D3[n] - D2[n];
    f.a2[n] = D4[n] - D3[n];
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    f.g0[n] = fma(3.0, D2[n], -D1[n]);
    f.g1[n] = D2[n] + D3[n];
    f.g2[n] = fma(3.0, D3[n], -D4[n]);
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    s0[n] = fma(k13 * f.a0[n], f.a0[n], eps4);
    s1[n] = fma(k13 * f.a1[n], f.a1[n], eps4);
    s2[n] = fma(k13 * f.a2[n], f.a2[n], eps4);
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    s0[n] = fma(f.g0[n], f.g0[n], s0[n]);
    s1[n] = fma(f.g1[n], f.g1[n], s1[n]);
    s2[n] = fma(f.g2[n], f.g2[n], s2[n]);
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    s0[n] *= s0[n];
    s1[n] *= s1[n];
    s2[n] *= s2[n];
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    f.t0[n] = s1[n] * s2[n];
    f.t1[n] = s0[n] * s2[n];
    f.t2[n] = s0[n] * s1[n];
  }
}

template <int N>
__device__ __forceinline__ void fast_rcp_v(const double (&x)[N], double (&r)[N]) {
  double e[N];
#pragma unroll
  for (int n = 0; n < N; ++n) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r[n]) : "d"(x[n]));
#pragma unroll
  for (int n = 0; n < N; ++n) e[n] = fma(-x[n], r[n], 1.0);
#pragma unroll
  for (int n = 0; n < N; ++n) r[n] = fma(r[n], e[n], r[n]);
#pragma unroll
  for (int n = 0; n < N; ++n) e[n] = fma(-x[n], r[n], 1.0);
#pragma unroll
  for (int n = 0; n < N; ++n) r[n] = fma(r[n], e[n], r[n]);
}

/* WENO5-JS values at BOTH edges of the middle cell for N stencils: vl at x = -1/2, vr at x = +1/2.
 * Candidate k at x = +-1/2 is q2 +- g_k/4 + a_k/12; linear weights (.1,.6,.3) right, mirrored left;
 * nonlinear weights over the common denominator (one reciprocal for both edges). */
template <int N>
__device__ __forceinline__ void weno5_edges_v(const double (&q)[5][N], double eps, double (&vl)[N], double (&vr)[N]) {
  double D1[N], D2[N], D3[N], D4[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    D1[n] = q[1][n] - q[0][n];
    D2[n] = q[2][n] - q[1][n];
    D3[n] = q[3][n] - q[2][n];
    D4[n] = q[4][n] - q[3][n];
  }
  JsFrontV<N> f;
  js_front_v<N>(D1, D2, D3, D4, eps, f);
  const double w6 = GKC[4], w12 = GKC[5];
  double numr[N], numl[N], denr[N], denl[N], prod[N], r0[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    /* linear weights (.1,.6,.3)/.6 right, (.3,.6,.1)/.6 left; candidates 12 (p_k - q2) = a_k +- 3 g_k */
    const double ug0 = f.t0[n] * f.g0[n], ug1 = f.t1[n] * f.g1[n], ug2 = f.t2[n] * f.g2[n];
    const double ua0 = f.t0[n] * f.a0[n], ua1 = f.t1[n] * f.a1[n], ua2 = f.t2[n] * f.a2[n];
    const double Gr = fma(w6, ug0, fma(0.5, ug2, ug1)), Ar = fma(w6, ua0, fma(0.5, ua2, ua1));
    const double Gl = fma(0.5, ug0, fma(w6, ug2, ug1)), Al = fma(0.5, ua0, fma(w6, ua2, ua1));
    numr[n] = fma(3.0, Gr, Ar);
    numl[n] = fma(-3.0, Gl, Al);
    denr[n] = fma(w6, f.t0[n], fma(0.5, f.t2[n], f.t1[n]));
    denl[n] = fma(0.5, f.t0[n], fma(w6, f.t2[n], f.t1[n]));
    prod[n] = denr[n] * denl[n];
  }
#pragma unroll
  for (int n = 0; n < N; ++n) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0[n]) : "d"(prod[n]));
#pragma unroll
  for (int n = 0; n < N; ++n) {
    /* 1/prod = r0 (1 + e + e^2 + ...), e = 1 - prod r0 ~ 2^-23: the cubic truncation is below 2^-66 (one Newton step
       alone, 2^-46 of the correction, is visible in dF/dt, whose terms cancel to O(Ma^2): measured 5e-12 of max |dF/dt|) */
    const double e = fma(-prod[n], r0[n], 1.0);
    const double t = fma(e, e, e);
    const double rw = fma(r0[n], t, r0[n]) * w12;
    vr[n] = fma(numr[n] * denl[n], rw, q[2][n]);
    vl[n] = fma(numl[n] * denr[n], rw, q[2][n]);
  }
}

/* WENO5-JS values at the Gauss points (vm at -sqrt(3)/6, vp at +sqrt(3)/6; S7) and the derivative of
 * the quartic through the 5 averages there (S8; per unit cell width; dead code when unused), N stencils.
 * At x^2 = 1/12 the quadratic term of every candidate vanishes: candidate k is q2 +- (x_G/2) g_k. */
template <int N, bool LIN = false>
__device__ __forceinline__ void weno5_gauss_v(const double (&q)[5][N], double eps, double (&vm)[N], double (&vp)[N],
                                              double (&sm)[N], double (&sp)[N]) {
  double D1[N], D2[N], D3[N], D4[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    D1[n] = q[1][n] - q[0][n];
    D2[n] = q[2][n] - q[1][n];
    D3[n] = q[3][n] - q[2][n];
    D4[n] = q[4][n] - q[3][n];
  }
  if (LIN) {
    /* scheme variant: the candidates q2 +- h g_k combined with the LINEAR weights (quartic interpolation) */
    const double dA = GKC[1], dC = GKC[2], hb = GKC[10];
    const double e1 = GKC[6], e2 = GKC[7], e3 = GKC[8], e4 = GKC[9];
#pragma unroll
    for (int n = 0; n < N; ++n) {
      const double g0 = fma(3.0, D2[n], -D1[n]), g1 = D2[n] + D3[n], g2 = fma(3.0, D3[n], -D4[n]);
      vp[n] = fma(hb, fma(dA, g0, fma(dC, g2, g1)), q[2][n]);
      vm[n] = fma(-hb, fma(dC, g0, fma(dA, g2, g1)), q[2][n]);
      sp[n] = fma(e4, D4[n], fma(e3, D3[n], fma(e2, D2[n], e1 * D1[n])));
      sm[n] = fma(e1, D4[n], fma(e2, D3[n], fma(e3, D2[n], e4 * D1[n])));
    }
    return;
  }
  JsFrontV<N> f;
  js_front_v<N>(D1, D2, D3, D4, eps, f);
  const double dA = GKC[1], dC = GKC[2], h = GKC[3];
  double nump[N], numm[N], denp[N], denm[N], prod[N], r0[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    const double u0 = f.t0[n] * f.g0[n], u1 = f.t1[n] * f.g1[n], u2 = f.t2[n] * f.g2[n];
    nump[n] = fma(dA, u0, fma(dC, u2, u1));
    numm[n] = fma(dC, u0, fma(dA, u2, u1));
    denp[n] = fma(dA, f.t0[n], fma(dC, f.t2[n], f.t1[n]));
    denm[n] = fma(dC, f.t0[n], fma(dA, f.t2[n], f.t1[n]));
    prod[n] = denp[n] * denm[n];
  }
#pragma unroll
  for (int n = 0; n < N; ++n) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r0[n]) : "d"(prod[n]));
  const double e1 = GKC[6], e2 = GKC[7], e3 = GKC[8], e4 = GKC[9];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    /* 1/prod = r0 (1 + e + e^2 + ...), e = 1 - prod r0 ~ 2^-23: the cubic truncation is below 2^-66 */
    const double e = fma(-prod[n], r0[n], 1.0);
    const double t = fma(e, e, e);
    const double rh = fma(r0[n], t, r0[n]) * h;
    vp[n] = fma(nump[n] * denm[n], rh, q[2][n]);
    vm[n] = fma(-(numm[n] * denp[n]), rh, q[2][n]);
    sp[n] = fma(e4, D4[n], fma(e3, D3[n], fma(e2, D2[n], e1 * D1[n])));
    sm[n] = fma(e1, D4[n], fma(e2, D3[n], fma(e3, D2[n], e4 * D1[n])));
  }
}

/* scalar wrappers (unfused cross-check kernels) */
__device__ __forceinline__ void weno5_edges(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vl, double &vr) {
  const double q[5][1] = {{q0}, {q1}, {q2}, {q3}, {q4}};
  double l[1], r[1];
  weno5_edges_v<1>(q, eps, l, r);
  vl = l[0];
  vr = r[0];
}
__device__ __forceinline__ void weno5_gauss(double q0, double q1, double q2, double q3, double q4,
                                            double eps, double &vm, double &vp, bool linear = false) {
  const double q[5][1] = {{q0}, {q1}, {q2}, {q3}, {q4}};
  double m[1], p[1], a[1], b[1];
  if (linear) weno5_gauss_v<1, true>(q, eps, m, p, a, b);
  else weno5_gauss_v<1, false>(q, eps, m, p, a, b);
  vm = m[0];
  vp = p[0];
}
__device__ __forceinline__ void quartic_slope_gauss(double q0, double q1, double q2, double q3, double q4,
                                                    double &sm, double &sp) {
  const double D1 = q1 - q0, D2 = q2 - q1, D3 = q3 - q2, D4 = q4 - q3;
  const double e1 = GKC[6], e2 = GKC[7], e3 = GKC[8], e4 = GKC[9];
  sp = fma(e4, D4, fma(e3, D3, fma(e2, D2, e1 * D1)));
  sm = fma(e1, D4, fma(e2, D3, fma(e3, D2, e4 * D1)));
}

/* 12 x the index-space slope at the face between qb and qc from 4 averages qa,qb,qc,qd (S5); the factor 1/12 is
 * folded into the metric table GksGrid::inv_12hn */
__device__ __forceinline__ double normal_slope12(double qa, double qb, double qc, double qd) {
  return fma(15.0, qc - qb, qa - qd);
}

/* Half-range Maxwellian moments (S4) need erf(z) and exp(-z^2), z = sqrt(lambda) U_n.  For |z| <= 1/2
 * (normal Mach number below 0.7: every cell of a weakly compressible flow) both come from their
 * Maclaurin series in z^2 (terms fall like 0.25^n/n!; 12 and 14 terms reach 1e-17), about 26 DFMA with
 * constant-bank coefficients; otherwise the CUDA math library is used. */
#define GKS_2ISPI 1.1283791670955125739 /* 2/sqrt(pi) */
static __constant__ double GK_ERF[12] = {
    GKS_2ISPI / 1.0,          -GKS_2ISPI / 3.0,           GKS_2ISPI / (2.0 * 5.0),       -GKS_2ISPI / (6.0 * 7.0),
    GKS_2ISPI / (24.0 * 9.0), -GKS_2ISPI / (120.0 * 11.0), GKS_2ISPI / (720.0 * 13.0),   -GKS_2ISPI / (5040.0 * 15.0),
    GKS_2ISPI / (40320.0 * 17.0), -GKS_2ISPI / (362880.0 * 19.0), GKS_2ISPI / (3628800.0 * 21.0),
    -GKS_2ISPI / (39916800.0 * 23.0)};
static __constant__ double GK_EXP[14] = {1.0, -1.0, 1.0 / 2.0, -1.0 / 6.0, 1.0 / 24.0, -1.0 / 120.0, 1.0 / 720.0,
                                         -1.0 / 5040.0, 1.0 / 40320.0, -1.0 / 362880.0, 1.0 / 3628800.0,
                                         -1.0 / 39916800.0, 1.0 / 479001600.0, -1.0 / 6227020800.0};

/* erf(z) and exp(-z^2) */
__device__ __forceinline__ void erf_expm2(double z, double &erfz, double &ex) {
  const double w = z * z;
  if (w <= 0.25) {
    double pe = GK_ERF[11], px = GK_EXP[13];
    px = fma(px, w, GK_EXP[12]);
#pragma unroll
    for (int n = 10; n >= 0; --n) {
      pe = fma(pe, w, GK_ERF[n]);
      px = fma(px, w, GK_EXP[n + 1]);
    }
    px = fma(px, w, GK_EXP[0]);
    erfz = pe * z;
    ex = px;
  } else {
    erfz = erf(z);
    ex = exp(-w);
  }
}

/* N independent arguments at once (statement-interleaved Horner chains); the library fallback for
 * |z| > 1/2 is taken per element afterwards */
template <int N>
__device__ __forceinline__ void erf_expm2_v(const double (&z)[N], double (&erfz)[N], double (&ex)[N]) {
  double w[N], pe[N], px[N];
#pragma unroll
  for (int n = 0; n < N; ++n) {
    w[n] = z[n] * z[n];
    pe[n] = GK_ERF[11];
    px[n] = fma(GK_EXP[13], w[n], GK_EXP[12]);
  }
#pragma unroll
  for (int k = 10; k >= 0; --k) {
#pragma unroll
    for (int n = 0; n < N; ++n) {
      pe[n] = fma(pe[n], w[n], GK_ERF[k]);
      px[n] = fma(px[n], w[n], GK_EXP[k + 1]);
    }
  }
#pragma unroll
  for (int n = 0; n < N; ++n) {
    erfz[n] = pe[n] * z[n];
    ex[n] = fma(px[n], w[n], GK_EXP[0]);
    if (w[n] > 0.25) {
      erfz[n] = erf(z[n]);
      ex[n] = exp(-w[n]);
    }
  }
}

/* erf(z) and exp(-z^2) inside a warp-uniform choice of series length: when every lane has z^2 <= 1/64
 * (normal Mach number below 0.18; garbage lanes with NaN count as small) 8 terms of either Maclaurin
 * series reach 1e-19; otherwise the 12/14-term series or the library (erf_expm2). */
__device__ __forceinline__ void erf_expm2_warp(double z, double &erfz, double &ex) {
  const double w = z * z;
  const bool small = !(w > 1.0 / 64.0);
  if (__all_sync(0xffffffffu, small)) {
    double pe = GK_ERF[7], px = GK_EXP[7];
#pragma unroll
    for (int n = 6; n >= 0; --n) {
      pe = fma(pe, w, GK_ERF[n]);
      px = fma(px, w, GK_EXP[n]);
    }
    erfz = pe * z;
    ex = px;
  } else {
    erf_expm2(z, erfz, ex);
  }
}

/* one of the two functions per lane: func = 0 -> erf(z), func = 1 -> exp(-z^2); the lanes of a warp run the
 * same Horner recurrence on their own coefficient set cf[n] = func ? GK_EXP[n] : GK_ERF[n], chosen once per thread
 * (series length chosen warp-uniformly as above) */
__device__ __forceinline__ void series_coefficients(int func, double (&cf)[8]) {
#pragma unroll
  for (int n = 0; n < 8; ++n) cf[n] = func ? GK_EXP[n] : GK_ERF[n];
}
__device__ __forceinline__ double erf_or_expm2_warp(double z, int func, const double *cf /* 8 coefficients of this lane's function */) {
  const double w = z * z;
  const bool small = !(w > 1.0 / 64.0);
  if (__all_sync(0xffffffffu, small)) {
    double p = cf[7];
#pragma unroll
    for (int n = 6; n >= 0; --n) p = fma(p, w, cf[n]);
    return func ? p : p * z;
  }
  double erfz, ex;
  erf_expm2(z, erfz, ex);
  return func ? ex : erfz;
}

/* collision factors from the normal velocities of the left / right states (S4):
 * el = <u^0>_{>0}(Ul), xl = exp(-lam Ul^2)/(2 sqrt(pi lam)); er = <u^0>_{<0}(Ur), xr likewise (positive) */
__device__ __forceinline__ void collision_factors(double Ul, double Ur, double lambda, double &el,
                                                  double &xl, double &er, double &xr) {
  const double theta = sqrt(lambda);
  const double c = 0.5 / sqrt(3.14159265358979323846 * lambda);
  double fl, fr, gl, gr;
  erf_expm2(theta * Ul, fl, gl);
  erf_expm2(theta * Ur, fr, gr);
  el = 0.5 + 0.5 * fl; /* erfc(-z)/2 */
  er = 0.5 - 0.5 * fr; /* erfc(+z)/2 */
  xl = c * gl;
  xr = c * gr;
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

/* Gauss-point flux in closed form.  dQ[s][c] = d_s Q0_c, s = x,y,z.  F and dF/dt of direction DIR.
 * Written with w_si = d_s m_i - U_i d_s rho (= rho d_s U_i), so that only the reciprocal of rho that the
 * velocities need is taken:  Q_t = -div F_Euler,
 *   rho_t = -sum_s d_s m_s,   m_i,t = -sum_s U_s d_s m_i - U_i sum_s w_ss - RT d_i rho,
 *   dF/dt = (dF_Euler/dQ) Q_t:  dF_0 = m_n,t,  dF_i = U_n m_i,t + U_i (m_n,t - U_n rho_t) (+ RT rho_t for i = n),
 *   F_0 = m_n,  F_i = m_i U_n - (mu / rho)(w_ni + w_in) (+ rho RT for i = n);   n = DIR. */
template <int DIR, bool NEED_F>
__device__ __forceinline__ void gauss_point_flux(const double Q0[4], const double dQ[3][4], double RT,
                                                 double mu, double F[4], double dF[4]) {
  const double rho = Q0[0];
  const double ir = fast_rcp3(rho);
  const double u[3] = {Q0[1] * ir, Q0[2] * ir, Q0[3] * ir};
  const double ud = u[DIR];
  double wd[3]; /* w_ss */
#pragma unroll
  for (int i = 0; i < 3; ++i) wd[i] = fma(-u[i], dQ[i][0], dQ[i][1 + i]);
  const double trw = (wd[0] + wd[1]) + wd[2];
  const double divm = (dQ[0][1] + dQ[1][2]) + dQ[2][3]; /* -rho_t */
  double m_t[3];
#pragma unroll
  for (int i = 0; i < 3; ++i)
    m_t[i] = fma(-u[0], dQ[0][1 + i], fma(-u[1], dQ[1][1 + i], fma(-u[2], dQ[2][1 + i], fma(-u[i], trw, -RT * dQ[i][0]))));
  const double k = fma(ud, divm, m_t[DIR]); /* m_n,t - U_n rho_t */
  dF[0] = m_t[DIR];
#pragma unroll
  for (int i = 0; i < 3; ++i) dF[1 + i] = fma(u[i], k, ud * m_t[i]);
  dF[1 + DIR] = fma(-RT, divm, dF[1 + DIR]);
  if (NEED_F) {
    const double mir = mu * ir;
    F[0] = Q0[1 + DIR];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const double wsum = i == DIR ? wd[DIR] + wd[DIR]
                                   : fma(-u[i], dQ[DIR][0], dQ[DIR][1 + i]) + fma(-ud, dQ[i][0], dQ[i][1 + DIR]);
      F[1 + i] = fma(-mir, wsum, Q0[1 + i] * ud);
    }
    F[1 + DIR] = fma(rho, RT, F[1 + DIR]);
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
