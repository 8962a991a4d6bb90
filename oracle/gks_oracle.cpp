/*
 * gks_oracle.cpp — the CPU ORACLE for the S2O4 gas-kinetic step with ALM + IBM forcing.
 *
 * TEST INFRASTRUCTURE ONLY (see gks_oracle.h).  Plain, slow, fp64, one loop nest per step of the
 * method, in the paper's order and notation.  Nothing here is tuned; OpenMP is used only across
 * independent faces / cells.  It shares no code, header, table or constant with the CUDA path.
 *
 * Passages followed (PAPER.md = /root/reference/PAPER.md, arxiv/paper_2603_11102):
 *   Eq. 2   isothermal Maxwellian, lambda = 1/(2RT)
 *   Eq. 4-5 finite-volume operator L
 *   Eq. 6   2x2 Gauss points per face
 *   Eq. 7   f = g0 (1 - tau (a1 u + a2 v + a3 w + A) + A t), tau=mu/p
 *   Eq. 8   <a_s> = dQ0/ds, <a1 u + a2 v + a3 w + A> = 0
 *   WENO5 [30], dimension-by-dimension; two-stage fourth-order
 *   Appendix: moment recursion, 4x4 solve, A from compatibility
 *   Eq. 10  ALM Gaussian projection, cut at 3 eps
 *   Eq. 11-12 IBM direct forcing
 *   Eq. 13  momentum update with body force
 *   multi-direct-forcing passes of the IBM, stop rule
 *   ALM front half: trilinear sampling, Eq. 9, free-stream correction
 *   Eq. 14  tip correction
 *   CFL time step
 * Readings S1..S27 (where the paper is silent) are those of DESIGN.md / SURVEY.md §8(c).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): moment recursion vs quadrature (P1), polynomial
 * exactness of every reconstruction operator (P2), Appendix solve (P3), collision special cases
 * (P4), Navier-Stokes flux identity + brute-force velocity-space quadrature (P5, P13), free-stream
 * preservation (P6), conservation (P7), order of accuracy on an exact simple wave (P8), viscous
 * decay (P9), acoustic speed (P10), ALM integral (P11), IBM delta identities (P12), axis
 * permutation symmetry (P14), IBM passes: closed-form contraction of an isolated point (P15), CFL time step:
 * hand-worked numbers (P16), ALM front half: geometry, exact sampling of trilinear fields, lift normal / drag
 * parallel to the relative flow, correction identities, a worked tip factor (P17), linear-weight tangential
 * variant: SURVEY's value row, exactness for quartics, order of accuracy (P18), stretched-grid metrics (S10):
 * the Couette stress -mu a through every face family and the decay rate of a wall-bounded vortex, both second
 * order under refinement (P19), inflow density (S19): the Rankine-Hugoniot plateau, velocity and injected mass of
 * the piston problem (P20), convective outflow (S20): an exactly advected vortical pulse leaves without reflection
 * (P21), no-slip wall (S17) and body force: decaying shear mode and steady Poiseuille profile between walls (P22),
 * mirror symmetry of the whole step with every boundary kind, ALM and IBM (P23).
 * The paper prints no numbers for S10, S17, S19, S20; the pins are exact solutions of the equations it solves.
 */
#include "gks_oracle.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

namespace {

const int NG = 3; /* ghost layers per side: the widest stencil reaches 3 cells beyond a face */
const double PI = 3.14159265358979323846264338327950288;

std::string g_error;
int fail(const std::string &m) {
  g_error = m;
  return 1;
}

enum { BC_PERIODIC = 0, BC_NOSLIP = 1, BC_SLIP = 2, BC_INFLOW = 3, BC_OUTFLOW = 4, BC_EXTRAP = 5 };

/* ------------------------------------------------------------------------------------------
 * Appendix: moments of the Maxwellian, <u^0> = 1, <u^1> = U,
 * <u^{n+2}> = (n+1)/(2 lambda) <u^n> + U <u^{n+1}>.
 * ------------------------------------------------------------------------------------------ */
void moments(double U, double lambda, int nmax, double *M) {
  M[0] = 1.0;
  if (nmax >= 1) M[1] = U;
  for (int n = 0; n + 2 <= nmax; ++n) M[n + 2] = (n + 1) / (2.0 * lambda) * M[n] + U * M[n + 1];
}

/* Appendix solve, reading S2: d = (1/rho0) dQ0/ds,
 * r_m = d_m - U_m d_1, a^m = 2 lambda r_m (m = 2,3,4), a^1 = d_1 - U a^2 - V a^3 - W a^4. */
void micro_solve(double U, double V, double W, double lambda, const double d[4], double a[4]) {
  const double r2 = d[1] - U * d[0];
  const double r3 = d[2] - V * d[0];
  const double r4 = d[3] - W * d[0];
  a[1] = 2.0 * lambda * r2;
  a[2] = 2.0 * lambda * r3;
  a[3] = 2.0 * lambda * r4;
  a[0] = d[0] - U * a[1] - V * a[2] - W * a[3];
}

/* ------------------------------------------------------------------------------------------
 * Reconstruction operators (ref [30] Jiang-Shu; readings S5-S8).
 * ------------------------------------------------------------------------------------------ */
/* Jiang-Shu smoothness indicators of the three 3-cell sub-stencils */
void js_beta(const double q[5], double beta[3]) {
  const double a0 = q[0] - 2.0 * q[1] + q[2], b0 = q[0] - 4.0 * q[1] + 3.0 * q[2];
  const double a1 = q[1] - 2.0 * q[2] + q[3], b1 = q[1] - q[3];
  const double a2 = q[2] - 2.0 * q[3] + q[4], b2 = 3.0 * q[2] - 4.0 * q[3] + q[4];
  beta[0] = 13.0 / 12.0 * a0 * a0 + 0.25 * b0 * b0;
  beta[1] = 13.0 / 12.0 * a1 * a1 + 0.25 * b1 * b1;
  beta[2] = 13.0 / 12.0 * a2 * a2 + 0.25 * b2 * b2;
}

/* nonlinear combination: alpha_k = d_k/(eps + beta_k)^2, w_k = alpha_k / sum(alpha) */
double js_combine(const double p[3], const double d[3], const double beta[3], double eps) {
  double alpha[3], s = 0.0;
  for (int k = 0; k < 3; ++k) {
    alpha[k] = d[k] / ((eps + beta[k]) * (eps + beta[k]));
    s += alpha[k];
  }
  double v = 0.0;
  for (int k = 0; k < 3; ++k) v += (alpha[k] / s) * p[k];
  return v;
}

/* WENO5-JS value at the right edge (x = +1/2) of the middle cell q[2] */
double weno5_face(const double q[5], double eps) {
  const double p[3] = {(2.0 * q[0] - 7.0 * q[1] + 11.0 * q[2]) / 6.0,
                       (-q[1] + 5.0 * q[2] + 2.0 * q[3]) / 6.0,
                       (2.0 * q[2] + 5.0 * q[3] - q[4]) / 6.0};
  const double d[3] = {0.1, 0.6, 0.3};
  double beta[3];
  js_beta(q, beta);
  return js_combine(p, d, beta, eps);
}

/* WENO5-JS value at the Gauss point x = +sqrt(3)/6 (cell widths from the centre of q[2]).
 * Candidates are the quadratics matching the averages of each 3-cell sub-stencil, evaluated at
 * the point; linear weights make their combination the quartic through all 5 averages (S7). */
double weno5_gauss_plus(const double q[5], double eps) {
  const double s3 = std::sqrt(3.0);
  const double p[3] = {s3 / 12.0 * q[0] - s3 / 3.0 * q[1] + (1.0 + s3 / 4.0) * q[2],
                       -s3 / 12.0 * q[1] + q[2] + s3 / 12.0 * q[3],
                       (1.0 - s3 / 4.0) * q[2] + s3 / 3.0 * q[3] - s3 / 12.0 * q[4]};
  const double d[3] = {(210.0 - s3) / 1080.0, 11.0 / 18.0, (210.0 + s3) / 1080.0};
  double beta[3];
  js_beta(q, beta);
  return js_combine(p, d, beta, eps);
}

/* The same candidates combined with the LINEAR weights d_k (reading S7's alternative): the value
 * at the Gauss point of the quartic through all five averages. */
double linear5_gauss_plus(const double q[5]) {
  const double s3 = std::sqrt(3.0);
  const double p[3] = {s3 / 12.0 * q[0] - s3 / 3.0 * q[1] + (1.0 + s3 / 4.0) * q[2],
                       -s3 / 12.0 * q[1] + q[2] + s3 / 12.0 * q[3],
                       (1.0 - s3 / 4.0) * q[2] + s3 / 3.0 * q[3] - s3 / 12.0 * q[4]};
  const double d[3] = {(210.0 - s3) / 1080.0, 11.0 / 18.0, (210.0 + s3) / 1080.0};
  return d[0] * p[0] + d[1] * p[1] + d[2] * p[2];
}

/* tangential reconstruction of one field: WENO5-JS (S7) or, with `linear`, the linear-weight variant */
void tangential_gauss(const double q[5], double eps, bool linear, double out[2]);

/* values at (-sqrt(3)/6, +sqrt(3)/6); the minus point is the mirror image (reverse the stencil) */
void weno5_gauss(const double q[5], double eps, double out[2]) {
  const double qr[5] = {q[4], q[3], q[2], q[1], q[0]};
  out[0] = weno5_gauss_plus(qr, eps);
  out[1] = weno5_gauss_plus(q, eps);
}

void tangential_gauss(const double q[5], double eps, bool linear, double out[2]) {
  if (!linear) {
    weno5_gauss(q, eps, out);
    return;
  }
  const double qr[5] = {q[4], q[3], q[2], q[1], q[0]};
  out[0] = linear5_gauss_plus(qr);
  out[1] = linear5_gauss_plus(q);
}

/* derivative at x = +-sqrt(3)/6 of the quartic whose 5 cell averages are q, per unit cell width (S8) */
void quartic_slope_gauss(const double q[5], double out[2]) {
  const double s3 = std::sqrt(3.0);
  const double c[5] = {1.0 / 12.0 - s3 / 54.0, -2.0 / 3.0 + 13.0 * s3 / 54.0, -4.0 * s3 / 9.0,
                       2.0 / 3.0 + 13.0 * s3 / 54.0, -1.0 / 12.0 - s3 / 54.0};
  double plus = 0.0, minus = 0.0;
  for (int m = 0; m < 5; ++m) {
    plus += c[m] * q[m];
    minus += -c[m] * q[4 - m]; /* mirrored: reverse and negate */
  }
  out[0] = minus;
  out[1] = plus;
}

/* derivative at the face between q[1] and q[2] of the cubic matching 4 averages, per unit spacing (S5) */
double normal_slope(const double q[4]) { return (-(q[3] - q[0]) + 15.0 * (q[2] - q[1])) / 12.0; }

/* ------------------------------------------------------------------------------------------
 * Collision (reading S4): the equilibrium state at the face is the one whose conserved moments
 * equal those of the left Maxwellian over u_n > 0 plus the right Maxwellian over u_n < 0,
 * int psi g0 = int_{u_n>0} psi g_l + int_{u_n<0} psi g_r   ("g0 is the collisional equilibrium
 * state").  Half moments of a 1-D Maxwellian (mean U, lambda):
 *   <u^0>_{>0} = erfc(-sqrt(lambda) U)/2,  <u^1>_{>0} = U <u^0>_{>0} + exp(-lambda U^2)/(2 sqrt(pi lambda))
 *   <u^0>_{<0} = erfc(+sqrt(lambda) U)/2,  <u^1>_{<0} = U <u^0>_{<0} - exp(-lambda U^2)/(2 sqrt(pi lambda))
 * ------------------------------------------------------------------------------------------ */
void collision(const double Ql[4], const double Qr[4], int dir, double RT, double Q0[4]) {
  const double lambda = 1.0 / (2.0 * RT);
  const double theta = std::sqrt(lambda);
  const int n = 1 + dir; /* index of the momentum component normal to the face */
  const double Ul = Ql[n] / Ql[0], Ur = Qr[n] / Qr[0];
  const double el = 0.5 * std::erfc(-theta * Ul);
  const double xl = 0.5 * std::exp(-lambda * Ul * Ul) / std::sqrt(PI * lambda);
  const double er = 0.5 * std::erfc(theta * Ur);
  const double xr = -0.5 * std::exp(-lambda * Ur * Ur) / std::sqrt(PI * lambda);
  Q0[0] = Ql[0] * el + Qr[0] * er;
  for (int c = 1; c < 4; ++c) {
    if (c == n)
      Q0[c] = Ql[0] * (Ul * el + xl) + Qr[0] * (Ur * er + xr);
    else
      Q0[c] = Ql[c] * el + Qr[c] * er;
  }
}

/* ------------------------------------------------------------------------------------------
 * Gauss-point flux (Eq. 6-8 and Appendix).  Q0 and its slopes dQ[s][c] (s = x,y,z) are given.
 *   <.> = (1/rho0) int (.) g0 dXi,  M(al,be,ga) = <u^al><v^be><w^ga>
 *   mom(a; al,be,ga) = <a u^al v^be w^ga>,  a = a^1 + a^2 u + a^3 v + a^4 w
 *   Psi(a; al,be,ga) = <a psi u^al v^be w^ga>,  psi = (1,u,v,w)
 *   B = <A psi> = -[Psi(a_x;1,0,0) + Psi(a_y;0,1,0) + Psi(a_z;0,0,1)]
 *   A = Appendix solve applied to B
 *   x-face:  F = rho0 { Psi(1;1,0,0) - tau [Psi(a_x;2,0,0) + Psi(a_y;1,1,0) + Psi(a_z;1,0,1) + Psi(A;1,0,0)] }
 *            dF/dt = rho0 Psi(A;1,0,0)                      (Eq. 7 is linear in t: F(t) = F + t dF/dt)
 *   tau = mu/p = rho_ref nu/(rho0 RT)  (reading S3).  y/z-faces raise the v/w exponent.
 * ------------------------------------------------------------------------------------------ */
struct Mom {
  double u[7], v[7], w[7];
  double M(int al, int be, int ga) const { return u[al] * v[be] * w[ga]; }
  double mom(const double a[4], int al, int be, int ga) const {
    return a[0] * M(al, be, ga) + a[1] * M(al + 1, be, ga) + a[2] * M(al, be + 1, ga) +
           a[3] * M(al, be, ga + 1);
  }
  void Psi(const double a[4], int al, int be, int ga, double out[4]) const {
    out[0] = mom(a, al, be, ga);
    out[1] = mom(a, al + 1, be, ga);
    out[2] = mom(a, al, be + 1, ga);
    out[3] = mom(a, al, be, ga + 1);
  }
};

void gauss_point_flux(const double Q0[4], const double dQ[3][4], int dir, double RT, double nu,
                      double rho_ref, double F[4], double dF[4]) {
  const double lambda = 1.0 / (2.0 * RT);
  const double rho0 = Q0[0];
  const double U = Q0[1] / rho0, V = Q0[2] / rho0, W = Q0[3] / rho0;
  Mom m;
  moments(U, lambda, 6, m.u);
  moments(V, lambda, 6, m.v);
  moments(W, lambda, 6, m.w);

  double a[3][4]; /* a_x, a_y, a_z */
  for (int s = 0; s < 3; ++s) {
    const double d[4] = {dQ[s][0] / rho0, dQ[s][1] / rho0, dQ[s][2] / rho0, dQ[s][3] / rho0};
    micro_solve(U, V, W, lambda, d, a[s]);
  }
  const int E[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};

  double B[4] = {0, 0, 0, 0}, t[4];
  for (int s = 0; s < 3; ++s) {
    m.Psi(a[s], E[s][0], E[s][1], E[s][2], t);
    for (int c = 0; c < 4; ++c) B[c] -= t[c];
  }
  double A[4];
  micro_solve(U, V, W, lambda, B, A);

  const double tau = rho_ref * nu / (rho0 * RT);
  const int *e = E[dir];
  const double one[4] = {1.0, 0.0, 0.0, 0.0};
  double eq[4], visc[4] = {0, 0, 0, 0}, At[4];
  m.Psi(one, e[0], e[1], e[2], eq);
  for (int s = 0; s < 3; ++s) {
    m.Psi(a[s], e[0] + E[s][0], e[1] + E[s][1], e[2] + E[s][2], t);
    for (int c = 0; c < 4; ++c) visc[c] += t[c];
  }
  m.Psi(A, e[0], e[1], e[2], At);
  for (int c = 0; c < 4; ++c) {
    F[c] = rho0 * (eq[c] - tau * (visc[c] + At[c]));
    dF[c] = rho0 * At[c];
  }
}

/* 3-point discrete delta (reading S13) */
double delta3(double r) {
  const double x = std::fabs(r);
  if (x <= 0.5) return (1.0 + std::sqrt(1.0 - 3.0 * x * x)) / 3.0;
  if (x <= 1.5) return (5.0 - 3.0 * x - std::sqrt(1.0 - 3.0 * (1.0 - x) * (1.0 - x))) / 6.0;
  return 0.0;
}

/* Eq. 10: Gaussian kernel per unit point force */
double alm_kernel(double r, double eps) {
  return std::exp(-(r / eps) * (r / eps)) / (eps * eps * eps * std::pow(PI, 1.5));
}

/* ------------------------------------------------------------------------------------------
 * Grid axis with 3 ghost layers (reading S10): rectilinear cells from face coordinates.
 * ------------------------------------------------------------------------------------------ */
struct Axis {
  int n = 0;
  bool periodic = false;
  std::vector<double> xf_, xc_, w_; /* faces -3..n+3, centres/widths -3..n+2 */
  double xf(int i) const { return xf_[i + NG]; }
  double xc(int i) const { return xc_[i + NG]; }
  double w(int i) const { return w_[i + NG]; }
  double lo() const { return xf(0); }
  double hi() const { return xf(n); }
  double len() const { return hi() - lo(); }

  void build(int n_, const double *faces, double x0, double dx, bool per) {
    n = n_;
    periodic = per;
    xf_.assign(n + 2 * NG + 1, 0.0);
    xc_.assign(n + 2 * NG, 0.0);
    w_.assign(n + 2 * NG, 0.0);
    if (!faces) { /* uniform: exact width dx everywhere */
      for (int i = -NG; i <= n + NG; ++i) xf_[i + NG] = x0 + i * dx;
      for (int i = -NG; i < n + NG; ++i) {
        w_[i + NG] = dx;
        xc_[i + NG] = x0 + (i + 0.5) * dx;
      }
      return;
    }
    for (int i = 0; i <= n; ++i) xf_[i + NG] = faces[i];
    for (int g = 1; g <= NG; ++g) {
      if (per) { /* periodic image */
        xf_[-g + NG] = faces[0] - (faces[n] - faces[n - g]);
        xf_[n + g + NG] = faces[n] + (faces[g] - faces[0]);
      } else { /* mirror image of the spacing about the boundary face */
        xf_[-g + NG] = faces[0] - (faces[g] - faces[0]);
        xf_[n + g + NG] = faces[n] + (faces[n] - faces[n - g]);
      }
    }
    for (int i = -NG; i < n + NG; ++i) {
      w_[i + NG] = xf_[i + 1 + NG] - xf_[i + NG];
      xc_[i + NG] = 0.5 * (xf_[i + NG] + xf_[i + 1 + NG]);
    }
  }
  /* interior cell containing x (x in [lo, hi]); -1 if outside */
  int find_cell(double x) const {
    if (!(x >= lo() && x <= hi())) return -1;
    int a = 0, b = n; /* xf(a) <= x <= xf(b) */
    while (b - a > 1) {
      const int mid = (a + b) / 2;
      if (x >= xf(mid)) a = mid; else b = mid;
    }
    return a;
  }
  /* centre of the cell with unwrapped index i (any integer on a periodic axis) */
  double xc_ext(int i) const {
    int m = i / n;
    int r = i - m * n;
    if (r < 0) { r += n; m -= 1; }
    return xc(r) + m * len();
  }
  static int wrap(int i, int n) { int r = i % n; return r < 0 ? r + n : r; }
};

} /* namespace */

/* ------------------------------------------------------------------------------------------ */
struct gkso_ctx {
  int n[3];
  Axis ax[3];
  double RT, nu, rho_ref, eps;
  int bc[6];
  double inflow[4];
  bool have_state = false;
  std::vector<double> W; /* padded state, [c][k][j][i] with ghosts; outflow ghosts are state */

  double g[3] = {0, 0, 0};
  int bulk_axis = -1;
  double bulk_target = 0;
  int n_alm = 0;
  std::vector<double> alm_pos, alm_force;
  double alm_eps = 0, alm_cut = 3.0;
  int n_ibm = 0;
  std::vector<double> ibm_pos, ibm_vol, ibm_vel;
  /* on-line actuator-line rotor (Eq. 9, Eq. 14): when set, every step samples the flow at
     the actuator points, evaluates the blade-element forces and replaces the point set of alm_set_points */
  struct Rotor {
    bool on = false;
    int nb = 0, np = 0, fs_corr = 0, tip_corr = 0;
    double hub[3] = {0, 0, 0}, R = 0, rhub = 0, omega = 0, theta0 = 0, uref = 0, time = 0;
    std::vector<double> chord, twist, pa, pcl, pcd;
    std::vector<double> radius, width;   /* per station (S28); even spacing when the caller gave none */
    std::vector<double> sec_r;           /* radii of the airfoil sections; pcl, pcd: [section][alpha] */
  } rotor;
  bool tangential_linear = false; /* scheme variant: linear weights in the two tangential passes (f4) */
  int ibm_maxit = 1;       /* multi-direct-forcing passes per step; 1 = single pass (S15) */
  double ibm_tol = 0.0;    /* stop once max_p |v_p - U_p| < tol (checked from the second pass on) */

  int P(int a) const { return n[a] + 2 * NG; }
  size_t ncell_p() const { return (size_t)P(0) * P(1) * P(2); }
  size_t ncell() const { return (size_t)n[0] * n[1] * n[2]; }
  /* padded index, i,j,k in [-3, n+3) */
  size_t id(int c, int i, int j, int k) const {
    return (((size_t)c * P(2) + (k + NG)) * P(1) + (j + NG)) * P(0) + (i + NG);
  }
  size_t idp(int c, const int p[3]) const { return id(c, p[0], p[1], p[2]); }
  /* interior index */
  size_t ii(int c, int i, int j, int k) const {
    return (((size_t)c * n[2] + k) * n[1] + j) * n[0] + i;
  }
};

namespace {

/* ------------------------------------------------------------------------------------------
 * Ghost fill (readings S17-S21).  Pass x covers interior (j,k); pass y covers all i (ghosts
 * included) and interior k; pass z covers all (i,j): edges and corners end up defined.
 * ------------------------------------------------------------------------------------------ */
void fill_ghost_line(const gkso_ctx &s, std::vector<double> &W, int a, int p[3]) {
  const int n = s.n[a];
  const double cs = std::sqrt(s.RT);
  for (int side = 0; side < 2; ++side) {
    const int kind = s.bc[2 * a + side];
    for (int g = 1; g <= NG; ++g) {
      const int ghost = side == 0 ? -g : n - 1 + g;
      const int mirror = side == 0 ? g - 1 : n - g;       /* interior cell at the same distance */
      const int image = side == 0 ? n - g : g - 1;        /* periodic image */
      const int first = side == 0 ? 0 : n - 1;            /* interior cell next to the face */
      int pg[3] = {p[0], p[1], p[2]}, pm[3] = {p[0], p[1], p[2]};
      pg[a] = ghost;
      double q[4];
      switch (kind) {
        case BC_PERIODIC:
          pm[a] = image;
          for (int c = 0; c < 4; ++c) q[c] = W[s.idp(c, pm)];
          break;
        case BC_NOSLIP: /* S17: rho even, all momenta odd */
          pm[a] = mirror;
          q[0] = W[s.idp(0, pm)];
          for (int c = 1; c < 4; ++c) q[c] = -W[s.idp(c, pm)];
          break;
        case BC_SLIP: /* S18: rho and tangential momenta even, normal momentum odd */
          pm[a] = mirror;
          for (int c = 0; c < 4; ++c) q[c] = W[s.idp(c, pm)];
          q[1 + a] = -q[1 + a];
          break;
        case BC_INFLOW: { /* S19: velocity prescribed, rho from the outgoing invariant U_n + c_s ln rho */
          pm[a] = first;
          const double sign = side == 0 ? -1.0 : 1.0; /* outward normal */
          const double rhoI = W[s.idp(0, pm)];
          const double UnI = sign * W[s.idp(1 + a, pm)] / rhoI;
          const double Unb = sign * s.inflow[1 + a];
          const double rhob = rhoI * std::exp((UnI - Unb) / cs);
          q[0] = rhob;
          for (int c = 1; c < 4; ++c) q[c] = rhob * s.inflow[c];
          break;
        }
        case BC_OUTFLOW: /* S20: ghosts are state, on every line this pass covers */
          continue;
        case BC_EXTRAP: /* S21 */
        default:
          pm[a] = first;
          for (int c = 0; c < 4; ++c) q[c] = W[s.idp(c, pm)];
          break;
      }
      for (int c = 0; c < 4; ++c) W[s.idp(c, pg)] = q[c];
    }
  }
}

/* the lines pass a covers: x interior (j,k); y all i, interior k; z all (i,j).  f(p) is called with p[a] = 0 */
template <class F>
void for_lines_of_pass(const gkso_ctx &s, int a, F f) {
  const int t1 = a == 0 ? 1 : 0, t2 = a == 2 ? 1 : 2;
  /* a tangential axis is covered with its ghosts when its own pass ran before this one */
  const int lo1 = t1 < a ? -NG : 0, hi1 = t1 < a ? s.n[t1] + NG : s.n[t1];
  const int lo2 = t2 < a ? -NG : 0, hi2 = t2 < a ? s.n[t2] + NG : s.n[t2];
  int p[3];
  p[a] = 0;
  for (p[t2] = lo2; p[t2] < hi2; ++p[t2])
    for (p[t1] = lo1; p[t1] < hi1; ++p[t1]) f(p);
}

void fill_pass(const gkso_ctx &s, std::vector<double> &W, int a) {
  for_lines_of_pass(s, a, [&](int p[3]) { fill_ghost_line(s, W, a, p); });
}

void fill_ghosts(const gkso_ctx &s, std::vector<double> &W) {
  for (int a = 0; a < 3; ++a) fill_pass(s, W, a);
}

/* ------------------------------------------------------------------------------------------
 * Face flux of one sweep direction (steps 2a-2g of DESIGN.md "oracle algorithm").
 * Face f (0..n_a) lies between cells f-1 and f along the normal axis a.
 * Tangential axes: t1 < t2 (reading S9: lower axis first).
 * Output Ff, dFf: [c][face-k][face-j][face-i] with n_a+1 entries along a, interior tangentially.
 * ------------------------------------------------------------------------------------------ */
struct FaceBox {
  int a, t1, t2;
  int nf, n1, n2;       /* faces along a; cells along t1, t2 */
  int P1, P2;           /* padded tangential sizes (range -2..n+1 => n+4) */
  size_t at(int f, int i1, int i2) const { return ((size_t)f * P1 + (i1 + 2)) * P2 + (i2 + 2); }
  size_t count() const { return (size_t)nf * P1 * P2; }
};

void face_flux(const gkso_ctx &s, const std::vector<double> &W, int dir, std::vector<double> &Ff,
               std::vector<double> &dFf) {
  FaceBox fb;
  fb.a = dir;
  fb.t1 = dir == 0 ? 1 : 0;
  fb.t2 = dir == 2 ? 1 : 2;
  fb.nf = s.n[fb.a] + 1;
  fb.n1 = s.n[fb.t1];
  fb.n2 = s.n[fb.t2];
  fb.P1 = fb.n1 + 4;
  fb.P2 = fb.n2 + 4;
  const Axis &An = s.ax[fb.a], &A1 = s.ax[fb.t1], &A2 = s.ax[fb.t2];
  const double eps = s.eps;

  /* 2a-2c: normal reconstruction and collision on every face whose tangential index is within
   * two cells of the interior.  Stored per face: Q0[4], Dn[4]. */
  std::vector<double> NQ(fb.count() * 8);
#pragma omp parallel for collapse(2) schedule(static)
  for (int f = 0; f < fb.nf; ++f)
    for (int i1 = -2; i1 < fb.n1 + 2; ++i1)
      for (int i2 = -2; i2 < fb.n2 + 2; ++i2) {
        double Ql[4], Qr[4], Dn[4], Q0[4];
        const double hn = An.xc(f) - An.xc(f - 1); /* centre-to-centre distance (S10) */
        for (int c = 0; c < 4; ++c) {
          double q[6]; /* cells f-3 .. f+2 */
          for (int m = 0; m < 6; ++m) {
            int p[3];
            p[fb.a] = f - 3 + m;
            p[fb.t1] = i1;
            p[fb.t2] = i2;
            q[m] = W[s.idp(c, p)];
          }
          const double ql[5] = {q[0], q[1], q[2], q[3], q[4]}; /* cells f-3..f+1: right edge of cell f-1 */
          const double qr[5] = {q[5], q[4], q[3], q[2], q[1]}; /* cells f+2..f-2: left edge of cell f  */
          Ql[c] = weno5_face(ql, eps);
          Qr[c] = weno5_face(qr, eps);
          Dn[c] = normal_slope(&q[1]) / hn;
        }
        collision(Ql, Qr, dir, s.RT, Q0);
        double *o = &NQ[fb.at(f, i1, i2) * 8];
        for (int c = 0; c < 4; ++c) {
          o[c] = Q0[c];
          o[4 + c] = Dn[c];
        }
      }

  /* 2d: tangential pass 1 along t1.  Per face and Gauss point g1: Q0[4], Dn[4], Dt1[4]. */
  std::vector<double> T1(fb.count() * 24);
#pragma omp parallel for collapse(2) schedule(static)
  for (int f = 0; f < fb.nf; ++f)
    for (int i1 = 0; i1 < fb.n1; ++i1)
      for (int i2 = -2; i2 < fb.n2 + 2; ++i2) {
        double *o = &T1[fb.at(f, i1, i2) * 24];
        for (int fld = 0; fld < 8; ++fld) {
          double q[5], v[2];
          for (int m = 0; m < 5; ++m) q[m] = NQ[fb.at(f, i1 - 2 + m, i2) * 8 + fld];
          tangential_gauss(q, eps, s.tangential_linear, v);
          o[0 * 12 + fld] = v[0];
          o[1 * 12 + fld] = v[1];
          if (fld < 4) { /* slope of Q0 along t1 */
            quartic_slope_gauss(q, v);
            o[0 * 12 + 8 + fld] = v[0] / A1.w(i1);
            o[1 * 12 + 8 + fld] = v[1] / A1.w(i1);
          }
        }
      }

  /* 2e-2g: tangential pass 2 along t2, Gauss-point fluxes, face average with weights 1/4 (S1). */
  const size_t nface_out = (size_t)(s.n[0] + (dir == 0)) * (s.n[1] + (dir == 1)) * (s.n[2] + (dir == 2));
  Ff.assign(4 * nface_out, 0.0);
  dFf.assign(4 * nface_out, 0.0);
  int fn[3] = {s.n[0] + (dir == 0), s.n[1] + (dir == 1), s.n[2] + (dir == 2)};
#pragma omp parallel for collapse(2) schedule(static)
  for (int f = 0; f < fb.nf; ++f)
    for (int i1 = 0; i1 < fb.n1; ++i1)
      for (int i2 = 0; i2 < fb.n2; ++i2) {
        double Fsum[4] = {0, 0, 0, 0}, dFsum[4] = {0, 0, 0, 0};
        for (int g1 = 0; g1 < 2; ++g1) {
          double val[12][2], Dt2[4][2];
          for (int fld = 0; fld < 12; ++fld) {
            double q[5];
            for (int m = 0; m < 5; ++m) q[m] = T1[fb.at(f, i1, i2 - 2 + m) * 24 + g1 * 12 + fld];
            tangential_gauss(q, eps, s.tangential_linear, val[fld]);
            if (fld < 4) {
              quartic_slope_gauss(q, Dt2[fld]);
              Dt2[fld][0] /= A2.w(i2);
              Dt2[fld][1] /= A2.w(i2);
            }
          }
          for (int g2 = 0; g2 < 2; ++g2) {
            double Q0[4], dQ[3][4], F[4], dF[4];
            for (int c = 0; c < 4; ++c) {
              Q0[c] = val[c][g2];
              dQ[fb.a][c] = val[4 + c][g2];
              dQ[fb.t1][c] = val[8 + c][g2];
              dQ[fb.t2][c] = Dt2[c][g2];
            }
            gauss_point_flux(Q0, dQ, dir, s.RT, s.nu, s.rho_ref, F, dF);
            for (int c = 0; c < 4; ++c) {
              Fsum[c] += 0.25 * F[c];
              dFsum[c] += 0.25 * dF[c];
            }
          }
        }
        int p[3];
        p[fb.a] = f;
        p[fb.t1] = i1;
        p[fb.t2] = i2;
        for (int c = 0; c < 4; ++c) {
          const size_t o = (((size_t)c * fn[2] + p[2]) * fn[1] + p[1]) * fn[0] + p[0];
          Ff[o] = Fsum[c];
          dFf[o] = dFsum[c];
        }
      }
}

/* Eq. 5: L = -(1/|Omega|) sum_p F_p = -sum_d (F_{d+} - F_{d-})/Delta_d for face-averaged fluxes;
 * dL likewise from dF/dt.  Interior layout [c][k][j][i]. */
void eval_L(const gkso_ctx &s, const std::vector<double> &Wp, std::vector<double> &L,
            std::vector<double> &dL) {
  L.assign(4 * s.ncell(), 0.0);
  dL.assign(4 * s.ncell(), 0.0);
  for (int dir = 0; dir < 3; ++dir) {
    std::vector<double> F, dF;
    face_flux(s, Wp, dir, F, dF);
    const int fn[3] = {s.n[0] + (dir == 0), s.n[1] + (dir == 1), s.n[2] + (dir == 2)};
    for (int c = 0; c < 4; ++c)
      for (int k = 0; k < s.n[2]; ++k)
        for (int j = 0; j < s.n[1]; ++j)
          for (int i = 0; i < s.n[0]; ++i) {
            const int p[3] = {i, j, k};
            int q[3] = {i, j, k};
            q[dir] += 1;
            const size_t lo = (((size_t)c * fn[2] + p[2]) * fn[1] + p[1]) * fn[0] + p[0];
            const size_t hi = (((size_t)c * fn[2] + q[2]) * fn[1] + q[1]) * fn[0] + q[0];
            const double w = s.ax[dir].w(p[dir]);
            L[s.ii(c, i, j, k)] -= (F[hi] - F[lo]) / w;
            dL[s.ii(c, i, j, k)] -= (dF[hi] - dF[lo]) / w;
          }
  }
}

/* ------------------------------------------------------------------------------------------
 * Forcing (step 6; Eq. 10-13; readings S12-S16, S22, S23).  Every increment is computed from the
 * un-forced field W and returned in dM[3][k][j][i]; the caller adds them.
 * ------------------------------------------------------------------------------------------ */
struct Support3 { int idx[3][3]; double phi[3][3]; }; /* [axis][m]: cell index (or -1) and delta weight */

int ibm_support(const gkso_ctx &s, const double X[3], Support3 &sp) {
  for (int a = 0; a < 3; ++a) {
    const Axis &A = s.ax[a];
    const int c0 = A.find_cell(X[a]);
    if (c0 < 0) return fail("ibm: point outside the domain");
    const double h = A.w(c0);
    for (int m = 0; m < 3; ++m) {
      const int i = c0 - 1 + m;
      if (std::fabs(A.w(i) - h) > 1e-9 * h) return fail("ibm: grid not locally uniform over the support");
      sp.phi[a][m] = delta3((A.xc(i) - X[a]) / h);
      if (i < 0 || i >= A.n) sp.idx[a][m] = A.periodic ? Axis::wrap(i, A.n) : -1; /* outside a non-periodic face: dropped */
      else sp.idx[a][m] = i;
    }
  }
  return 0;
}

void ibm_interpolate(const gkso_ctx &s, const std::vector<double> &Wp, std::vector<double> &Up) {
  Up.assign(3 * (size_t)s.n_ibm, 0.0);
  for (int p = 0; p < s.n_ibm; ++p) {
    Support3 sp;
    ibm_support(s, &s.ibm_pos[3 * p], sp);
    for (int mk = 0; mk < 3; ++mk)
      for (int mj = 0; mj < 3; ++mj)
        for (int mi = 0; mi < 3; ++mi) {
          const int i = sp.idx[0][mi], j = sp.idx[1][mj], k = sp.idx[2][mk];
          if (i < 0 || j < 0 || k < 0) continue;
          const double wgt = sp.phi[0][mi] * sp.phi[1][mj] * sp.phi[2][mk];
          const double rho = Wp[s.id(0, i, j, k)];
          for (int c = 0; c < 3; ++c) Up[3 * p + c] += wgt * Wp[s.id(1 + c, i, j, k)] / rho;
        }
  }
}

/* ------------------------------------------------------------------------------------------
 * Actuator-line front half: flow sampling, force calculation.
 * ------------------------------------------------------------------------------------------ */
/* trilinear interpolation of (rho, U, V, W) between the 8 cell centres around X ("The trilinear interpolation
 * method is used to interpolate the simulated velocity to each actuator point"); velocities, not
 * momenta, are interpolated.  Periodic axes wrap; beyond the outermost centres of a non-periodic axis the
 * outermost cell is used (zero gradient; ghost cells of the un-forced field are not defined) - reading S26. */
void sample_trilinear(const gkso_ctx &s, const std::vector<double> &Wp, const double X[3], double out[4]) {
  int i0[3], i1[3];
  double t[3];
  for (int a = 0; a < 3; ++a) {
    const Axis &A = s.ax[a];
    double x = X[a];
    if (A.periodic) x -= std::floor((x - A.lo()) / A.len()) * A.len();
    int c = A.find_cell(x);
    if (c < 0) c = x < A.lo() ? 0 : A.n - 1;
    const int lo = x < A.xc(c) ? c - 1 : c; /* xc(lo) <= x < xc(lo+1), centres of ghost cells included */
    t[a] = (x - A.xc(lo)) / (A.xc(lo + 1) - A.xc(lo));
    i0[a] = lo;
    i1[a] = lo + 1;
    if (A.periodic) {
      i0[a] = (i0[a] + A.n) % A.n;
      i1[a] = i1[a] % A.n;
    } else {
      i0[a] = std::min(std::max(i0[a], 0), A.n - 1);
      i1[a] = std::min(std::max(i1[a], 0), A.n - 1);
    }
  }
  for (int c = 0; c < 4; ++c) out[c] = 0.0;
  for (int dk = 0; dk < 2; ++dk)
    for (int dj = 0; dj < 2; ++dj)
      for (int di = 0; di < 2; ++di) {
        const int i = di ? i1[0] : i0[0], j = dj ? i1[1] : i0[1], k = dk ? i1[2] : i0[2];
        const double wgt = (di ? t[0] : 1.0 - t[0]) * (dj ? t[1] : 1.0 - t[1]) * (dk ? t[2] : 1.0 - t[2]);
        const double rho = Wp[s.id(0, i, j, k)];
        out[0] += wgt * rho;
        for (int c = 1; c < 4; ++c) out[c] += wgt * Wp[s.id(c, i, j, k)] / rho;
      }
}

/* tabulated 2-D airfoil data of one section (table `sec`), linear in alpha, end values beyond the table */
void polar_lookup_section(const gkso_ctx::Rotor &r, int sec, double alpha, double &cl, double &cd) {
  const int n = (int)r.pa.size();
  const double *pcl = r.pcl.data() + (size_t)sec * n, *pcd = r.pcd.data() + (size_t)sec * n;
  if (alpha <= r.pa[0]) { cl = pcl[0]; cd = pcd[0]; return; }
  if (alpha >= r.pa[n - 1]) { cl = pcl[n - 1]; cd = pcd[n - 1]; return; }
  int m = 0;
  while (r.pa[m + 1] < alpha) ++m;
  const double t = (alpha - r.pa[m]) / (r.pa[m + 1] - r.pa[m]);
  cl = pcl[m] + t * (pcl[m + 1] - pcl[m]);
  cd = pcd[m] + t * (pcd[m + 1] - pcd[m]);
}

/* C_L, C_D of the station at radius rad: linear in the radius between the two nearby airfoil sections
 * (reading S28), the first / last section's inside / outside of them */
void polar_lookup(const gkso_ctx::Rotor &r, double rad, double alpha, double &cl, double &cd) {
  const int ns = (int)r.sec_r.size();
  if (ns <= 1 || rad <= r.sec_r[0]) { polar_lookup_section(r, 0, alpha, cl, cd); return; }
  if (rad >= r.sec_r[ns - 1]) { polar_lookup_section(r, ns - 1, alpha, cl, cd); return; }
  int m = 0;
  while (r.sec_r[m + 1] < rad) ++m;
  const double t = (rad - r.sec_r[m]) / (r.sec_r[m + 1] - r.sec_r[m]);
  double cl0, cd0, cl1, cd1;
  polar_lookup_section(r, m, alpha, cl0, cd0);
  polar_lookup_section(r, m + 1, alpha, cl1, cd1);
  cl = cl0 + t * (cl1 - cl0);
  cd = cd0 + t * (cd1 - cd0);
}

/* Eq. 14: f_tip = 2/pi acos(exp(-g1 N (R - r)/(2 r sin phi))), g1 = exp(-c1 (N lambda - c2)) + 0.1 */
double tip_factor(int N, double R, double r, double sinphi, double tsr, double c1, double c2) {
  if (!(sinphi > 0.0)) return 1.0; /* reading S27: no correction for a reversed flow angle */
  const double g1 = std::exp(-c1 * (N * tsr - c2)) + 0.1;
  return 2.0 / PI * std::acos(std::exp(-g1 * N * (R - r) / (2.0 * r * sinphi)));
}

/* positions of the actuator points at the rotor's clock and the point forces ON THE FLUID.
 * Rotor axis +x; blade b at azimuth psi = theta0 + omega t + 2 pi b/N; radial unit (0, cos psi, sin psi),
 * rotational unit e_theta = (0, -sin psi, cos psi); station k at r = r_hub + (k + 1/2) w, w = (R - r_hub)/npts, unless
 * the caller gave radii and widths (S28). */
void rotor_forces(const gkso_ctx &s, const std::vector<double> &Wp, std::vector<double> &pos,
                  std::vector<double> &force) {
  const gkso_ctx::Rotor &R = s.rotor;
  pos.assign(3 * (size_t)R.nb * R.np, 0.0);
  force.assign(3 * (size_t)R.nb * R.np, 0.0);
  for (int b = 0; b < R.nb; ++b) {
    const double psi = R.theta0 + R.omega * R.time + 2.0 * PI * b / R.nb;
    const double er[3] = {0.0, std::cos(psi), std::sin(psi)}, et[3] = {0.0, -std::sin(psi), std::cos(psi)};
    for (int k = 0; k < R.np; ++k) {
      const size_t p = (size_t)b * R.np + k;
      const double r = R.radius[k], w = R.width[k], c = R.chord[k];   /* station radius, element width (S28) */
      double X[3], q[4];
      for (int a = 0; a < 3; ++a) X[a] = R.hub[a] + r * er[a];
      sample_trilinear(s, Wp, X, q);                         /* flow sampling */
      double Ux = q[1], Ut = q[2] * et[1] + q[3] * et[2];   /* U^2D = (U_x, U_theta) */
      double phi = std::atan2(Ux, R.omega * r - Ut);         /* flow angle between U_rel and the rotor plane */
      double cl, cd;
      polar_lookup(R, r, phi - R.twist[k], cl, cd);          /* alpha = phi - gamma */
      if (R.fs_corr) { /* U_inf^2D = U^2D / (1 - C_D c /(4 sqrt(pi) eps)), then U_rel again */
        const double f = 1.0 / (1.0 - cd * c / (4.0 * std::sqrt(PI) * s.alm_eps));
        Ux *= f;
        Ut *= f;
        phi = std::atan2(Ux, R.omega * r - Ut);
        polar_lookup(R, r, phi - R.twist[k], cl, cd);
      }
      const double urel2 = Ux * Ux + (Ut - R.omega * r) * (Ut - R.omega * r);
      const double L = 0.5 * q[0] * c * w * cl * urel2, D = 0.5 * q[0] * c * w * cd * urel2; /* Eq. 9 */
      double Fx = L * std::cos(phi) + D * std::sin(phi), Ft = L * std::sin(phi) - D * std::cos(phi);
      if (R.tip_corr) {
        const double tsr = R.omega * R.R / R.uref;
        Fx *= tip_factor(R.nb, R.R, r, std::sin(phi), tsr, 0.1219, 21.52);
        Ft *= tip_factor(R.nb, R.R, r, std::sin(phi), tsr, 0.0984, 13.026);
      }
      for (int a = 0; a < 3; ++a) {
        pos[3 * p + a] = X[a];
        force[3 * p + a] = -(a == 0 ? Fx : Ft * et[a]);       /* reaction on the fluid */
      }
    }
  }
}

void eval_forcing(const gkso_ctx &s, const std::vector<double> &Wp, double dt, std::vector<double> &dM) {
  const size_t N = s.ncell();
  dM.assign(3 * N, 0.0);
  auto at = [&](int c, int i, int j, int k) -> double & { return dM[s.ii(c, i, j, k)]; }; /* c = 0..2 */

  /* uniform acceleration: dt * rho * g */
  for (int c = 0; c < 3; ++c)
    if (s.g[c] != 0.0)
      for (int k = 0; k < s.n[2]; ++k)
        for (int j = 0; j < s.n[1]; ++j)
          for (int i = 0; i < s.n[0]; ++i) at(c, i, j, k) += dt * Wp[s.id(0, i, j, k)] * s.g[c];

  /* S16: constant-mass-flux correction, sum in fixed k,j,i order */
  if (s.bulk_axis >= 0) {
    double sm = 0.0, sv = 0.0;
    for (int k = 0; k < s.n[2]; ++k)
      for (int j = 0; j < s.n[1]; ++j)
        for (int i = 0; i < s.n[0]; ++i) {
          const double vol = s.ax[0].w(i) * s.ax[1].w(j) * s.ax[2].w(k);
          sm += Wp[s.id(1 + s.bulk_axis, i, j, k)] * vol;
          sv += vol;
        }
    const double delta = s.bulk_target - sm / sv;
    for (int k = 0; k < s.n[2]; ++k)
      for (int j = 0; j < s.n[1]; ++j)
        for (int i = 0; i < s.n[0]; ++i) at(s.bulk_axis, i, j, k) += delta;
  }

  /* IBM (S13-S15, S25): pass s interpolates U_p^s from the un-forced field plus the increments of the passes
     before it (Eq. 11), spreads rho_ijk (v_p - U_p^s) phi phi phi V_p/|Omega_ijk|, and the increments add up
     (Eq. 12).  From the second pass on the iteration stops once max_p |v_p - U_p^s| < tol. */
  if (s.n_ibm > 0) {
    std::vector<double> Wit(Wp), Up;
    for (int pass = 0; pass < s.ibm_maxit; ++pass) {
      ibm_interpolate(s, Wit, Up);
      if (pass > 0) {
        double res = 0.0;
        for (int p = 0; p < s.n_ibm; ++p) {
          double r2 = 0.0;
          for (int c = 0; c < 3; ++c) r2 += (s.ibm_vel[3 * p + c] - Up[3 * p + c]) * (s.ibm_vel[3 * p + c] - Up[3 * p + c]);
          res = std::max(res, std::sqrt(r2));
        }
        if (res < s.ibm_tol) break;
      }
      for (int p = 0; p < s.n_ibm; ++p) {
        Support3 sp;
        ibm_support(s, &s.ibm_pos[3 * p], sp);
        for (int mk = 0; mk < 3; ++mk)
          for (int mj = 0; mj < 3; ++mj)
            for (int mi = 0; mi < 3; ++mi) {
              const int i = sp.idx[0][mi], j = sp.idx[1][mj], k = sp.idx[2][mk];
              if (i < 0 || j < 0 || k < 0) continue;
              const double wgt = sp.phi[0][mi] * sp.phi[1][mj] * sp.phi[2][mk];
              const double vol = s.ax[0].w(i) * s.ax[1].w(j) * s.ax[2].w(k);
              const double rho = Wp[s.id(0, i, j, k)];
              for (int c = 0; c < 3; ++c) {
                const double inc = rho * (s.ibm_vel[3 * p + c] - Up[3 * p + c]) * wgt * s.ibm_vol[p] / vol;
                at(c, i, j, k) += inc;
                Wit[s.id(1 + c, i, j, k)] += inc;
              }
            }
      }
    }
  }

  /* ALM (Eq. 10, S22-S23): dt * F exp(-r^2/eps^2)/(eps^3 pi^1.5) at cell centres with r <= cut*eps */
  for (int p = 0; p < s.n_alm; ++p) {
    const double *X = &s.alm_pos[3 * p], *Fp = &s.alm_force[3 * p];
    const double e = s.alm_eps;
    const double R = s.alm_cut > 0 ? s.alm_cut * e : 1e300;
    int lo[3], hi[3];
    for (int a = 0; a < 3; ++a) { /* unwrapped index range whose centres lie within R of X[a] */
      const Axis &A = s.ax[a];
      int c0, imin, imax;
      if (A.periodic) { /* bring X into the domain to find its cell, then shift the index back */
        const double L = A.len();
        const double m = std::floor((X[a] - A.lo()) / L);
        c0 = A.find_cell(X[a] - m * L);
        if (c0 < 0) c0 = 0;
        c0 += (int)m * A.n;
        imin = c0 - A.n + 1;
        imax = c0 + A.n - 1;
      } else { /* cells outside a non-periodic face receive nothing */
        c0 = A.find_cell(X[a]);
        if (c0 < 0) c0 = X[a] < A.lo() ? 0 : A.n - 1;
        imin = 0;
        imax = A.n - 1;
      }
      lo[a] = hi[a] = c0;
      while (lo[a] - 1 >= imin && X[a] - A.xc_ext(lo[a] - 1) <= R) --lo[a];
      while (hi[a] + 1 <= imax && A.xc_ext(hi[a] + 1) - X[a] <= R) ++hi[a];
    }
    for (int k = lo[2]; k <= hi[2]; ++k)
      for (int j = lo[1]; j <= hi[1]; ++j)
        for (int i = lo[0]; i <= hi[0]; ++i) {
          const double rx = s.ax[0].xc_ext(i) - X[0];
          const double ry = s.ax[1].xc_ext(j) - X[1];
          const double rz = s.ax[2].xc_ext(k) - X[2];
          const double r2 = rx * rx + ry * ry + rz * rz;
          if (r2 > R * R) continue;
          const double kern = std::exp(-r2 / (e * e)) / (e * e * e * std::pow(PI, 1.5));
          const int iw = Axis::wrap(i, s.n[0]), jw = Axis::wrap(j, s.n[1]), kw = Axis::wrap(k, s.n[2]);
          for (int c = 0; c < 3; ++c) at(c, iw, jw, kw) += dt * Fp[c] * kern;
        }
  }
}

/* S20: the convective-outflow ghost state of axis a, on every line pass a covers (the ghosts of the tangential
 * axes that pass a reads must be current: call after the passes of the lower axes).
 * dt < 0: start from the last interior value; dt >= 0: phi_g -= C (phi_g - phi_{g-1}), g = 1,2,3 in order */
void outflow_state_of_axis(const gkso_ctx &s, std::vector<double> &W, int a, double dt) {
  for (int side = 0; side < 2; ++side) {
    if (s.bc[2 * a + side] != BC_OUTFLOW) continue;
    const double Uc = std::fabs(s.inflow[1 + a]);
    for_lines_of_pass(s, a, [&](int p[3]) {
      for (int c = 0; c < 4; ++c)
        for (int g = 1; g <= NG; ++g) {
          int pg[3] = {p[0], p[1], p[2]}, pm[3] = {p[0], p[1], p[2]};
          pg[a] = side == 0 ? -g : s.n[a] - 1 + g;
          if (dt < 0) {
            pm[a] = side == 0 ? 0 : s.n[a] - 1;
            W[s.idp(c, pg)] = W[s.idp(c, pm)];
          } else {
            pm[a] = side == 0 ? -g + 1 : s.n[a] - 2 + g; /* g-1: one cell closer to the interior */
            const double C = Uc * dt / std::fabs(s.ax[a].xc(pg[a]) - s.ax[a].xc(pm[a]));
            double &phi = W[s.idp(c, pg)];
            phi = phi - C * (phi - W[s.idp(c, pm)]);
          }
        }
    });
  }
}

/* initialise (dt < 0) or advance the outflow ghost state of every axis; the passes of the lower axes run in
 * between so that the lines through their ghosts see current values */
void outflow_state(const gkso_ctx &s, std::vector<double> &W, double dt) {
  bool any = false;
  for (int f = 0; f < 6; ++f) any = any || s.bc[f] == BC_OUTFLOW;
  if (!any) return;
  for (int a = 0; a < 3; ++a) {
    outflow_state_of_axis(s, W, a, dt);
    fill_pass(s, W, a);
  }
}

int validate(const gkso_config &c) {
  if (c.nx < 6 || c.ny < 6 || c.nz < 6) return fail("nx, ny, nz must be >= 6");
  if (!(c.RT > 0)) return fail("RT must be > 0");
  if (!(c.nu >= 0)) return fail("nu must be >= 0");
  if (!(c.rho_ref > 0)) return fail("rho_ref must be > 0");
  for (int a = 0; a < 3; ++a) {
    const int lo = c.bc[2 * a], hi = c.bc[2 * a + 1];
    if (lo < 0 || lo > 5 || hi < 0 || hi > 5) return fail("unknown boundary kind");
    if ((lo == BC_PERIODIC) != (hi == BC_PERIODIC)) return fail("periodic faces must be paired");
    const double *f = a == 0 ? c.xf : a == 1 ? c.yf : c.zf;
    const int n = a == 0 ? c.nx : a == 1 ? c.ny : c.nz;
    const double d = a == 0 ? c.dx : a == 1 ? c.dy : c.dz;
    if (f) {
      for (int i = 0; i < n; ++i)
        if (!(f[i + 1] > f[i])) return fail("face coordinates must be strictly increasing");
    } else if (!(d > 0))
      return fail("spacing must be > 0");
  }
  return 0;
}

} /* namespace */

/* ============================== C interface ============================== */
extern "C" {

const char *gkso_last_error(void) { return g_error.c_str(); }

int gkso_create(const gkso_config *cfg, gkso_ctx **out) {
  if (!cfg || !out) return fail("null argument");
  if (validate(*cfg)) return 1;
  gkso_ctx *s = new gkso_ctx;
  s->n[0] = cfg->nx;
  s->n[1] = cfg->ny;
  s->n[2] = cfg->nz;
  for (int i = 0; i < 6; ++i) s->bc[i] = cfg->bc[i];
  for (int i = 0; i < 4; ++i) s->inflow[i] = cfg->inflow[i];
  s->ax[0].build(cfg->nx, cfg->xf, cfg->x0, cfg->dx, cfg->bc[0] == BC_PERIODIC);
  s->ax[1].build(cfg->ny, cfg->yf, cfg->y0, cfg->dy, cfg->bc[2] == BC_PERIODIC);
  s->ax[2].build(cfg->nz, cfg->zf, cfg->z0, cfg->dz, cfg->bc[4] == BC_PERIODIC);
  s->RT = cfg->RT;
  s->nu = cfg->nu;
  s->rho_ref = cfg->rho_ref;
  s->eps = cfg->weno_eps > 0 ? cfg->weno_eps : 1e-6;
  s->W.assign(4 * s->ncell_p(), 0.0);
  *out = s;
  return 0;
}

void gkso_destroy(gkso_ctx *s) { delete s; }

int gkso_set_state(gkso_ctx *s, const double *Win) {
  if (!s || !Win) return fail("null argument");
  for (int c = 0; c < 4; ++c)
    for (int k = 0; k < s->n[2]; ++k)
      for (int j = 0; j < s->n[1]; ++j)
        for (int i = 0; i < s->n[0]; ++i) s->W[s->id(c, i, j, k)] = Win[s->ii(c, i, j, k)];
  /* S20: convective-outflow ghosts start from the last interior value */
  outflow_state(*s, s->W, -1.0);
  s->have_state = true;
  return 0;
}

int gkso_get_state(gkso_ctx *s, double *Wout) {
  if (!s || !Wout) return fail("null argument");
  if (!s->have_state) return fail("no state set");
  for (int c = 0; c < 4; ++c)
    for (int k = 0; k < s->n[2]; ++k)
      for (int j = 0; j < s->n[1]; ++j)
        for (int i = 0; i < s->n[0]; ++i) Wout[s->ii(c, i, j, k)] = s->W[s->id(c, i, j, k)];
  return 0;
}

/* One step W^n -> W~^{n+1} (steps 1-7). */
int gkso_step(gkso_ctx *s, double dt) {
  if (!s) return fail("null argument");
  if (!s->have_state) return fail("gkso_step before gkso_set_state");
  if (!(dt > 0)) return fail("dt must be > 0");
  const size_t N = s->ncell();
  /* 1-3: ghost fill of W^n, L and dL, first stage W* = W^n + dt/2 L + dt^2/8 dL */
  std::vector<double> &Wn = s->W;
  fill_ghosts(*s, Wn);
  std::vector<double> L, dL;
  eval_L(*s, Wn, L, dL);
  std::vector<double> Ws = Wn; /* outflow ghost state is held fixed during both stages (S20) */
  for (int c = 0; c < 4; ++c)
    for (int k = 0; k < s->n[2]; ++k)
      for (int j = 0; j < s->n[1]; ++j)
        for (int i = 0; i < s->n[0]; ++i) {
          const size_t o = s->ii(c, i, j, k);
          Ws[s->id(c, i, j, k)] = Wn[s->id(c, i, j, k)] + 0.5 * dt * L[o] + dt * dt / 8.0 * dL[o];
        }
  /* 4: ghost fill of W*, dL* */
  fill_ghosts(*s, Ws);
  std::vector<double> L2, dL2;
  eval_L(*s, Ws, L2, dL2);
  /* 5: W^{n+1} = W^n + dt L + dt^2/6 (dL + 2 dL*) */
  std::vector<double> Wnew = Wn;
  for (int c = 0; c < 4; ++c)
    for (int k = 0; k < s->n[2]; ++k)
      for (int j = 0; j < s->n[1]; ++j)
        for (int i = 0; i < s->n[0]; ++i) {
          const size_t o = s->ii(c, i, j, k);
          Wnew[s->id(c, i, j, k)] =
              Wn[s->id(c, i, j, k)] + dt * L[o] + dt * dt / 6.0 * (dL[o] + 2.0 * dL2[o]);
        }
  /* 6: forcing increments from the un-forced W^{n+1}, then added (Eq. 13; density gets none) */
  if (s->rotor.on) { /* ALM front half on the un-forced field at the rotor's clock t^n (S12, S26) */
    rotor_forces(*s, Wnew, s->alm_pos, s->alm_force);
    s->n_alm = s->rotor.nb * s->rotor.np;
    s->rotor.time += dt;
  }
  std::vector<double> dM;
  eval_forcing(*s, Wnew, dt, dM);
  for (int c = 0; c < 3; ++c)
    for (int k = 0; k < s->n[2]; ++k)
      for (int j = 0; j < s->n[1]; ++j)
        for (int i = 0; i < s->n[0]; ++i) Wnew[s->id(1 + c, i, j, k)] += dM[s->ii(c, i, j, k)];
  /* 7: convective-outflow ghosts */
  outflow_state(*s, Wnew, dt);
  (void)N;
  s->W.swap(Wnew);
  return 0;
}

int gkso_set_body_force(gkso_ctx *s, double gx, double gy, double gz) {
  if (!s) return fail("null argument");
  s->g[0] = gx; s->g[1] = gy; s->g[2] = gz;
  return 0;
}

int gkso_set_bulk_flux(gkso_ctx *s, int axis, double target) {
  if (!s) return fail("null argument");
  if (axis > 2) return fail("axis must be 0, 1, 2 or negative");
  s->bulk_axis = axis < 0 ? -1 : axis;
  s->bulk_target = target;
  return 0;
}

int gkso_alm_set_points(gkso_ctx *s, int n, const double *pos, const double *force, double eps) {
  if (!s || n < 0) return fail("bad argument");
  if (n > 0 && (!pos || !force)) return fail("null argument");
  if (n > 0 && !(eps > 0)) return fail("eps must be > 0");
  if (n > 0)
    for (int a = 0; a < 3; ++a) {
      const Axis &A = s->ax[a];
      if (A.periodic && 2.0 * s->alm_cut * eps > A.len()) return fail("alm: support wider than a periodic axis");
    }
  s->n_alm = n;
  s->alm_eps = eps;
  s->alm_pos.assign(pos, pos + 3 * (size_t)n);
  s->alm_force.assign(force, force + 3 * (size_t)n);
  return 0;
}

int gkso_alm_set_cut(gkso_ctx *s, double cut) {
  if (!s) return fail("null argument");
  s->alm_cut = cut;
  return 0;
}

int gkso_ibm_set_points(gkso_ctx *s, int n, const double *pos, const double *weights) {
  if (!s || n < 0) return fail("bad argument");
  if (n > 0 && (!pos || !weights)) return fail("null argument");
  for (int p = 0; p < n; ++p) {
    Support3 sp;
    if (ibm_support(*s, &pos[3 * p], sp)) return 1;
  }
  s->n_ibm = n;
  s->ibm_pos.assign(pos, pos + 3 * (size_t)n);
  s->ibm_vol.assign(weights, weights + (size_t)n);
  s->ibm_vel.assign(3 * (size_t)n, 0.0);
  return 0;
}

int gkso_set_reconstruction(gkso_ctx *s, int tangential_linear) {
  if (!s) return fail("null argument");
  if (tangential_linear != 0 && tangential_linear != 1) return fail("tangential_linear must be 0 or 1");
  s->tangential_linear = tangential_linear != 0;
  return 0;
}

int gkso_ibm_set_iterations(gkso_ctx *s, int max_iter, double tol) {
  if (!s) return fail("null argument");
  if (max_iter < 1 || !(tol >= 0.0)) return fail("ibm: max_iter must be >= 1 and tol >= 0");
  s->ibm_maxit = max_iter;
  s->ibm_tol = tol;
  return 0;
}

int gkso_ibm_set_velocities(gkso_ctx *s, const double *vel) {
  if (!s) return fail("null argument");
  if (vel) s->ibm_vel.assign(vel, vel + 3 * (size_t)s->n_ibm);
  else s->ibm_vel.assign(3 * (size_t)s->n_ibm, 0.0);
  return 0;
}

int gkso_eval_flux(gkso_ctx *s, int dir, double *F, double *dFdt) {
  if (!s || !F || !dFdt || dir < 0 || dir > 2) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  std::vector<double> Wp = s->W, Ff, dFf;
  fill_ghosts(*s, Wp);
  face_flux(*s, Wp, dir, Ff, dFf);
  std::memcpy(F, Ff.data(), Ff.size() * sizeof(double));
  std::memcpy(dFdt, dFf.data(), dFf.size() * sizeof(double));
  return 0;
}

int gkso_eval_L(gkso_ctx *s, double *L, double *dL) {
  if (!s || !L || !dL) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  std::vector<double> Wp = s->W, l, dl;
  fill_ghosts(*s, Wp);
  eval_L(*s, Wp, l, dl);
  std::memcpy(L, l.data(), l.size() * sizeof(double));
  std::memcpy(dL, dl.data(), dl.size() * sizeof(double));
  return 0;
}

int gkso_get_padded(gkso_ctx *s, double *Wp) {
  if (!s || !Wp) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  std::vector<double> W = s->W;
  fill_ghosts(*s, W);
  std::memcpy(Wp, W.data(), W.size() * sizeof(double));
  return 0;
}

int gkso_alm_set_rotor(gkso_ctx *s, const gkso_rotor *r) {
  if (!s) return fail("null argument");
  if (!r) { /* NULL clears the rotor and its points */
    s->rotor = gkso_ctx::Rotor();
    s->n_alm = 0;
    return 0;
  }
  if (r->nblades < 1 || r->npts < 1 || !r->chord || !r->twist || r->npolar < 2 || !r->alpha || !r->cl || !r->cd)
    return fail("rotor: bad sizes or null tables");
  if (!(r->R > r->r_hub) || !(r->r_hub >= 0) || !(r->eps > 0)) return fail("rotor: need R > r_hub >= 0 and eps > 0");
  if (r->tip_correction && !(r->u_ref > 0)) return fail("rotor: the tip correction needs u_ref > 0 (tip speed ratio)");
  for (int m = 1; m < r->npolar; ++m)
    if (!(r->alpha[m] > r->alpha[m - 1])) return fail("rotor: polar angles must increase");
  if ((r->radius == nullptr) != (r->width == nullptr)) return fail("rotor: radius and width come together");
  if (r->radius)
    for (int k = 0; k < r->npts; ++k)
      if (!(r->radius[k] > 0) || !(r->radius[k] <= r->R) || !(r->width[k] > 0)) return fail("rotor: need 0 < radius <= R and width > 0");
  if (r->nsections > 1) {
    if (!r->section_r) return fail("rotor: section radii missing");
    for (int m = 1; m < r->nsections; ++m)
      if (!(r->section_r[m] > r->section_r[m - 1])) return fail("rotor: section radii must increase");
  }
  for (int a = 0; a < 3; ++a) {
    const Axis &A = s->ax[a];
    if (A.periodic && 2.0 * s->alm_cut * r->eps > A.len()) return fail("alm: support wider than a periodic axis");
  }
  gkso_ctx::Rotor &R = s->rotor;
  R.on = true;
  R.nb = r->nblades; R.np = r->npts;
  for (int a = 0; a < 3; ++a) R.hub[a] = r->hub[a];
  R.R = r->R; R.rhub = r->r_hub; R.omega = r->omega; R.theta0 = r->theta0; R.uref = r->u_ref; R.time = 0.0;
  R.fs_corr = r->freestream_correction; R.tip_corr = r->tip_correction;
  R.chord.assign(r->chord, r->chord + r->npts);
  R.twist.assign(r->twist, r->twist + r->npts);
  const int ns = r->nsections > 1 ? r->nsections : 1;
  R.pa.assign(r->alpha, r->alpha + r->npolar);
  R.pcl.assign(r->cl, r->cl + (size_t)ns * r->npolar);
  R.pcd.assign(r->cd, r->cd + (size_t)ns * r->npolar);
  R.sec_r.clear();
  if (ns > 1) R.sec_r.assign(r->section_r, r->section_r + ns);
  R.radius.resize(r->npts);
  R.width.resize(r->npts);
  for (int k = 0; k < r->npts; ++k) {
    const double w = (r->R - r->r_hub) / r->npts;
    R.radius[k] = r->radius ? r->radius[k] : r->r_hub + (k + 0.5) * w;
    R.width[k] = r->width ? r->width[k] : w;
  }
  s->alm_eps = r->eps;
  s->n_alm = 0;
  return 0;
}

/* test hook: positions and forces on the fluid of the actuator points for the CURRENT state and rotor clock */
int gkso_alm_rotor_eval(gkso_ctx *s, double *pos, double *force) {
  if (!s || !pos || !force) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  if (!s->rotor.on) return fail("no rotor set");
  std::vector<double> p, f;
  rotor_forces(*s, s->W, p, f);
  std::memcpy(pos, p.data(), p.size() * sizeof(double));
  std::memcpy(force, f.data(), f.size() * sizeof(double));
  return 0;
}

int gkso_eval_forcing(gkso_ctx *s, double dt, double *dM) {
  if (!s || !dM) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  if (s->rotor.on) {
    rotor_forces(*s, s->W, s->alm_pos, s->alm_force);
    s->n_alm = s->rotor.nb * s->rotor.np;
  }
  std::vector<double> d;
  eval_forcing(*s, s->W, dt, d);
  std::memcpy(dM, d.data(), d.size() * sizeof(double));
  return 0;
}

/* Time step of the CFL condition: dt = CFL min{dx, dy, dz} / (|U|_max + C), C = sqrt(1/(2 lambda))
 * = sqrt(RT); |U|_max over the interior cells of the current state, the minimum over every cell width. */
int gkso_cfl_dt(gkso_ctx *s, double cfl, double *dt) {
  if (!s || !dt) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  if (!(cfl > 0.0)) return fail("cfl must be > 0");
  double umax = 0.0, dmin = 1e300;
  for (int k = 0; k < s->n[2]; ++k)
    for (int j = 0; j < s->n[1]; ++j)
      for (int i = 0; i < s->n[0]; ++i) {
        const double rho = s->W[s->id(0, i, j, k)];
        const double mx = s->W[s->id(1, i, j, k)], my = s->W[s->id(2, i, j, k)], mz = s->W[s->id(3, i, j, k)];
        umax = std::max(umax, std::sqrt(mx * mx + my * my + mz * mz) / rho);
      }
  for (int a = 0; a < 3; ++a)
    for (int i = 0; i < s->n[a]; ++i) dmin = std::min(dmin, s->ax[a].w(i));
  *dt = cfl * dmin / (umax + std::sqrt(s->RT));
  return 0;
}

int gkso_ibm_interpolate(gkso_ctx *s, double *Up) {
  if (!s || !Up) return fail("bad argument");
  if (!s->have_state) return fail("no state set");
  std::vector<double> u;
  ibm_interpolate(*s, s->W, u);
  std::memcpy(Up, u.data(), u.size() * sizeof(double));
  return 0;
}

void gkso_moments(double U, double lambda, int nmax, double *out) { moments(U, lambda, nmax, out); }
void gkso_micro_solve(double U, double V, double W, double lambda, const double d[4], double a[4]) {
  micro_solve(U, V, W, lambda, d, a);
}
double gkso_weno5_face(const double q[5], double eps) { return weno5_face(q, eps); }
void gkso_weno5_gauss(const double q[5], double eps, double out[2]) { weno5_gauss(q, eps, out); }
void gkso_linear5_gauss(const double q[5], double out[2]) { tangential_gauss(q, 0.0, true, out); }
void gkso_quartic_slope_gauss(const double q[5], double out[2]) { quartic_slope_gauss(q, out); }
double gkso_normal_slope(const double q[4]) { return normal_slope(q); }
void gkso_collision(const double Ql[4], const double Qr[4], int dir, double RT, double Q0[4]) {
  collision(Ql, Qr, dir, RT, Q0);
}
void gkso_gauss_point_flux(const double Q0[4], const double dQ[12], int dir, double RT, double nu,
                           double rho_ref, double F[4], double dF[4]) {
  double d[3][4];
  for (int s = 0; s < 3; ++s)
    for (int c = 0; c < 4; ++c) d[s][c] = dQ[4 * s + c];
  gauss_point_flux(Q0, d, dir, RT, nu, rho_ref, F, dF);
}
double gkso_delta3(double r) { return delta3(r); }
double gkso_alm_kernel(double r, double eps) { return alm_kernel(r, eps); }

} /* extern "C" */
