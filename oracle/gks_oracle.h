/*
 * gks_oracle.h — C interface of the CPU ORACLE (libgks_oracle.so).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code with the CUDA path
 * (paper_2603_11102_b200/csrc, include/gks.h): this header, the oracle's structs and every
 * constant in gks_oracle.cpp are its own.
 *
 * The oracle is the algorithm of arxiv/paper_2603_11102 written out step by step, slowly, in fp64:
 * PAPER.md §2 (:41-93), Appendix (:501-558), §3.1 Eq. 10 (:135-139, :293), §3.2 (:141-175),
 * §3.3 (:177-191), the ALM front half (:101-127, Eq. 14 :388-399), the CFL condition (:91), with the readings
 * S1..S27 of DESIGN.md where the paper is silent.
 *
 * All pointers are HOST pointers.  Layouts: W[c][k][j][i] interior cells only, c in
 * {rho, rhoU, rhoV, rhoW}.  Return value 0 = ok, non-zero = error (gkso_last_error()).
 */
#ifndef GKS_ORACLE_H
#define GKS_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct gkso_ctx gkso_ctx;

/* boundary kinds: 0 periodic, 1 no-slip wall, 2 slip wall / symmetry, 3 inflow,
 * 4 convective outflow, 5 extrapolate (zero gradient) */
typedef struct {
  int nx, ny, nz;
  const double *xf, *yf, *zf; /* n+1 face coordinates or NULL (uniform: x0 + i*dx) */
  double x0, y0, z0, dx, dy, dz;
  double RT, nu, rho_ref;
  int bc[6];
  double inflow[4];
  double weno_eps; /* 0 => 1e-6 */
} gkso_config;

int gkso_create(const gkso_config *cfg, gkso_ctx **out);
void gkso_destroy(gkso_ctx *ctx);
int gkso_set_state(gkso_ctx *ctx, const double *W);
int gkso_get_state(gkso_ctx *ctx, double *W);
int gkso_step(gkso_ctx *ctx, double dt);
int gkso_set_body_force(gkso_ctx *ctx, double gx, double gy, double gz);
int gkso_set_bulk_flux(gkso_ctx *ctx, int axis, double target);
int gkso_alm_set_points(gkso_ctx *ctx, int n, const double *pos, const double *force, double eps);
int gkso_alm_set_cut(gkso_ctx *ctx, double cut_in_eps); /* test flag: radius of the cut in units of eps (default 3; <=0 => no cut) */
int gkso_ibm_set_points(gkso_ctx *ctx, int n, const double *pos, const double *weights);
int gkso_ibm_set_velocities(gkso_ctx *ctx, const double *vel);
/* scheme variant (the alternative of reading S7): 1 = the two tangential passes combine the
 * sub-stencil candidates with the linear weights (quartic interpolation); 0 = WENO5-JS everywhere (default) */
int gkso_set_reconstruction(gkso_ctx *ctx, int tangential_linear);
/* multi-direct-forcing passes per step (Eq. 11-12; S25); default 1, tol 0 */
int gkso_ibm_set_iterations(gkso_ctx *ctx, int max_iter, double tol);
/* face-averaged F and dF/dt of the current state, direction dir; F[c][k][j][i] with n_dir+1 faces along dir */
int gkso_eval_flux(gkso_ctx *ctx, int dir, double *F, double *dFdt);
/* L and dL/dt (Eq. 5) of the current state, interior cells, [c][k][j][i] */
int gkso_eval_L(gkso_ctx *ctx, double *L, double *dL);
/* padded copy (3 ghost layers per side, after ghost fill) of the current state: 4*(nz+6)*(ny+6)*(nx+6) */
int gkso_get_padded(gkso_ctx *ctx, double *Wp);
/* momentum increments of the forcing terms for the current state and dt: dM[3][k][j][i] */
int gkso_eval_forcing(gkso_ctx *ctx, double dt, double *dM);
/* interpolated fluid velocity at the IBM points (n*3) for the current state */
int gkso_ibm_interpolate(gkso_ctx *ctx, double *Up);
/* On-line actuator-line rotor (Eq. 9, Eq. 14; S26-S27): axis +x, blade b at azimuth
 * theta0 + omega t + 2 pi b / nblades, station k at r_hub + (k + 1/2)(R - r_hub)/npts.  Every step samples the
 * un-forced field at the points (trilinear), evaluates lift and drag from the tabulated polar and spreads the
 * reaction with Eq. 10.  NULL clears.  The rotor clock starts at 0 and advances by dt per step. */
typedef struct {
  int nblades, npts;
  double hub[3];
  double R, r_hub, omega, theta0, u_ref, eps;
  const double *chord, *twist;         /* npts each: chord length and local twist angle gamma [rad] */
  int npolar;
  const double *alpha, *cl, *cd;       /* tabulated 2-D airfoil data, alpha [rad] increasing */
  int freestream_correction;           /* U_inf^2D = U^2D / (1 - C_D c/(4 sqrt(pi) eps)) */
  int tip_correction;                  /* Eq. 14, (c1, c2) = (0.1219, 21.52) axial, (0.0984, 13.026) tangential */
  /* optional refinements, reading S28 (NULL / 0: the even stations and the single polar above):
     radius, width: npts each - station radii r_k and element widths w_k of Eq. 9, for actuator points "locally refined
       at the tip and root of the blade";
     nsections > 1: cl and cd hold nsections tables of npolar values each, [section][alpha], of airfoil sections at the
       radii section_r[] (increasing); C_L, C_D at a station are linear in r between the two nearby sections ("the
       interpolation of the lift and drag tables between nearby airfoil sections"), the first / last
       section's inside / outside of them */
  const double *radius, *width;
  int nsections;
  const double *section_r;
} gkso_rotor;
int gkso_alm_set_rotor(gkso_ctx *ctx, const gkso_rotor *rotor);
int gkso_alm_rotor_eval(gkso_ctx *ctx, double *pos, double *force); /* test hook: nblades*npts*3 each */
/* dt of the CFL condition */
int gkso_cfl_dt(gkso_ctx *ctx, double cfl, double *dt);
const char *gkso_last_error(void);

/* ---- building blocks, exported so that tests can pin each one separately ---- */
/* <u^n>, n = 0..nmax, of a 1-D Maxwellian with mean U and lambda (Appendix) */
void gkso_moments(double U, double lambda, int nmax, double *out);
/* Appendix solve: a from d = (1/rho) dQ/ds */
void gkso_micro_solve(double U, double V, double W, double lambda, const double d[4], double a[4]);
/* WENO5-JS value at the right edge of the middle cell from 5 cell averages (ref [30]) */
double gkso_weno5_face(const double q[5], double eps);
/* WENO5-JS values at the two Gauss points -sqrt(3)/6, +sqrt(3)/6 of the middle cell (S7) */
void gkso_weno5_gauss(const double q[5], double eps, double out[2]);
void gkso_linear5_gauss(const double q[5], double out[2]);
/* derivative (per unit cell width) of the quartic through 5 averages at the two Gauss points (S8) */
void gkso_quartic_slope_gauss(const double q[5], double out[2]);
/* index-space normal slope at the face between q[1] and q[2] from 4 averages q[0..3] (S5) */
double gkso_normal_slope(const double q[4]);
/* collision: equilibrium state Q0 from left/right states, normal direction dir (S4) */
void gkso_collision(const double Ql[4], const double Qr[4], int dir, double RT, double Q0[4]);
/* Gauss-point flux F and dF/dt (Eq. 7 moments) from Q0 and its slopes dQ[s][c], s = x,y,z */
void gkso_gauss_point_flux(const double Q0[4], const double dQ[12], int dir, double RT, double nu,
                           double rho_ref, double F[4], double dF[4]);
/* 3-point discrete delta (S13) */
double gkso_delta3(double r);
/* Gaussian ALM kernel value per unit force (Eq. 10) */
double gkso_alm_kernel(double r, double eps);

#ifdef __cplusplus
}
#endif
#endif
