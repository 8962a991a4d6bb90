/*
 * gks.h — C ABI of libgks_b200: one two-stage fourth-order (S2O4) step of the high-order
 * gas-kinetic scheme (GKS) for 3-D weakly compressible isothermal flow on a rectilinear
 * Cartesian grid, plus the body-force term carrying ALM and IBM forcing.
 *
 * Source of the method: arxiv/paper_2603_11102.  Citations are "PAPER.md:<line>".
 *   state            Q = (rho, rho*U, rho*V, rho*W)
 *   equilibrium      isothermal Maxwellian, lambda = 1/(2 RT) constant    PAPER.md:49-51 (Eq. 2)
 *   finite volume    dQ/dt = L(Q) = -(1/|Omega|) sum_p F_p(t)             PAPER.md:59-66 (Eq. 4-5)
 *   face flux        2x2 Gauss points per face                            PAPER.md:68-71 (Eq. 6)
 *   distribution     f = g0 (1 - tau (a1 u + a2 v + a3 w + A) + A t)      PAPER.md:75-81 (Eq. 7), tau = mu/p
 *   coefficients     <a_s> = dQ0/ds, <a1 u + a2 v + a3 w + A> = 0         PAPER.md:84 (Eq. 8), Appendix :501-558
 *   reconstruction   5th-order WENO, dimension by dimension
 *   time stepping    two-stage fourth-order
 *   ALM              f = F/(eps^3 pi^1.5) exp(-(r/eps)^2), cut at 3 eps    PAPER.md:137 (Eq. 10), :293
 *   IBM              direct forcing with Lagrangian points                PAPER.md:143-175 (Eq. 11-12)
 *   momentum update  (rho U)~ = (rho U)^{n+1} + f dt/V                    PAPER.md:189 (Eq. 13)
 * Every point on which the paper is silent is fixed by a numbered reading S1..S24 in DESIGN.md.
 *
 * Conventions
 *   - All floating point is IEEE fp64.  Field layout W[c][k][j][i], i fastest, c in {rho, rhoU, rhoV, rhoW},
 *     interior cells only (4*nz*ny*nx doubles) at this boundary; the library keeps its own padded copy.
 *   - Pointers marked "host or device" are classified with cudaPointerGetAttributes; the copy is
 *     enqueued on the context's stream.  The caller owns every array it passes; the library copies
 *     what it needs during the call and never retains a caller pointer, except `workspace`.
 *     A DEVICE array is read or written asynchronously ON THE CONTEXT'S STREAM: the caller orders its own
 *     streams against that one (what another stream wrote must be complete before the call; the array must
 *     stay allocated, and untouched by other streams, until the context's stream has passed the copy).
 *   - `workspace` is DEVICE memory owned by the caller (e.g. a torch tensor), at least
 *     gks_workspace_bytes(cfg) bytes, 256-byte aligned, kept alive until gks_destroy.  No call
 *     allocates device memory.  All kernels are enqueued on `cuda_stream` (a cudaStream_t; NULL = the
 *     legacy default stream).  gks_step is asynchronous; gks_get_state synchronises the stream when
 *     the destination is host memory.
 *   - Every call returns a gks_status, never throws or aborts.  On error the context is unchanged
 *     and gks_last_error(ctx) (or gks_last_error(NULL) for gks_create failures) holds a message.
 *   - A context belongs to the CUDA device that is current at gks_create (the workspace must live there); every
 *     later call must find that device current, else GKS_ERR_STATE.
 *   - A context is not thread-safe.
 *   - There is no CPU fallback: without a CUDA device gks_create returns GKS_ERR_CUDA.
 */
#ifndef GKS_B200_H
#define GKS_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gks_ctx gks_ctx; /* opaque */

typedef enum {
  GKS_OK = 0,
  GKS_ERR_INVALID_ARG = 1,
  GKS_ERR_WORKSPACE = 2, /* workspace NULL, too small or misaligned */
  GKS_ERR_CUDA = 3,      /* a CUDA runtime call failed; message in gks_last_error */
  GKS_ERR_STATE = 4,     /* call order, e.g. gks_step before gks_set_state */
  GKS_ERR_NONFINITE = 5  /* gks_check_finite found a NaN/Inf */
} gks_status;

/* Boundary kinds (PAPER.md:215 periodic + no-slip isothermal wall; :267 Riemann-invariant
 * inlet/outlet + extrapolation; :287 slip wall; :374 symmetry).  Ghost-cell formulas: DESIGN.md S17-S21. */
typedef enum {
  GKS_BC_PERIODIC = 0,
  GKS_BC_WALL_NOSLIP = 1,
  GKS_BC_WALL_SLIP = 2, /* also "symmetry" */
  GKS_BC_INFLOW = 3,
  GKS_BC_OUTFLOW_CONVECTIVE = 4,
  GKS_BC_EXTRAPOLATE = 5,
  GKS_BC_HALO = 6 /* cut face of a domain decomposition: the 3 ghost layers are supplied with gks_halo_unpack */
} gks_bc;

typedef struct {
  int nx, ny, nz;               /* interior cells per axis, each >= 6 */
  const double *xf, *yf, *zf;   /* HOST face coordinates, n+1 each, strictly increasing; NULL => uniform */
  double x0, y0, z0;            /* origin of the low faces (used when the axis is uniform) */
  double dx, dy, dz;            /* spacing (used when the axis is uniform), > 0 */
  double RT;                    /* isothermal constant R*T > 0; lambda = 1/(2 RT), c_s = sqrt(RT) */
  double nu;                    /* kinematic viscosity >= 0; mu = rho_ref*nu, tau = mu/p */
  double rho_ref;               /* reference density > 0 (1 in all configs) */
  int bc[6];                    /* gks_bc for xlo, xhi, ylo, yhi, zlo, zhi; periodic must be paired */
  double inflow[4];             /* rho, U, V, W for GKS_BC_INFLOW; |velocity normal to an outflow face| is
                                   the convective speed of GKS_BC_OUTFLOW_CONVECTIVE */
  double weno_eps;              /* WENO-JS epsilon; 0 => 1e-6; otherwise >= 1e-30 */
} gks_config;

/* Bytes of device workspace gks_create needs for this configuration (0 if cfg is invalid). */
size_t gks_workspace_bytes(const gks_config *cfg);

/* Validate cfg, carve `workspace` (device), upload coordinates.  *out is set only on GKS_OK. */
gks_status gks_create(const gks_config *cfg, void *workspace, size_t workspace_bytes,
                      void *cuda_stream, gks_ctx **out);
gks_status gks_destroy(gks_ctx *ctx);

/* W: host or device, 4*nz*ny*nx doubles, W[c][k][j][i].  set_state also initialises the
 * convective-outflow ghost state (S20).  get_state synchronises for host destinations.
 * Inside a split step (between gks_step_begin and gks_step_force) gks_set_state returns GKS_ERR_STATE; gks_get_state
 * is allowed there and reads W^n after gks_step_begin, the un-forced W^{n+1} after gks_step_finish. */
gks_status gks_set_state(gks_ctx *ctx, const double *W);
gks_status gks_get_state(gks_ctx *ctx, double *W);

/* One S2O4 step W^n -> W^{n+1} (W* = W^n + dt/2 L + dt^2/8 dL,
 * W^{n+1} = W^n + dt L + dt^2/6 (dL(W^n) + 2 dL(W*))) computed without external force
 * (PAPER.md:187), then the forcing of Eq. 13: uniform/bulk term, IBM, ALM.  dt > 0.
 * Asynchronous on the context's stream. */
gks_status gks_step(gks_ctx *ctx, double dt);

/* Domain decomposition (x-slabs over several GPUs).  A sub-domain is an
 * ordinary context whose cut faces carry GKS_BC_HALO.  Only x faces may (x-slabs), on a uniform x axis; a convective
 * outflow may then only sit on that same axis.
 * The ghost fill leaves HALO ghosts alone; the driver moves them:
 *   gks_halo_pack(ctx, which, face, buf)   copies the 3 interior planes next to `face` (0..5 = xlo,xhi,ylo,...)
 *       of state `which` (0: W^n / W^{n+1}, 1: the first-stage state W*) to buf, a DEVICE or host array of
 *       gks_halo_doubles(ctx, face) doubles laid out [c][layer][v][u] (layer = increasing index along the axis,
 *       u the lower and v the higher of the two tangential axes, interior cells only);
 *   gks_halo_unpack(ctx, which, face, buf) writes the 3 ghost planes beyond `face` from such an array (what the
 *       neighbour packed at its opposite face).
 * gks_step is split at the points where it needs its neighbours:
 *   gks_step_begin(ctx, dt)   ghosts of W^n (HALO ghosts must be in place), sweeps, W* and P;
 *   gks_step_finish(ctx, dt)  ghosts of W* (HALO ghosts of W* must be in place), sweeps, un-forced W^{n+1};
 *   gks_step_force(ctx, dt)   forcing of Eq. 13.  IBM points within 1.5 cells of a cut read across it: with IBM
 *       the HALO ghosts of the un-forced W^{n+1} (which = 0) must be in place.  Every sub-domain is given the
 *       Lagrangian points that lie inside it or at most 2 cells beyond a HALO face, interpolates U_p from the
 *       same cells as its neighbour, and adds only to the cells it owns.  The bulk-flux forcing needs the
 *       global sum: between finish and force every sub-domain calls gks_bulk_partial (its sum of
 *       m_axis |Omega| over the un-forced field and its volume), the driver adds them up (one scalar
 *       all-reduce) and returns the totals with gks_bulk_set_global (sum: host or device pointer).
 *       More than one IBM pass (ibm_set_iterations) needs the neighbours' increments between the passes and a
 *       common stop decision: between finish and force the driver runs, for pass k = 0 .. max_iter-1,
 *       [k > 0: exchange of the HALO ghosts, which = 0]  gks_ibm_pass(ctx, k, 0) (interpolate; records this
 *       sub-domain's max slip)  [k > 0: gks_ibm_residual get -> MAX over the sub-domains -> set]
 *       gks_ibm_pass(ctx, k, 1) (spread; skipped on the device once the slip fell below tol); gks_step_force
 *       then leaves the IBM alone.  Not available on a sub-domain: alm_set_rotor (use alm_rotor_points).
 * gks_step = begin + finish + force.  The three parts of one step must be given the same dt.
 * Errors: GKS_ERR_INVALID_ARG (face without HALO, NULL, a dt that differs from gks_step_begin's), GKS_ERR_STATE
 * (order of the calls). */
/* Overlapping the exchange with the sweeps.  Either half of the step can be given in two parts:
 *   gks_step_begin_part(ctx, dt, 0)  ghosts of W^n (HALO ghosts may still be on their way), then the sweeps and the
 *       stage update of the INTERIOR: the tiles and cells that read no HALO ghost (all cells further than 32 from a
 *       HALO low face and further than 6 .. 37 from a HALO high face; none on a sub-domain narrower than about 70);
 *   gks_step_begin_part(ctx, dt, 1)  HALO ghosts of W^n must be in place: the ghost passes over the ghost columns
 *       beyond the HALO faces, then the sweeps and the stage update of the RIM.  Together = gks_step_begin, tile for
 *       tile and cell for cell the same arithmetic.
 *   gks_step_finish_part(ctx, dt, part) likewise for the second stage (HALO ghosts of W*).
 * The driver posts the transfer of a stage's halos, runs part 0, completes the transfer (gks_halo_unpack is allowed
 * between the parts), runs part 1 - and packs the next stage's halos right after it.  The kernels of the two parts
 * are enqueued on the context's stream; a transfer overlaps them when the driver moves it on a stream of its own.
 * Errors: GKS_ERR_STATE (order), GKS_ERR_INVALID_ARG (part, dt). */
gks_status gks_step_begin_part(gks_ctx *ctx, double dt, int part /* 0 interior, 1 rim */);
gks_status gks_step_finish_part(gks_ctx *ctx, double dt, int part);
size_t gks_halo_doubles(const gks_ctx *ctx, int face);
gks_status gks_halo_pack(gks_ctx *ctx, int which, int face, double *buf);
gks_status gks_halo_unpack(gks_ctx *ctx, int which, int face, const double *buf);
/* The exchange without buffers (one node: NVLink 5 / NVSwitch peer memory, or sub-domains that share a GPU).
 * gks_halo_window_get(ctx, which, &w) describes where a neighbour may write this context's padded state `which`
 * directly: device base pointer, extents and pitches.  gks_halo_push(ctx, which, face, &w_neighbour) writes the 3
 * interior planes next to x face `face` of THIS context straight into the ghost planes beyond the OPPOSITE x face of
 * the neighbour - pack, transfer and unpack in one kernel on this context's stream; with the neighbour on another GPU
 * the stores travel peer to peer (the driver enables peer access or maps the window through CUDA IPC, and orders the
 * neighbour's stream behind the push, e.g. with an event).  The window stays valid for the life of the neighbour's
 * context.  Errors: GKS_ERR_INVALID_ARG (not a HALO x face, NULL, y / z extents differ), GKS_ERR_STATE (as gks_halo_pack). */
typedef struct {
  double *W;                       /* device: padded state [c][k][j][i], 3 ghost layers on every side */
  int nx, ny, nz;                  /* interior cells of the neighbour */
  int pitch_x, pitch_y;            /* padded row length (>= nx + 6) and rows per plane (ny + 6), in doubles / rows */
  long long field_stride;          /* doubles between two components */
} gks_halo_window;
gks_status gks_halo_window_get(gks_ctx *ctx, int which, gks_halo_window *out);
gks_status gks_halo_push(gks_ctx *ctx, int which, int face, const gks_halo_window *to);
/* The windows of a sub-domain owned by ANOTHER PROCESS (one process per GPU), mapped with CUDA IPC:
 *   gks_halo_export_get(ctx, &e)        (owner) describes the device allocation that holds the workspace and where the
 *       padded states W^n and W* lie in it; `e` is plain bytes and may be sent to the neighbour's process.  The workspace
 *       must lie inside ONE cudaMalloc allocation (GKS_ERR_WORKSPACE / GKS_ERR_CUDA otherwise).
 *   gks_halo_export_open(&e, win, &map) (neighbour, with the device it pushes from current) maps that allocation -
 *       peer to peer over NVLink when it lives on another GPU - and fills win[0] (W^n) and win[1] (W*) for gks_halo_push.
 *       An allocation opens once per process: open once per neighbour rank.  GKS_ERR_CUDA if it cannot be mapped (also in
 *       the process that owns it); message in gks_last_error(NULL).
 *   gks_halo_export_close(map)          unmaps; the windows are dead afterwards.  Close before the owner frees.
 * The ORDER between the processes is the driver's (paper_2603_11102_b200/slab.py IpcPushTransport: interprocess events -
 * the owner's stream waits for "landed", the pusher's stream for "ghosts free"). */
typedef struct {
  unsigned char mem[64];           /* cudaIpcMemHandle_t of the allocation that holds the workspace */
  unsigned long long offset[2];    /* bytes from the allocation's base to the padded state W^n ([0]) and W* ([1]) */
  int nx, ny, nz, pitch_x, pitch_y;
  long long field_stride;
} gks_halo_export;
gks_status gks_halo_export_get(gks_ctx *ctx, gks_halo_export *out);
gks_status gks_halo_export_open(const gks_halo_export *in, gks_halo_window win[2], void **mapping);
gks_status gks_halo_export_close(void *mapping);
gks_status gks_step_begin(gks_ctx *ctx, double dt);
/* gks_step_begin whose stage update ALSO writes the 3 planes of W* next to the low / high x face into the ghost planes of
 * the neighbour given for that face (to_lo: the sub-domain beyond my low face, to_hi: beyond my high face; its window of
 * state 1 from gks_halo_window_get or gks_halo_export_open; NULL: nobody) - update, pack, transfer and unpack in one
 * kernel, peer-to-peer stores while the rest of the update runs.  Equal to gks_step_begin followed by
 * gks_halo_push(ctx, 1, face, to) for those faces.  The neighbour's W* ghosts must be free (its previous step's second
 * stage has run) and the neighbour must wait for this call's kernels before its gks_step_finish (the driver's order, as
 * for gks_halo_push).  Errors as gks_step_begin and gks_halo_push. */
gks_status gks_step_begin_push(gks_ctx *ctx, double dt, const gks_halo_window *to_lo, const gks_halo_window *to_hi);
gks_status gks_step_finish(gks_ctx *ctx, double dt);
gks_status gks_step_force(gks_ctx *ctx, double dt);
gks_status gks_ibm_pass(gks_ctx *ctx, int pass, int phase /* 0 interpolate, 1 spread */);
gks_status gks_ibm_residual(gks_ctx *ctx, int pass, double *value /* host or device */, int set /* 0 get, 1 set */);
gks_status gks_bulk_partial(gks_ctx *ctx, double *sum, double *volume /* host, may be NULL */);
gks_status gks_bulk_set_global(gks_ctx *ctx, const double *sum, double volume);

/* Uniform acceleration g: momentum += dt * rho * g each step.  (0,0,0) disables. */
gks_status gks_set_body_force(gks_ctx *ctx, double gx, double gy, double gz);
/* "Constant moment flux" forcing of the channel: after each step shift (rho U_axis)
 * uniformly so that its volume-weighted mean equals `target`.  axis in {0,1,2}; axis < 0 disables. */
gks_status gks_set_bulk_flux(gks_ctx *ctx, int axis, double target_bulk_momentum);

/* ALM (Eq. 10): n actuator points; pos and force are n*3 doubles (x,y,z per point),
 * host or device; force = point force ON THE FLUID; eps > 0 is the Gaussian width; the kernel is
 * sampled at cell centres and cut at r <= 3 eps.  n = 0 clears.  n <= GKS_MAX_ALM_POINTS.
 * Points may lie anywhere along a periodic axis (they act through their images); 6 eps must be smaller than every
 * periodic axis length (GKS_ERR_INVALID_ARG otherwise).  On a non-periodic axis the part of a support beyond the
 * domain is lost. */
gks_status alm_set_points(gks_ctx *ctx, int n, const double *pos, const double *force, double eps);

/* On-line actuator-line rotor (Eq. 9, Eq. 14; S26-S27): instead of prescribed point
 * forces, every gks_step (i) places nblades*npts actuator points - rotor axis +x, blade b at azimuth
 * theta0 + omega t + 2 pi b/nblades, station k at r_hub + (k+1/2)(R - r_hub)/npts (or at radius[k]), t = the rotor clock, 0 at this
 * call and advanced by dt per step -, (ii) samples (rho, U) of the un-forced W^{n+1} at the points by trilinear
 * interpolation, (iii) evaluates lift and drag (Eq. 9) from the tabulated polar at alpha = phi - twist,
 * phi = atan2(U_x, omega r - U_theta), optionally with the free-stream correction of PAPER.md:107 and the tip
 * correction of Eq. 14, and (iv) spreads the reaction with Eq. 10 - all on the device.
 * Tables (host or device pointers) are copied during the call: chord, twist [rad] npts each; alpha [rad,
 * increasing], cl, cd npolar each.  npts <= 4096, npolar <= 1024, nblades*npts <= GKS_MAX_ALM_POINTS.
 * NULL clears the rotor; alm_set_points also replaces it.  Errors: GKS_ERR_INVALID_ARG. */
typedef struct {
  int nblades, npts;
  double hub[3];
  double R, r_hub, omega, theta0, u_ref, eps;
  const double *chord, *twist;
  int npolar;
  const double *alpha, *cl, *cd;
  int freestream_correction, tip_correction;
  /* optional refinements, S28 (NULL / 0: the even stations and the single polar above).
     radius, width: npts each - station radii r_k (0 < r_k <= R) and element widths w_k of Eq. 9, for actuator points
       "locally refined at the tip and root of the blade"; they come together.
     nsections > 1 (<= 16, nsections * npolar <= 4096): cl and cd hold nsections tables of npolar values each,
       [section][alpha], of airfoil sections at the radii section_r[] (increasing); C_L, C_D at a station are linear in r
       between the two nearby sections ("the interpolation of the lift and drag tables between nearby airfoil sections",
       PAPER.md:127), the first / last section's inside / outside of them. */
  const double *radius, *width;
  int nsections;
  const double *section_r;
} alm_rotor;
gks_status alm_set_rotor(gks_ctx *ctx, const alm_rotor *rotor);
/* Test hook: positions and forces ON THE FLUID (nblades*npts*3 doubles each, host or device) of the actuator
 * points for the CURRENT state and rotor clock; synchronises the stream unless both pointers are device memory. */
gks_status alm_rotor_eval(gks_ctx *ctx, double *pos, double *force);

/* The on-line rotor on a sub-domain (x-slab decomposition).  alm_set_rotor is accepted on every sub-domain: each
 * keeps the rotor description and the rotor clock (advanced by dt in every gks_step_force, so all clocks agree), but
 * the sampling reads across cuts, so a sub-domain does not evaluate the blade forces inside gks_step_force.  Between
 * gks_step_finish and gks_step_force the driver (i) has the sub-domain that contains the disc evaluate them with
 * alm_rotor_eval (device pointers: asynchronous), (ii) broadcasts the two small arrays and (iii) hands them to every
 * sub-domain with alm_rotor_supply(ctx, pos, force, x_shift): nblades*npts*3 doubles each, host or device; x_shift is
 * added to every x coordinate (a slab beyond the seam of a periodic x axis meets the disc through its image; else 0).
 * gks_step_force on a sub-domain with a rotor set and nothing supplied for the step: GKS_ERR_STATE. */
gks_status alm_rotor_supply(gks_ctx *ctx, const double *pos, const double *force, double x_shift);

/* The same front half without state in the context: positions and forces ON THE FLUID of the actuator points of
 * `rotor` at rotor time t, sampled from the CURRENT state (between gks_step_finish and gks_step_force: the
 * un-forced W^{n+1}).  For drivers that own the rotor clock - the x-slab driver evaluates the rotor on the
 * sub-domain that contains the disc (sampling reads the first HALO ghost layer), broadcasts the forces and hands
 * them to every sub-domain with alm_set_points.  pos, force: nblades*npts*3 doubles each, host (the call then
 * synchronises) or device.  GKS_ERR_STATE while a rotor is set with alm_set_rotor. */
gks_status alm_rotor_points(gks_ctx *ctx, const alm_rotor *rotor, double t, double *pos, double *force);

/* IBM: n Lagrangian points; pos n*3 doubles, weights n doubles = V_p = dx*dS
 * (PAPER.md:155); host or device.  Velocities default to 0 (stationary body).
 * Each point must lie inside the domain and the grid must be locally uniform over its 3x3x3
 * support, else GKS_ERR_INVALID_ARG.  n = 0 clears.  n <= GKS_MAX_IBM_POINTS. */
gks_status ibm_set_points(gks_ctx *ctx, int n, const double *pos, const double *weights);
gks_status ibm_set_velocities(gks_ctx *ctx, const double *vel /* n*3, or NULL => 0 */);

/* IBM multi-direct-forcing passes per step (Eq. 11-12; S25): pass s interpolates
 * U_p^s from the un-forced field plus the IBM increments of the passes before it and spreads
 * rho_ijk (v_p - U_p^s) phi phi phi V_p/|Omega_ijk|; the increments add up (Eq. 12).  From the second pass
 * on the passes stop once max_p |v_p - U_p^s| < tol (decided on the device: gks_step stays asynchronous).
 * Default max_iter = 1, tol = 0 (single pass).  1 <= max_iter <= 64, tol >= 0, else GKS_ERR_INVALID_ARG. */
gks_status ibm_set_iterations(gks_ctx *ctx, int max_iter, double tol);

/* Scheme variant for cost comparison (the alternative of DESIGN.md reading S7): with
 * tangential_linear = 1 the two tangential passes combine the sub-stencil candidates with the LINEAR weights
 * (quartic interpolation to the Gauss points) instead of the WENO5-JS nonlinear ones; the normal reconstruction,
 * the slopes and everything else are unchanged.  Default 0.  Other values: GKS_ERR_INVALID_ARG. */
gks_status gks_set_reconstruction(gks_ctx *ctx, int tangential_linear);

/* Time step of the CFL condition: dt = cfl * min{dx, dy, dz} / (|U|_max + sqrt(RT)), |U|_max over
 * the interior cells of the current state (one reduction kernel), the minimum over every cell width.
 * `dt` may be a host pointer (the call then synchronises the stream) or a device pointer (asynchronous).
 * cfl <= 0 -> GKS_ERR_INVALID_ARG; before gks_set_state -> GKS_ERR_STATE. */
gks_status gks_cfl_dt(gks_ctx *ctx, double cfl, double *dt);

/* The same time step for callers that cannot allocate device memory (CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): no context and no workspace.  The reduction's scratch (one partial maximum per
 * block of GKS_NOALLOC_CELLS_PER_BLOCK cells) is a file-scope __device__ array of GKS_NOALLOC_MAX_BLOCKS doubles
 * (512 KB, held by every GPU that loads the library until the process exits); the call allocates and frees nothing.
 *   W     DEVICE, 4*nz*ny*nx doubles, W[c][k][j][i] (the layout of gks_set_state); read only; owned by the caller
 *   dmin  smallest cell width over the three axes (> 0); RT > 0; cfl > 0
 *   dt    DEVICE, one double, written asynchronously on cuda_stream (a cudaStream_t; NULL = legacy default stream)
 * The CUDA device that holds W and dt must be current.  Asynchronous: two kernels on cuda_stream, no synchronisation.
 * Errors (message in gks_noalloc_last_error(), per thread): NULL or host pointers, sizes < 1, non-positive dmin / RT / cfl
 * -> GKS_ERR_INVALID_ARG; nx*ny*nz > GKS_NOALLOC_MAX_CELLS -> GKS_ERR_INVALID_ARG (use gks_cfl_dt with a workspace);
 * a failing CUDA call -> GKS_ERR_CUDA.  dt is untouched on error.
 * All calls on a device SHARE the scratch array: calls whose kernels may overlap on the GPU (different streams with no
 * ordering between them) race; calls on one stream, or ordered by events, are safe.  Nothing in the array has to be
 * cleared between calls (every slot that is read was written by the same call first). */
#define GKS_NOALLOC_CELLS_PER_BLOCK 4096
#define GKS_NOALLOC_MAX_BLOCKS 65536
#define GKS_NOALLOC_MAX_CELLS ((long long)GKS_NOALLOC_MAX_BLOCKS * GKS_NOALLOC_CELLS_PER_BLOCK) /* 2^28 = 268 435 456 */
gks_status gks_cfl_dt_noalloc(const double *W, int nx, int ny, int nz, double dmin, double RT, double cfl, double *dt,
                              void *cuda_stream);
const char *gks_noalloc_last_error(void);

/* Test hook: fill ghosts of the CURRENT state and evaluate the face-averaged flux F and its
 * time derivative dF/dt (Eq. 6-7) for sweep direction dir in {0,1,2}.  Output (host or device):
 * 4 * (faces) doubles each, faces laid out like cells but with n_dir+1 entries along `dir`,
 * component-major: F[c][k][j][i].  Does not modify the state.  GKS_ERR_STATE inside a split step. */
gks_status gks_debug_eval_flux(gks_ctx *ctx, int dir, double *F, double *dFdt);

/* Synchronising check of the current state; GKS_ERR_NONFINITE if any interior value is NaN/Inf. */
gks_status gks_check_finite(gks_ctx *ctx);

/* Per-kernel-class device timing.  When enabled, gks_step brackets each class of kernels with CUDA
 * events on the context's stream; gks_profile_read synchronises, ADDS the elapsed milliseconds and
 * interval counts of everything recorded since the last read into ms[GKS_PROF_N] / count[GKS_PROF_N]
 * (host arrays the caller zeroes) and resets the recorder.  At most 4096 intervals are kept between
 * reads (later ones are dropped). */
enum { GKS_PROF_GHOST = 0, GKS_PROF_SWEEP_X = 1, GKS_PROF_SWEEP_Y = 2, GKS_PROF_SWEEP_Z = 3,
       GKS_PROF_UPDATE = 4, GKS_PROF_FORCING = 5, GKS_PROF_N = 6 };
gks_status gks_profile_enable(gks_ctx *ctx, int on);
gks_status gks_profile_read(gks_ctx *ctx, double *ms, long long *count);

/* Number of kernels this context has launched since gks_create (for bench.py's gpu_launches). */
long long gks_launch_count(const gks_ctx *ctx);

const char *gks_last_error(const gks_ctx *ctx);

#define GKS_MAX_ALM_POINTS 65536
#define GKS_MAX_IBM_POINTS 4194304

#ifdef __cplusplus
}
#endif
#endif /* GKS_B200_H */
