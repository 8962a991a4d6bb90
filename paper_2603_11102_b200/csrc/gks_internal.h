/*
 * gks_internal.h — internal declarations of libgks_b200 (CUDA path).  Not part of the C ABI.
 *
 * HBM layout.  Every field lives in ONE index space: the padded cell box with NG = 3 ghost layers,
 *   idx(i,j,k) = ((k+3)*PY + (j+3))*PX + (i+3),   i fastest, PX = round_up(nx+6, 4) doubles,
 * fields are separated by FS = PX*PY*PZ doubles (component-major, W[c][k][j][i]).
 * Face-based arrays (fluxes of sweep direction d) reuse the same index space: face f along d
 * (between cells f-1 and f, f = 0..n_d) is stored at cell index f.
 */
#ifndef GKS_INTERNAL_H
#define GKS_INTERNAL_H

#include <cuda_runtime.h>
#include <stddef.h>

#include "../../include/gks.h"
#ifdef GKS_DEBUG
#include "../../include/gks_debug.h"
#endif

#define GKS_NG 3

/* Geometry handed to kernels by value. */
struct GksGrid {
  int n[3];          /* interior cells */
  int P[3];          /* padded extents (P[0] is the pitch) */
  long long st[3];   /* strides of i, j, k in doubles: 1, PX, PX*PY */
  long long FS;      /* field stride */
  /* per-axis coordinate tables on the device, indexed with (cell index + 3), length n+6 (+1 for xf) */
  const double *xf[3];     /* faces  -3 .. n+3 */
  const double *xc[3];     /* centres -3 .. n+2 */
  const double *w[3];      /* widths */
  const double *inv_w[3];  /* 1/width */
  const double *inv_12hn[3]; /* 1/(12 (xc[f]-xc[f-1])) for face f = -2 .. n+2, stored at f+3 (normal slope S5) */
  int uniform[3];
  double x0[3], dx[3];
  double inv_w_u[3], inv_12hn_u[3];   /* uniform axis: the one value of inv_w / inv_12hn (kernel-parameter operands) */
  int periodic[3];
  int halo[6];       /* face carries GKS_BC_HALO: its ghost layers hold the neighbouring sub-domain's cells */
  int wrapf[3];      /* face n of this axis is not stored: it is face 0 (periodic axis, see gks_create) */
  __host__ __device__ long long idx(int i, int j, int k) const {
    return ((long long)(k + GKS_NG) * P[1] + (j + GKS_NG)) * P[0] + (i + GKS_NG);
  }
};

struct GksPhys {
  double RT, lambda, mu, weno_eps4; /* mu = rho_ref*nu; 4 x the WENO epsilon (the smoothness indicators are carried x 4) */
  double theta, cx;                /* sqrt(lambda), 1/(2 sqrt(pi lambda)): collision constants */
  double inflow[4];
  int bc[6];
  int tang_linear;                 /* scheme variant: linear weights in the tangential passes */
};

/* on-line actuator-line rotor handed to the kernel by value; table pointers are device memory */
struct GksRotor {
  int nb, np, npolar, fs_corr, tip_corr, nsec;
  double hub[3], R, rhub, omega, theta0, uref;
  const double *chord, *twist, *radius, *width;   /* np each; radius / width always filled (even spacing by default) */
  const double *alpha, *cl, *cd, *sec_r;          /* alpha npolar; cl, cd [nsec][npolar]; sec_r nsec */
};
#define GKS_MAX_ROTOR_STATIONS 4096
#define GKS_MAX_POLAR 1024
#define GKS_MAX_SECTIONS 16                        /* nsections * npolar <= GKS_MAX_SECTIONS * GKS_MAX_POLAR / 4 */
#define GKS_ROTOR_TAB_DOUBLES (4 * GKS_MAX_ROTOR_STATIONS + GKS_MAX_POLAR + 2 * 4 * GKS_MAX_POLAR + GKS_MAX_SECTIONS)

struct gks_ctx {
  gks_config cfg;
  GksGrid g;
  GksPhys ph;
  cudaStream_t stream;
  bool have_state;
  int mid_step;               /* 0 idle, 1 after gks_step_begin, 2 after gks_step_finish (forcing pending) */
  double step_dt;             /* dt of the step in flight (gks_step_begin): finish and force must be given the same */
  int device;                 /* CUDA device of the workspace and stream: every call must find it current */
  int sweep_mode;             /* 0 fused, 1 unfused (GKS_DEBUG builds only) */
  long long launches;
  char err[512];

  /* workspace carve (device) */
  double *Wn, *Ws, *Pbuf;      /* padded 4-field states; Pbuf doubles as staging between steps */
  double *flux[3];             /* per direction: F[4] then dF[4], padded index space */
  double *tmpN, *tmpT;         /* unfused cross-check sweep: 8 and 24 padded fields of intermediates; NULL unless
                                  GKS_DEBUG (the struct layout does not depend on the macro: objects are shared) */
  double *coords;              /* coordinate tables */
  double *red;                 /* reduction scratch (partials + result) */
  double *alm_pos, *alm_force; /* GKS_MAX_ALM_POINTS*3 each */
  double *ibm_pos, *ibm_vol, *ibm_vel, *ibm_coef; /* capacity fixed at create */
  int ibm_capacity;

  /* host-side mirrors of the coordinate tables (validation, bounding boxes) */
  double *h_xf[3], *h_xc[3], *h_w[3];

  /* forcing state */
  double gacc[3];
  int bulk_axis;
  double bulk_target, total_volume;
  int ibm_external;            /* sub-domain: this step's IBM passes were driven with gks_ibm_pass */
  int bulk_external;           /* sub-domain: the global sum was supplied with gks_bulk_set_global for this step */
  double bulk_volume_ext;      /* and the global volume */
  double dmin;                 /* smallest cell width of the grid (CFL condition) */
  int n_alm;
  double alm_eps;
  int alm_lo[3], alm_cnt[3];   /* bounding box of the ALM support in (unwrapped) cell indices */
  GksRotor rotor;              /* valid when rotor_on */
  int rotor_on;
  int rotor_external;          /* sub-domain: this step's actuator points were supplied with alm_rotor_supply */
  double rotor_time;           /* rotor clock: 0 at alm_set_rotor, + dt per step */
  double *rotor_out;           /* device scratch of alm_rotor_points: pos, force (GKS_MAX_ALM_POINTS*3 each) */
  double *rotor_tab;           /* device: chord, twist, radius, width (GKS_MAX_ROTOR_STATIONS each), alpha (GKS_MAX_POLAR),
                                  cl, cd (4 GKS_MAX_POLAR each: all sections), section radii: GKS_ROTOR_TAB_DOUBLES */
  int n_ibm;
  int ibm_maxit;               /* multi-direct-forcing passes per step (1 = single pass) */
  double ibm_tol;              /* stop once max_p |v_p - U_p| < tol, from the second pass on */

  /* TMA tensor maps of the two state buffers (Wn, Ws) for the three sweep directions (opaque CUtensorMap) */
  alignas(64) unsigned char tmaps[2][3][128];
  int num_sms;                 /* SMs of the device: the fused sweep launches persistent CTAs */
  /* interior / rim split of a sub-domain (gks_step_begin_part): tiles [part_t0, part_t1) along x of every sweep
     direction and cells [part_x0, part_x1) read no HALO ghost; empty interior: part_x1 <= part_x0 */
  int part_t0[3], part_t1[3], part_x0, part_x1;

  /* per-class event timing (gks_profile.cu) */
  int prof_on, prof_n;
  cudaEvent_t *prof_ev;        /* 2 * GKS_PROF_MAX events, created on first enable */
  int *prof_cat;
};
#define GKS_IBM_MAX_PASSES 64
#define GKS_RED_BULK_SUM 1024  /* ctx->red + this: sum of m_axis |Omega| (gks_forcing.cu: RED_BLOCKS partials before it) */
#define GKS_RED_CFL 1680       /* ctx->red + this: |U|_max bits, dt */
#define GKS_RED_IBM_RES 1600   /* ctx->red + this: GKS_IBM_MAX_PASSES residual slots (bit patterns) */
#define GKS_PROF_MAX 4096
void gks_prof_begin(gks_ctx *ctx, int cat);
void gks_prof_end(gks_ctx *ctx);
void gks_prof_free(gks_ctx *ctx);

/* ---- programmatic dependent launch (PDL) ----
 * Every kernel of the library starts with gks_pdl_enter(): it lets the NEXT kernel on the stream be launched at once
 * (griddepcontrol.launch_dependents) and then waits until the PREVIOUS one has completed and its memory is visible
 * (griddepcontrol.wait) before it touches global memory - so the launch latency and the prologue of a kernel (barrier
 * set-up, index arithmetic) hide behind the tail of its predecessor while the data dependences of the stream stay what
 * they were.  gks_launch() launches with the attribute that allows this where it is safe (below); GKS_NO_PDL=1 in the
 * environment turns the attribute off (the device side is then a no-op).  Matters on small grids: a step is 14-18
 * short kernels.  The persistent sweep releases its successor only at its end (gks_sweep_fused.cu). */
#ifdef __CUDACC__
#include <cstdlib>
#include <cstring>
#include <utility>
__device__ __forceinline__ void gks_pdl_enter() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
inline bool gks_pdl_allowed() {
  static const bool on = [] {
    const char *e = getenv("GKS_NO_PDL");
    return !(e && e[0] == '1');
  }();
  return on;
}
/* The attribute replaces the stream dependency on the previous KERNEL by the programmatic one; it does not order the
 * launch against a memset / memcpy / event record enqueued in between (found on B200: a reduction kernel launched this
 * way overtook the memset of its accumulator).  So it is used only where the library itself has just launched the
 * previous operation of the stream and that operation was a kernel: inside gks_step_begin / _finish / _force
 * (GksPdlScope), from the second kernel of the call on, and not across a memset (gks_pdl_break). */
extern thread_local cudaStream_t gks_pdl_prev;   /* stream whose latest operation is a kernel of the current scope */
extern thread_local bool gks_pdl_scope;
inline void gks_pdl_break() { gks_pdl_prev = nullptr; }
struct GksPdlScope {
  explicit GksPdlScope(bool on) {
    gks_pdl_scope = on && gks_pdl_allowed();
    gks_pdl_prev = nullptr;
  }
  ~GksPdlScope() {
    gks_pdl_scope = false;
    gks_pdl_prev = nullptr;
  }
};
template <typename... KArgs, typename... Args>
inline cudaError_t gks_launch(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args &&...args) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = (gks_pdl_scope && s != nullptr && gks_pdl_prev == s) ? 1 : 0;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
  gks_pdl_prev = gks_pdl_scope ? s : nullptr;
  return e;
}
#endif

/* ---- host helpers shared by the API translation units ---- */
gks_status gks_set_err(gks_ctx *ctx, gks_status st, const char *fmt, ...);
gks_status gks_check_device(gks_ctx *ctx);   /* GKS_ERR_STATE unless the context's device is the current one */
bool gks_is_device_ptr(const void *p);
int gks_host_find_cell(const gks_ctx *ctx, int a, double x); /* interior cell containing x, or -1 */

/* ---- kernel launchers (each returns the number of kernels it enqueued) ---- */
int gks_launch_ghost_fill(const GksGrid &g, const GksPhys &ph, double *W, const double *Wstate, cudaStream_t s);
int gks_launch_outflow_init(const GksGrid &g, const GksPhys &ph, double *W, cudaStream_t s);
int gks_launch_outflow_advance(const GksGrid &g, const GksPhys &ph, double *W, double dt, cudaStream_t s);
int gks_launch_pack(const GksGrid &g, const double *Wint, double *Wpad, cudaStream_t s);
int gks_launch_unpack(const GksGrid &g, const double *Wpad, double *Wint, cudaStream_t s);
int gks_launch_halo(const GksGrid &g, double *W, double *buf, int face, int unpack, cudaStream_t s);
int gks_launch_halo_push(const GksGrid &g, const double *W, int side, double *dstW, int dnx, int dPX, int dPY,
                         long long dFS, cudaStream_t s);
int gks_launch_unpack_faces(const GksGrid &g, int dir, const double *Fpad, double *Fout, cudaStream_t s);

#ifdef GKS_DEBUG
/* unfused cross-check sweep of one direction: fills flux[dir] (F and dF; stage 2 needs only dF) */
int gks_launch_sweep_unfused(const GksGrid &g, const GksPhys &ph, int dir, const double *W, double *tmpN,
                             double *tmpT, double *flux, bool need_F, cudaStream_t s);
#endif

/* fused sweep (gks_sweep_fused.cu); which = 0 reads Wn, 1 reads Ws */
bool gks_fused_init(gks_ctx *ctx);
int gks_launch_sweep_fused(gks_ctx *ctx, int dir, int which, double *flux, bool need_F, int part = 0);
void gks_fused_tiles_x(const GksGrid &g, int ta[3]);

/* where the stage-1 update also stores the 3 planes of W* next to a cut x face: the padded state of the sub-domain
   beyond my low face ([0]: its HIGH ghosts) and beyond my high face ([1]: its low ghosts); W = NULL: nobody */
struct GksPush {
  double *W[2];
  int nx[2], PX[2], PY[2];
  long long FS[2];
};
/* stage updates of the cells with x index in [x0, x1) (x1 < 0: the whole grid) */
int gks_launch_stage1(const GksGrid &g, const double *Wn, double *const flux[3], double dt, double *Ws,
                      double *Pbuf, cudaStream_t s, int x0 = 0, int x1 = -1, const GksPush *push = nullptr);
int gks_launch_stage2(const GksGrid &g, const double *Pbuf, double *const flux[3], double dt, double *Wn,
                      cudaStream_t s, int x0 = 0, int x1 = -1);
/* y and z ghost passes over the x-ghost columns beyond the HALO faces only (after a halo unpack) */
int gks_launch_ghost_fill_xcols(const GksGrid &g, const GksPhys &ph, double *W, const double *Wstate, cudaStream_t s);

int gks_launch_bulk_reduce(const GksGrid &g, const double *W, int axis, double *red, cudaStream_t s);
int gks_launch_uniform_force(const GksGrid &g, double *W, double dt, const double gacc[3], int bulk_axis,
                             double bulk_target, double total_volume, const double *red, cudaStream_t s);
int gks_launch_ibm_interp(const GksGrid &g, const double *W, int n, const double *pos, const double *vol,
                          const double *vel, double *coef, int pass, double tol, unsigned long long *res,
                          cudaStream_t s);
int gks_launch_ibm_spread(const GksGrid &g, double *W, int n, const double *pos, const double *coef, int pass,
                          double tol, const unsigned long long *res, cudaStream_t s);
int gks_launch_alm(const GksGrid &g, double *W, int n, const double *pos, const double *force, double eps,
                   double dt, const int lo[3], const int cnt[3], cudaStream_t s);
int gks_launch_cfl_dt(const GksGrid &g, const double *W, double cfl, double dmin, double cs, double *scratch,
                      cudaStream_t s);
int gks_launch_shift_x(double *pos, int n, double shift, cudaStream_t s);
int gks_launch_rotor_forces(const GksGrid &g, const double *W, const GksRotor &r, double time, double eps,
                            double *pos, double *force, cudaStream_t s);
int gks_launch_check_finite(const GksGrid &g, const double *W, int *flag, cudaStream_t s);

#endif
