/*
 * gks_api.cu — the C ABI of include/gks.h: validation, workspace carving, coordinate tables,
 * state transfer and the sequence of kernels that makes one S2O4 step with forcing.
 * Host code only orchestrates; every step of the path runs in the kernels of this directory.
 */
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "gks_internal.h"

namespace {

char g_create_error[512] = "";

} /* namespace */

thread_local cudaStream_t gks_pdl_prev = nullptr;
thread_local bool gks_pdl_scope = false;

gks_status gks_set_err(gks_ctx *ctx, gks_status st, const char *fmt, ...) {
  char *dst = ctx ? ctx->err : g_create_error;
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(dst, 512, fmt, ap);
  va_end(ap);
  return st;
}
#define set_err gks_set_err

namespace {

#define CUDA_TRY(ctx, call)                                                                              \
  do {                                                                                                   \
    cudaError_t e_ = (call);                                                                             \
    if (e_ != cudaSuccess) return set_err(ctx, GKS_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));   \
  } while (0)

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

const char *validate(const gks_config *c) {
  if (!c) return "config is NULL";
  if (c->nx < 6 || c->ny < 6 || c->nz < 6) return "nx, ny, nz must each be >= 6";
  /* kernels index a padded field with 32 bits (a field of 2^31 doubles is 17 GB; 36 of them exceed any one GPU) */
  if (((long long)c->nx + 9) * ((long long)c->ny + 6) * ((long long)c->nz + 6) >= 2147483647LL)
    return "too many cells: a padded field must hold fewer than 2^31 doubles";
  if (!(c->RT > 0)) return "RT must be > 0";
  if (!(c->nu >= 0)) return "nu must be >= 0";
  if (!(c->rho_ref > 0)) return "rho_ref must be > 0";
  /* the common-denominator WENO weights carry products of about eps^8: below 1e-30 they leave the fp64 range */
  if (c->weno_eps < 0 || (c->weno_eps > 0 && c->weno_eps < 1e-30)) return "weno_eps must be 0 (default 1e-6) or >= 1e-30";
  const int n[3] = {c->nx, c->ny, c->nz};
  const double *f[3] = {c->xf, c->yf, c->zf};
  const double d[3] = {c->dx, c->dy, c->dz};
  for (int a = 0; a < 3; ++a) {
    const int lo = c->bc[2 * a], hi = c->bc[2 * a + 1];
    if (lo < 0 || lo > 6 || hi < 0 || hi > 6) return "unknown boundary kind";
    if ((lo == GKS_BC_HALO || hi == GKS_BC_HALO) && a != 0) return "HALO faces are built for x-slabs: x faces only";
    if ((lo == GKS_BC_HALO || hi == GKS_BC_HALO) && f[a]) return "a HALO face needs a uniform axis";
    if (lo == GKS_BC_HALO || hi == GKS_BC_HALO)
      for (int b = 0; b < 3; ++b)
        if (b != a && (c->bc[2 * b] == GKS_BC_OUTFLOW_CONVECTIVE || c->bc[2 * b + 1] == GKS_BC_OUTFLOW_CONVECTIVE))
          return "with a HALO face a convective outflow may only sit on the same axis";
    if ((lo == GKS_BC_PERIODIC) != (hi == GKS_BC_PERIODIC)) return "periodic faces must be paired";
    if (f[a]) {
      for (int i = 0; i < n[a]; ++i)
        if (!(f[a][i + 1] > f[a][i])) return "face coordinates must be strictly increasing";
    } else if (!(d[a] > 0)) {
      return "spacing must be > 0";
    }
  }
  return nullptr;
}

struct Layout {
  int P[3];
  size_t FS;       /* doubles per padded field */
  size_t off_Wn, off_Ws, off_P, off_flux[3], off_coords, off_red, off_alm_pos,
      off_alm_force, off_rotor, off_rotor_out, off_ibm_pos, off_ibm_vol, off_ibm_vel, off_ibm_coef, total;
  size_t coords_doubles;
  int ibm_capacity;
#ifdef GKS_DEBUG
  size_t off_tmpN, off_tmpT;   /* intermediates of the unfused cross-check sweep: debug library only */
#endif
};

Layout make_layout(const gks_config *c) {
  Layout L;
  L.P[0] = (int)align_up((size_t)c->nx + 2 * GKS_NG, 4);
  L.P[1] = c->ny + 2 * GKS_NG;
  L.P[2] = c->nz + 2 * GKS_NG;
  L.FS = align_up((size_t)L.P[0] * L.P[1] * L.P[2], 32);
  size_t off = 0;
  auto take = [&](size_t doubles) {
    size_t o = off;
    off = align_up(off + doubles * sizeof(double), 256);
    return o;
  };
  L.off_Wn = take(4 * L.FS);
  L.off_Ws = take(4 * L.FS);
  L.off_P = take(4 * L.FS);
  for (int d = 0; d < 3; ++d) L.off_flux[d] = take(8 * L.FS);
#ifdef GKS_DEBUG
  L.off_tmpN = take(8 * L.FS);
  L.off_tmpT = take(24 * L.FS);
#endif
  /* per axis: xf (n+7), xc, w, inv_w, inv_12hn (n+6 each) */
  L.coords_doubles = 0;
  const int n[3] = {c->nx, c->ny, c->nz};
  for (int a = 0; a < 3; ++a) L.coords_doubles += 5 * (size_t)(n[a] + 8);
  L.off_coords = take(L.coords_doubles);
  L.off_red = take(2048);
  L.off_alm_pos = take(3 * (size_t)GKS_MAX_ALM_POINTS);
  L.off_alm_force = take(3 * (size_t)GKS_MAX_ALM_POINTS);
  L.off_rotor = take((size_t)GKS_ROTOR_TAB_DOUBLES);
  L.off_rotor_out = take(6 * (size_t)GKS_MAX_ALM_POINTS);
  /* IBM capacity: one point per 8 cells, at least 65536, at most GKS_MAX_IBM_POINTS */
  size_t cap = (size_t)c->nx * c->ny * c->nz / 8;
  if (cap < 65536) cap = 65536;
  if (cap > GKS_MAX_IBM_POINTS) cap = GKS_MAX_IBM_POINTS;
  L.ibm_capacity = (int)cap;
  L.off_ibm_pos = take(3 * cap);
  L.off_ibm_vol = take(cap);
  L.off_ibm_vel = take(3 * cap);
  L.off_ibm_coef = take(3 * cap);
  L.total = off;
  return L;
}

/* host coordinate tables of one axis (S10): uniform axes use x0 + i dx with exact width;
 * given faces are extended by the periodic image or by mirroring the spacing about the boundary */
void build_axis(int n, const double *faces, double x0, double dx, bool periodic, double *xf, double *xc,
                double *w) {
  if (!faces) {
    for (int i = -GKS_NG; i <= n + GKS_NG; ++i) xf[i + GKS_NG] = x0 + i * dx;
    for (int i = -GKS_NG; i < n + GKS_NG; ++i) {
      w[i + GKS_NG] = dx;
      xc[i + GKS_NG] = x0 + (i + 0.5) * dx;
    }
    return;
  }
  for (int i = 0; i <= n; ++i) xf[i + GKS_NG] = faces[i];
  for (int gi = 1; gi <= GKS_NG; ++gi) {
    if (periodic) {
      xf[GKS_NG - gi] = faces[0] - (faces[n] - faces[n - gi]);
      xf[GKS_NG + n + gi] = faces[n] + (faces[gi] - faces[0]);
    } else {
      xf[GKS_NG - gi] = faces[0] - (faces[gi] - faces[0]);
      xf[GKS_NG + n + gi] = faces[n] + (faces[n] - faces[n - gi]);
    }
  }
  for (int i = 0; i < n + 2 * GKS_NG; ++i) {
    w[i] = xf[i + 1] - xf[i];
    xc[i] = 0.5 * (xf[i] + xf[i + 1]);
  }
}

} /* namespace */

bool gks_is_device_ptr(const void *p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

gks_status gks_check_device(gks_ctx *ctx) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device)
    return gks_set_err(ctx, GKS_ERR_STATE, "the context was created on CUDA device %d but device %d is current", ctx->device, dev);
  return GKS_OK;
}

int gks_host_find_cell(const gks_ctx *ctx, int a, double x) {
  const int n = ctx->g.n[a];
  const double *xf = ctx->h_xf[a] + GKS_NG;
  if (!(x >= xf[0] && x <= xf[n])) return -1;
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    const int mid = (lo + hi) / 2;
    if (x >= xf[mid]) lo = mid; else hi = mid;
  }
  return lo;
}
#define is_device_ptr gks_is_device_ptr

extern "C" {

const char *gks_last_error(const gks_ctx *ctx) { return ctx ? ctx->err : g_create_error; }

long long gks_launch_count(const gks_ctx *ctx) { return ctx ? ctx->launches : 0; }

size_t gks_workspace_bytes(const gks_config *cfg) {
  if (validate(cfg)) return 0;
  return make_layout(cfg).total;
}

gks_status gks_create(const gks_config *cfg, void *workspace, size_t workspace_bytes, void *cuda_stream,
                      gks_ctx **out) {
  if (!out) return set_err(nullptr, GKS_ERR_INVALID_ARG, "out is NULL");
  if (const char *msg = validate(cfg)) return set_err(nullptr, GKS_ERR_INVALID_ARG, "%s", msg);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return set_err(nullptr, GKS_ERR_CUDA, "no CUDA device: libgks_b200 has no CPU fallback");
  }
  const Layout L = make_layout(cfg);
  if (!workspace) return set_err(nullptr, GKS_ERR_WORKSPACE, "workspace is NULL");
  if (((size_t)workspace & 255) != 0) return set_err(nullptr, GKS_ERR_WORKSPACE, "workspace must be 256-byte aligned");
  if (workspace_bytes < L.total)
    return set_err(nullptr, GKS_ERR_WORKSPACE, "workspace too small: %zu < %zu bytes", workspace_bytes, L.total);
  if (!is_device_ptr(workspace)) return set_err(nullptr, GKS_ERR_WORKSPACE, "workspace is not device memory");
  /* kernels, tensor maps and the SM count are those of the CURRENT device: it must be the workspace's */
  int cur_dev = -1;
  cudaPointerAttributes wat;
  if (cudaGetDevice(&cur_dev) != cudaSuccess || cudaPointerGetAttributes(&wat, workspace) != cudaSuccess) {
    cudaGetLastError();
    return set_err(nullptr, GKS_ERR_CUDA, "cannot query the current device");
  }
  if (wat.type == cudaMemoryTypeDevice && wat.device != cur_dev)
    return set_err(nullptr, GKS_ERR_WORKSPACE, "workspace lives on CUDA device %d but device %d is current", wat.device, cur_dev);

  gks_ctx *ctx = new (std::nothrow) gks_ctx();
  if (!ctx) return set_err(nullptr, GKS_ERR_INVALID_ARG, "out of host memory");
  memset(ctx, 0, sizeof(*ctx));
  ctx->cfg = *cfg;
  ctx->cfg.xf = ctx->cfg.yf = ctx->cfg.zf = nullptr; /* caller pointers are not retained */
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->device = cur_dev;         /* workspace, stream and tensor maps belong to the device that is current now */
  ctx->bulk_axis = -1;
  ctx->ibm_maxit = 1;
  char *base = (char *)workspace;
  ctx->Wn = (double *)(base + L.off_Wn);
  ctx->Ws = (double *)(base + L.off_Ws);
  ctx->Pbuf = (double *)(base + L.off_P);
  for (int d = 0; d < 3; ++d) ctx->flux[d] = (double *)(base + L.off_flux[d]);
#ifdef GKS_DEBUG
  ctx->tmpN = (double *)(base + L.off_tmpN);
  ctx->tmpT = (double *)(base + L.off_tmpT);
#endif
  ctx->coords = (double *)(base + L.off_coords);
  ctx->red = (double *)(base + L.off_red);
  ctx->alm_pos = (double *)(base + L.off_alm_pos);
  ctx->alm_force = (double *)(base + L.off_alm_force);
  ctx->rotor_tab = (double *)(base + L.off_rotor);
  ctx->rotor_out = (double *)(base + L.off_rotor_out);
  ctx->ibm_pos = (double *)(base + L.off_ibm_pos);
  ctx->ibm_vol = (double *)(base + L.off_ibm_vol);
  ctx->ibm_vel = (double *)(base + L.off_ibm_vel);
  ctx->ibm_coef = (double *)(base + L.off_ibm_coef);
  ctx->ibm_capacity = L.ibm_capacity;

  GksGrid &g = ctx->g;
  const int n[3] = {cfg->nx, cfg->ny, cfg->nz};
  const double *faces[3] = {cfg->xf, cfg->yf, cfg->zf};
  const double x0[3] = {cfg->x0, cfg->y0, cfg->z0}, dx[3] = {cfg->dx, cfg->dy, cfg->dz};
  for (int a = 0; a < 3; ++a) {
    g.n[a] = n[a];
    g.P[a] = L.P[a];
    g.uniform[a] = faces[a] == nullptr;
    g.x0[a] = x0[a];
    g.dx[a] = dx[a];
    g.inv_w_u[a] = 1.0 / dx[a];
    g.inv_12hn_u[a] = 1.0 / (12.0 * dx[a]);
    g.periodic[a] = cfg->bc[2 * a] == GKS_BC_PERIODIC;
    g.halo[2 * a] = cfg->bc[2 * a] == GKS_BC_HALO;
    g.halo[2 * a + 1] = cfg->bc[2 * a + 1] == GKS_BC_HALO;
  }
  /* On a periodic axis face n is face 0, cell for cell: the fused sweep stores n faces and readers wrap.
     (Holds next to a convective-outflow face of another axis too, since the ghost state of that axis is carried on
     this axis' ghost lines as the image of the interior lines' state, S20.) */
  for (int a = 0; a < 3; ++a) g.wrapf[a] = g.periodic[a];
  g.st[0] = 1;
  g.st[1] = g.P[0];
  g.st[2] = (long long)g.P[0] * g.P[1];
  g.FS = (long long)L.FS;

  std::vector<double> tab(L.coords_doubles, 0.0);
  size_t o = 0;
  double vol[3];
  ctx->dmin = 1e300;
  for (int a = 0; a < 3; ++a) {
    const size_t len = (size_t)n[a] + 8;
    double *xf = &tab[o], *xc = &tab[o + len], *w = &tab[o + 2 * len], *iw = &tab[o + 3 * len],
           *ihn = &tab[o + 4 * len];
    build_axis(n[a], faces[a], x0[a], dx[a], g.periodic[a], xf, xc, w);
    for (int i = 0; i < n[a] + 2 * GKS_NG; ++i) iw[i] = 1.0 / w[i];
    for (int i = 1; i < n[a] + 2 * GKS_NG; ++i) ihn[i] = 1.0 / (12.0 * (xc[i] - xc[i - 1]));
    g.xf[a] = ctx->coords + o;
    g.xc[a] = ctx->coords + o + len;
    g.w[a] = ctx->coords + o + 2 * len;
    g.inv_w[a] = ctx->coords + o + 3 * len;
    g.inv_12hn[a] = ctx->coords + o + 4 * len;
    ctx->h_xf[a] = (double *)malloc(3 * len * sizeof(double));
    ctx->h_xc[a] = ctx->h_xf[a] + len;
    ctx->h_w[a] = ctx->h_xf[a] + 2 * len;
    memcpy(ctx->h_xf[a], xf, 3 * len * sizeof(double));
    vol[a] = xf[GKS_NG + n[a]] - xf[GKS_NG];
    for (int i = 0; i < n[a]; ++i)
      if (w[GKS_NG + i] < ctx->dmin) ctx->dmin = w[GKS_NG + i];
    o += 5 * len;
  }
  ctx->total_volume = vol[0] * vol[1] * vol[2];

  GksPhys &ph = ctx->ph;
  ph.RT = cfg->RT;
  ph.lambda = 1.0 / (2.0 * cfg->RT);
  ph.mu = cfg->rho_ref * cfg->nu;
  ph.theta = sqrt(ph.lambda);
  ph.cx = 0.5 / sqrt(3.14159265358979323846 * ph.lambda);
  ph.weno_eps4 = 4.0 * (cfg->weno_eps > 0 ? cfg->weno_eps : 1e-6);
  for (int i = 0; i < 4; ++i) ph.inflow[i] = cfg->inflow[i];
  for (int i = 0; i < 6; ++i) ph.bc[i] = cfg->bc[i];

  cudaError_t e = cudaMemcpyAsync(ctx->coords, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice,
                                  ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) {
    set_err(nullptr, GKS_ERR_CUDA, "coordinate upload: %s", cudaGetErrorString(e));
    for (int a = 0; a < 3; ++a) free(ctx->h_xf[a]);
    delete ctx;
    return GKS_ERR_CUDA;
  }
  {
    /* interior / rim split of a sub-domain (gks_step_begin_part): the interior is what reads no HALO ghost.  Tiles of
       the y- and z-sweeps are 32 cells wide along x and stage cells a0-3 .. a0+33, tiles of the x-sweep hold 4 faces
       and stage cells a0-3 .. a0+5: on a HALO low side the interior starts at cell 32, on a HALO high side it ends at
       the largest multiple of 32 that leaves 6 cells to the face. */
    int ta[3];
    gks_fused_tiles_x(g, ta);
    const int nx = g.n[0], big = ta[1];
    int X0 = g.halo[0] ? big : 0;
    int X1 = g.halo[1] ? ((nx - 6) / big) * big : nx;
    if (X1 <= X0) X0 = X1 = 0;
    ctx->part_x0 = X0;
    ctx->part_x1 = X1;
    for (int d = 0; d < 3; ++d) {
      const int ext = nx + (d == 0 && !g.wrapf[0] ? 1 : 0), all = (ext + ta[d] - 1) / ta[d];
      ctx->part_t0[d] = X0 / ta[d];
      ctx->part_t1[d] = X1 <= X0 ? ctx->part_t0[d] : (g.halo[1] ? X1 / ta[d] + (d == 0 ? 1 : 0) : all);
    }
  }
  if (!gks_fused_init(ctx)) {
    set_err(nullptr, GKS_ERR_CUDA, "cuTensorMapEncodeTiled unavailable or failed (TMA descriptors of the fused sweep)");
    for (int a = 0; a < 3; ++a) free(ctx->h_xf[a]);
    delete ctx;
    return GKS_ERR_CUDA;
  }
  *out = ctx;
  return GKS_OK;
}

gks_status gks_destroy(gks_ctx *ctx) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  cudaStreamSynchronize(ctx->stream);
  gks_prof_free(ctx);
  for (int a = 0; a < 3; ++a) free(ctx->h_xf[a]);
  delete ctx;
  return GKS_OK;
}

} /* extern "C" */

/* the rest of the ABI (state transfer, step, forcing setters) is in gks_api_step.cu */
