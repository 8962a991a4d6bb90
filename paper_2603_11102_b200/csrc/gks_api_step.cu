/*
 * gks_api_step.cu — second half of the C ABI: state transfer, gks_step, forcing setters, test hooks.
 */
#include <cmath>
#include <cstring>
#include <vector>

#include "gks_internal.h"

#define CUDA_TRY(ctx, call)                                                                                  \
  do {                                                                                                       \
    cudaError_t e_ = (call);                                                                                 \
    if (e_ != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));   \
  } while (0)

namespace {

size_t interior_doubles(const gks_ctx *ctx) { return 4 * (size_t)ctx->g.n[0] * ctx->g.n[1] * ctx->g.n[2]; }

/* host copy of a small caller array that may live on the device */
gks_status fetch_host(gks_ctx *ctx, const double *src, size_t count, std::vector<double> &dst) {
  dst.resize(count);
  if (count == 0) return GKS_OK;
  if (gks_is_device_ptr(src)) {
    CUDA_TRY(ctx, cudaMemcpyAsync(dst.data(), src, count * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  } else {
    memcpy(dst.data(), src, count * sizeof(double));
  }
  return GKS_OK;
}

/* all sweeps of one stage into ctx->flux[]; part: 0 everything, 1 interior tiles, 2 rim tiles (gks_step_begin_part) */
void sweeps(gks_ctx *ctx, const double *W, bool need_F, int part = 0) {
  for (int d = 0; d < 3; ++d) {
    gks_prof_begin(ctx, GKS_PROF_SWEEP_X + d);
#ifdef GKS_DEBUG
    if (ctx->sweep_mode == 1)
      ctx->launches += gks_launch_sweep_unfused(ctx->g, ctx->ph, d, W, ctx->tmpN, ctx->tmpT, ctx->flux[d], need_F,
                                                ctx->stream);
    else
#endif
      ctx->launches += gks_launch_sweep_fused(ctx, d, W == ctx->Wn ? 0 : 1, ctx->flux[d], need_F, part);
    gks_prof_end(ctx);
  }
}

/* bounding box, in unwrapped cell indices, of the cells whose centre can lie within 3 eps of a point cloud
   spanning [pmin, pmax]; conservative by one cell, the kernel applies the exact cut */
gks_status alm_bbox(gks_ctx *ctx, const double pmin[3], const double pmax[3], double eps, int lo[3], int cnt[3]) {
  const double R = 3.0 * eps;
  for (int a = 0; a < 3; ++a) {
    const int nn = ctx->g.n[a];
    const double *xf = ctx->h_xf[a] + GKS_NG;
    const double L = xf[nn] - xf[0];
    if (!std::isfinite(pmin[a]) || !std::isfinite(pmax[a])) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "non-finite position");
    /* unwrapped index of the cell containing x (periodic: any x; else clamped to the domain) */
    auto cell_of = [&](double x) {
      long long m = 0;
      if (ctx->g.periodic[a]) {
        m = (long long)floor((x - xf[0]) / L);
        x -= m * L;
      }
      int c = gks_host_find_cell(ctx, a, x);
      if (c < 0) c = x < xf[0] ? 0 : nn - 1;
      return (long long)c + m * nn;
    };
    long long l = cell_of(pmin[a] - R) - 1, h = cell_of(pmax[a] + R) + 1;
    if (ctx->g.periodic[a]) {
      if (2.0 * R >= L) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "alm: 6 eps must be smaller than a periodic axis");
      if (h - l + 1 > nn) { /* the whole axis: k_alm takes the nearest image of every point along it */
        l = 0;
        h = nn - 1;
      }
    } else {
      if (l < 0) l = 0;
      if (h > nn - 1) h = nn - 1;
    }
    if (h < l) h = l;
    lo[a] = (int)l;
    cnt[a] = (int)(h - l + 1);
  }
  return GKS_OK;
}

} /* namespace */

extern "C" {

gks_status gks_set_state(gks_ctx *ctx, const double *W) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!W) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "W is NULL");
  if (gks_status st = gks_check_device(ctx)) return st;
  if (ctx->mid_step) return gks_set_err(ctx, GKS_ERR_STATE, "gks_set_state inside an unfinished step (between gks_step_begin and gks_step_force)");
  const double *src = W;
  if (!gks_is_device_ptr(W)) { /* host: stage through the flux buffer of the x-sweep (idle between the kernels of a step) */
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->flux[0], W, interior_doubles(ctx) * sizeof(double), cudaMemcpyHostToDevice,
                                  ctx->stream));
    src = ctx->flux[0];
  }
  ctx->launches += gks_launch_pack(ctx->g, src, ctx->Wn, ctx->stream);
  ctx->launches += gks_launch_outflow_init(ctx->g, ctx->ph, ctx->Wn, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  ctx->have_state = true;
  return GKS_OK;
}

gks_status gks_get_state(gks_ctx *ctx, double *W) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!W) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "W is NULL");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "gks_get_state before gks_set_state");
  if (gks_status st = gks_check_device(ctx)) return st;
  if (gks_is_device_ptr(W)) {
    ctx->launches += gks_launch_unpack(ctx->g, ctx->Wn, W, ctx->stream);
    CUDA_TRY(ctx, cudaGetLastError());
  } else {
    /* staged through the flux buffer of the x-sweep: free whenever no kernel of a step is in flight ahead of this
       call on the stream - also inside a split step, where Pbuf holds the predictor P (the state read is then W^n
       after gks_step_begin, the un-forced W^{n+1} after gks_step_finish) */
    double *stage = ctx->flux[0];
    ctx->launches += gks_launch_unpack(ctx->g, ctx->Wn, stage, ctx->stream);
    CUDA_TRY(ctx, cudaGetLastError());
    CUDA_TRY(ctx, cudaMemcpyAsync(W, stage, interior_doubles(ctx) * sizeof(double), cudaMemcpyDeviceToHost,
                                  ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  }
  return GKS_OK;
}

namespace {
gks_status step_begin_impl(gks_ctx *ctx, double dt, const GksPush *push);
}

gks_status gks_step_begin(gks_ctx *ctx, double dt) { return step_begin_impl(ctx, dt, nullptr); }

gks_status gks_step_begin_push(gks_ctx *ctx, double dt, const gks_halo_window *to_lo, const gks_halo_window *to_hi) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  GksPush push;
  memset(&push, 0, sizeof(push));
  const gks_halo_window *to[2] = {to_lo, to_hi};
  for (int f = 0; f < 2; ++f) {
    if (!to[f]) continue;
    if (!to[f]->W) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "the neighbour's window is NULL");
    if (ctx->ph.bc[f] != GKS_BC_HALO) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "face %d is not a GKS_BC_HALO x face", f);
    if (to[f]->ny != ctx->g.n[1] || to[f]->nz != ctx->g.n[2] || to[f]->nx < 6 || to[f]->pitch_x < to[f]->nx + 2 * GKS_NG ||
        to[f]->pitch_y != to[f]->ny + 2 * GKS_NG)
      return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "the neighbour's window does not match this sub-domain's y, z extents");
    push.W[f] = to[f]->W;
    push.nx[f] = to[f]->nx;
    push.PX[f] = to[f]->pitch_x;
    push.PY[f] = to[f]->pitch_y;
    push.FS[f] = to[f]->field_stride;
  }
  return step_begin_impl(ctx, dt, &push);
}

namespace {
gks_status step_begin_impl(gks_ctx *ctx, double dt, const GksPush *push) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "gks_step before gks_set_state");
  if (!(dt > 0) || !std::isfinite(dt)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "dt must be > 0");
  if (ctx->mid_step) return gks_set_err(ctx, GKS_ERR_STATE, "gks_step_begin inside an unfinished step");
  if (gks_status st = gks_check_device(ctx)) return st;
  ctx->step_dt = dt;
  GksPdlScope pdl(!ctx->prof_on);
  const GksGrid &g = ctx->g;
  const GksPhys &ph = ctx->ph;
  cudaStream_t s = ctx->stream;
  /* stage 1: ghosts of W^n, F and dF/dt of the three sweeps, W* and P */
  gks_prof_begin(ctx, GKS_PROF_GHOST);
  ctx->launches += gks_launch_ghost_fill(g, ph, ctx->Wn, ctx->Wn, s);
  gks_prof_end(ctx);
  sweeps(ctx, ctx->Wn, true);
  gks_prof_begin(ctx, GKS_PROF_UPDATE);
  ctx->launches += gks_launch_stage1(g, ctx->Wn, ctx->flux, dt, ctx->Ws, ctx->Pbuf, s, 0, -1, push);
  gks_prof_end(ctx);
  CUDA_TRY(ctx, cudaGetLastError());
  ctx->mid_step = 1;
  return GKS_OK;
}
} /* namespace */

gks_status gks_step_finish(gks_ctx *ctx, double dt) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (ctx->mid_step != 1) return gks_set_err(ctx, GKS_ERR_STATE, "gks_step_finish without gks_step_begin");
  if (!(dt > 0) || !std::isfinite(dt)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "dt must be > 0");
  if (dt != ctx->step_dt) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "gks_step_finish: dt = %.17g differs from the dt = %.17g of gks_step_begin", dt, ctx->step_dt);
  if (gks_status st = gks_check_device(ctx)) return st;
  GksPdlScope pdl(!ctx->prof_on);
  const GksGrid &g = ctx->g;
  const GksPhys &ph = ctx->ph;
  cudaStream_t s = ctx->stream;
  /* stage 2: ghosts of W* (outflow ghost state taken from W^n, S20), dF/dt only, W^{n+1} in place of W^n */
  gks_prof_begin(ctx, GKS_PROF_GHOST);
  ctx->launches += gks_launch_ghost_fill(g, ph, ctx->Ws, ctx->Wn, s);
  gks_prof_end(ctx);
  sweeps(ctx, ctx->Ws, false);
  gks_prof_begin(ctx, GKS_PROF_UPDATE);
  ctx->launches += gks_launch_stage2(g, ctx->Pbuf, ctx->flux, dt, ctx->Wn, s);
  gks_prof_end(ctx);
  CUDA_TRY(ctx, cudaGetLastError());
  ctx->mid_step = 2;
  return GKS_OK;
}

gks_status gks_step_force(gks_ctx *ctx, double dt) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (ctx->mid_step != 2) return gks_set_err(ctx, GKS_ERR_STATE, "gks_step_force without gks_step_finish");
  if (!(dt > 0) || !std::isfinite(dt)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "dt must be > 0");
  if (dt != ctx->step_dt) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "gks_step_force: dt = %.17g differs from the dt = %.17g of gks_step_begin", dt, ctx->step_dt);
  if (gks_status st = gks_check_device(ctx)) return st;
  GksPdlScope pdl(!ctx->prof_on);
  const GksGrid &g = ctx->g;
  const GksPhys &ph = ctx->ph;
  cudaStream_t s = ctx->stream;
  bool any_halo = false;
  for (int f = 0; f < 6; ++f) any_halo = any_halo || g.halo[f];
  if (any_halo && ctx->n_ibm > 0 && ctx->ibm_maxit > 1 && !ctx->ibm_external)
    return gks_set_err(ctx, GKS_ERR_STATE, "IBM passes > 1 on a sub-domain need an exchange per pass: drive them with gks_ibm_pass");
  if (any_halo && ctx->bulk_axis >= 0 && !ctx->bulk_external)
    return gks_set_err(ctx, GKS_ERR_STATE, "bulk-flux forcing on a sub-domain: gks_bulk_set_global must supply the global sum first");
  if (any_halo && ctx->rotor_on && !ctx->rotor_external)
    return gks_set_err(ctx, GKS_ERR_STATE, "the on-line rotor samples across cuts: on a sub-domain this step's points must be supplied with alm_rotor_supply");
  ctx->mid_step = 0;
  gks_prof_begin(ctx, GKS_PROF_FORCING);
  /* forcing (Eq. 13), every increment from the un-forced field: read-only kernels first */
  const bool uniform = ctx->gacc[0] != 0.0 || ctx->gacc[1] != 0.0 || ctx->gacc[2] != 0.0;
  if (ctx->rotor_on) { /* ALM front half on the un-forced field at the rotor clock t^n (S12, S26) */
    if (!ctx->rotor_external)                     /* sub-domain: evaluated by the slab that holds the disc and supplied */
      ctx->launches += gks_launch_rotor_forces(g, ctx->Wn, ctx->rotor, ctx->rotor_time, ctx->alm_eps, ctx->alm_pos,
                                               ctx->alm_force, s);
    ctx->rotor_external = 0;
    ctx->n_alm = ctx->rotor.nb * ctx->rotor.np;
    ctx->rotor_time += dt;
  }
  const bool ext = ctx->bulk_external != 0;       /* sub-domain: the global sum is already in place */
  ctx->bulk_external = 0;
  if (ctx->bulk_axis >= 0 && !ext) ctx->launches += gks_launch_bulk_reduce(g, ctx->Wn, ctx->bulk_axis, ctx->red, s);
  const bool ibm_done = ctx->ibm_external != 0;   /* sub-domain: the passes were driven with gks_ibm_pass */
  ctx->ibm_external = 0;
  if (ctx->n_ibm > 0 && !ibm_done) {
    /* multi-direct-forcing passes (Eq. 11-12): pass k interpolates from the un-forced field plus the IBM
       increments of the passes before it, in place; nothing else has touched the momentum yet (S12) */
    unsigned long long *res = reinterpret_cast<unsigned long long *>(ctx->red + GKS_RED_IBM_RES);
    if (ctx->ibm_maxit > 1) {
      CUDA_TRY(ctx, cudaMemsetAsync(res, 0, GKS_IBM_MAX_PASSES * sizeof(unsigned long long), s));
      gks_pdl_break();                /* the next kernel must not overtake the memset */
    }
    for (int pass = 0; pass < ctx->ibm_maxit; ++pass) {
      ctx->launches += gks_launch_ibm_interp(g, ctx->Wn, ctx->n_ibm, ctx->ibm_pos, ctx->ibm_vol, ctx->ibm_vel,
                                             ctx->ibm_coef, pass, ctx->ibm_tol, res, s);
      ctx->launches += gks_launch_ibm_spread(g, ctx->Wn, ctx->n_ibm, ctx->ibm_pos, ctx->ibm_coef, pass, ctx->ibm_tol,
                                             res, s);
    }
  }
  if (uniform || ctx->bulk_axis >= 0)
    ctx->launches += gks_launch_uniform_force(g, ctx->Wn, dt, ctx->gacc, ctx->bulk_axis, ctx->bulk_target,
                                              ext ? ctx->bulk_volume_ext : ctx->total_volume, ctx->red, s);
  if (ctx->n_alm > 0)
    ctx->launches += gks_launch_alm(g, ctx->Wn, ctx->n_alm, ctx->alm_pos, ctx->alm_force, ctx->alm_eps, dt,
                                    ctx->alm_lo, ctx->alm_cnt, s);
  ctx->launches += gks_launch_outflow_advance(g, ph, ctx->Wn, dt, s);
  gks_prof_end(ctx);
  CUDA_TRY(ctx, cudaGetLastError());
  return GKS_OK;
}

gks_status gks_step(gks_ctx *ctx, double dt) {
  if (gks_status st = gks_step_begin(ctx, dt)) return st;
  if (gks_status st = gks_step_finish(ctx, dt)) return st;
  return gks_step_force(ctx, dt);
}

/* one stage in two parts (include/gks.h): part 0 = everything that reads no HALO ghost, part 1 = the rest */
namespace {
gks_status stage_part(gks_ctx *ctx, double dt, int stage, int part) {
  const GksGrid &g = ctx->g;
  const GksPhys &ph = ctx->ph;
  cudaStream_t s = ctx->stream;
  double *W = stage == 1 ? ctx->Wn : ctx->Ws;
  GksPdlScope pdl(!ctx->prof_on);
  gks_prof_begin(ctx, GKS_PROF_GHOST);
  if (part == 0) ctx->launches += gks_launch_ghost_fill(g, ph, W, ctx->Wn, s);
  else ctx->launches += gks_launch_ghost_fill_xcols(g, ph, W, ctx->Wn, s);
  gks_prof_end(ctx);
  const bool split = ctx->part_x1 > ctx->part_x0;      /* no interior: part 1 does everything */
  if (part == 1 || split) {
    sweeps(ctx, W, stage == 1, part == 0 ? 1 : 2);
    gks_prof_begin(ctx, GKS_PROF_UPDATE);
    const int nx = g.n[0], X0 = ctx->part_x0, X1 = ctx->part_x1;
    const int lo[2] = {part == 0 ? X0 : 0, part == 0 ? 0 : X1}, hi[2] = {part == 0 ? X1 : X0, part == 0 ? 0 : nx};
    for (int r = 0; r < 2; ++r) {
      if (hi[r] <= lo[r]) continue;
      if (stage == 1) ctx->launches += gks_launch_stage1(g, ctx->Wn, ctx->flux, dt, ctx->Ws, ctx->Pbuf, s, lo[r], hi[r]);
      else ctx->launches += gks_launch_stage2(g, ctx->Pbuf, ctx->flux, dt, ctx->Wn, s, lo[r], hi[r]);
    }
    gks_prof_end(ctx);
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "stage %d part %d: %s", stage, part, cudaGetErrorString(e));
  return GKS_OK;
}
} /* namespace */

gks_status gks_step_begin_part(gks_ctx *ctx, double dt, int part) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (part != 0 && part != 1) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "part must be 0 (interior) or 1 (rim)");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "gks_step before gks_set_state");
  if (!(dt > 0) || !std::isfinite(dt)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "dt must be > 0");
  if (ctx->mid_step != (part == 0 ? 0 : 10))
    return gks_set_err(ctx, GKS_ERR_STATE, "gks_step_begin_part(%d): wrong place in the step (state %d)", part, ctx->mid_step);
  if (part == 1 && dt != ctx->step_dt) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "gks_step_begin_part: dt differs from part 0's");
  if (ctx->sweep_mode != 0) return gks_set_err(ctx, GKS_ERR_STATE, "the split step runs the fused sweep only");
  if (gks_status st = gks_check_device(ctx)) return st;
  if (part == 0) ctx->step_dt = dt;
  if (gks_status st = stage_part(ctx, dt, 1, part)) return st;
  ctx->mid_step = part == 0 ? 10 : 1;
  return GKS_OK;
}

gks_status gks_step_finish_part(gks_ctx *ctx, double dt, int part) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (part != 0 && part != 1) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "part must be 0 (interior) or 1 (rim)");
  if (ctx->mid_step != (part == 0 ? 1 : 11))
    return gks_set_err(ctx, GKS_ERR_STATE, "gks_step_finish_part(%d): wrong place in the step (state %d)", part, ctx->mid_step);
  if (!(dt > 0) || !std::isfinite(dt) || dt != ctx->step_dt)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "gks_step_finish_part: dt must be the dt of gks_step_begin");
  if (ctx->sweep_mode != 0) return gks_set_err(ctx, GKS_ERR_STATE, "the split step runs the fused sweep only");
  if (gks_status st = gks_check_device(ctx)) return st;
  if (gks_status st = stage_part(ctx, dt, 2, part)) return st;
  ctx->mid_step = part == 0 ? 11 : 2;
  return GKS_OK;
}

size_t gks_halo_doubles(const gks_ctx *ctx, int face) {
  if (!ctx || face < 0 || face > 5) return 0;
  const int ax = face >> 1, ua = ax == 0 ? 1 : 0, va = ax == 2 ? 1 : 2;
  return (size_t)4 * GKS_NG * ctx->g.n[ua] * ctx->g.n[va];
}

namespace {
gks_status halo_move(gks_ctx *ctx, int which, int face, double *buf, int unpack) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!buf) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "buf is NULL");
  if (face < 0 || face > 5 || ctx->ph.bc[face] != GKS_BC_HALO)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "face %d is not a GKS_BC_HALO face", face);
  if (which != 0 && which != 1) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "which must be 0 (W^n) or 1 (W*)");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "no state set");
  if (which == 1 && ctx->mid_step != 1 && ctx->mid_step != 11)
    return gks_set_err(ctx, GKS_ERR_STATE, "W* exists only between gks_step_begin and gks_step_finish");
  if (which == 0 && ctx->mid_step == 11)
    return gks_set_err(ctx, GKS_ERR_STATE, "between the two parts of gks_step_finish the buffer of W^n is half W^{n+1}");
  double *W = which == 0 ? ctx->Wn : ctx->Ws;
  const size_t bytes = gks_halo_doubles(ctx, face) * sizeof(double);
  if (gks_is_device_ptr(buf)) {
    ctx->launches += gks_launch_halo(ctx->g, W, buf, face, unpack, ctx->stream);
  } else { /* host buffer: stage through the flux buffer of the y-sweep (idle at every point a halo may move) */
    double *stage = ctx->flux[1];
    if (unpack) CUDA_TRY(ctx, cudaMemcpyAsync(stage, buf, bytes, cudaMemcpyHostToDevice, ctx->stream));
    ctx->launches += gks_launch_halo(ctx->g, W, stage, face, unpack, ctx->stream);
    if (!unpack) CUDA_TRY(ctx, cudaMemcpyAsync(buf, stage, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  }
  CUDA_TRY(ctx, cudaGetLastError());
  return GKS_OK;
}
} /* namespace */

gks_status gks_halo_pack(gks_ctx *ctx, int which, int face, double *buf) { return halo_move(ctx, which, face, buf, 0); }
gks_status gks_halo_unpack(gks_ctx *ctx, int which, int face, const double *buf) {
  return halo_move(ctx, which, face, const_cast<double *>(buf), 1);
}

gks_status gks_halo_window_get(gks_ctx *ctx, int which, gks_halo_window *out) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!out || (which != 0 && which != 1)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "out is NULL or which is not 0 / 1");
  out->W = which == 0 ? ctx->Wn : ctx->Ws;
  out->nx = ctx->g.n[0];
  out->ny = ctx->g.n[1];
  out->nz = ctx->g.n[2];
  out->pitch_x = ctx->g.P[0];
  out->pitch_y = ctx->g.P[1];
  out->field_stride = ctx->g.FS;
  return GKS_OK;
}

gks_status gks_halo_push(gks_ctx *ctx, int which, int face, const gks_halo_window *to) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!to || !to->W) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "the neighbour's window is NULL");
  if ((face != 0 && face != 1) || ctx->ph.bc[face] != GKS_BC_HALO)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "face %d is not a GKS_BC_HALO x face", face);
  if (which != 0 && which != 1) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "which must be 0 (W^n) or 1 (W*)");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "no state set");
  if (which == 1 && ctx->mid_step != 1 && ctx->mid_step != 11)
    return gks_set_err(ctx, GKS_ERR_STATE, "W* exists only between gks_step_begin and gks_step_finish");
  if (which == 0 && ctx->mid_step == 11)
    return gks_set_err(ctx, GKS_ERR_STATE, "between the two parts of gks_step_finish the buffer of W^n is half W^{n+1}");
  if (to->ny != ctx->g.n[1] || to->nz != ctx->g.n[2] || to->nx < 6 || to->pitch_x < to->nx + 2 * GKS_NG ||
      to->pitch_y != to->ny + 2 * GKS_NG)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "the neighbour's window does not match this sub-domain's y, z extents");
  if (gks_status st = gks_check_device(ctx)) return st;
  ctx->launches += gks_launch_halo_push(ctx->g, which == 0 ? ctx->Wn : ctx->Ws, face, to->W, to->nx, to->pitch_x,
                                        to->pitch_y, to->field_stride, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  return GKS_OK;
}

gks_status gks_set_body_force(gks_ctx *ctx, double gx, double gy, double gz) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!std::isfinite(gx) || !std::isfinite(gy) || !std::isfinite(gz))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "acceleration must be finite");
  ctx->gacc[0] = gx;
  ctx->gacc[1] = gy;
  ctx->gacc[2] = gz;
  return GKS_OK;
}

gks_status gks_set_bulk_flux(gks_ctx *ctx, int axis, double target) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (axis > 2) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "axis must be 0, 1, 2 or negative");

  ctx->bulk_axis = axis < 0 ? -1 : axis;
  ctx->bulk_target = target;
  return GKS_OK;
}

gks_status gks_ibm_pass(gks_ctx *ctx, int pass, int phase) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (pass < 0 || pass >= ctx->ibm_maxit || (phase != 0 && phase != 1))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "pass must be in [0, max_iter) and phase 0 (interpolate) or 1 (spread)");
  if (ctx->mid_step != 2) return gks_set_err(ctx, GKS_ERR_STATE, "gks_ibm_pass belongs between gks_step_finish and gks_step_force");
  unsigned long long *res = reinterpret_cast<unsigned long long *>(ctx->red + GKS_RED_IBM_RES);
  if (pass == 0 && phase == 0)
    CUDA_TRY(ctx, cudaMemsetAsync(res, 0, GKS_IBM_MAX_PASSES * sizeof(unsigned long long), ctx->stream));
  ctx->ibm_external = 1;
  if (ctx->n_ibm > 0) {
    if (phase == 0)
      ctx->launches += gks_launch_ibm_interp(ctx->g, ctx->Wn, ctx->n_ibm, ctx->ibm_pos, ctx->ibm_vol, ctx->ibm_vel,
                                             ctx->ibm_coef, pass, ctx->ibm_tol, res, ctx->stream);
    else
      ctx->launches += gks_launch_ibm_spread(ctx->g, ctx->Wn, ctx->n_ibm, ctx->ibm_pos, ctx->ibm_coef, pass, ctx->ibm_tol,
                                             res, ctx->stream);
    CUDA_TRY(ctx, cudaGetLastError());
  }
  return GKS_OK;
}

gks_status gks_ibm_residual(gks_ctx *ctx, int pass, double *value, int set) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!value || pass < 0 || pass >= GKS_IBM_MAX_PASSES) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "value is NULL or pass out of range");
  double *slot = ctx->red + GKS_RED_IBM_RES + pass;   /* a non-negative double (its bit pattern orders like an integer) */
  const bool dev = gks_is_device_ptr(value);
  if (set) CUDA_TRY(ctx, cudaMemcpyAsync(slot, value, sizeof(double), dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
  else CUDA_TRY(ctx, cudaMemcpyAsync(value, slot, sizeof(double), dev ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
  if (!dev) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  return GKS_OK;
}

gks_status gks_bulk_partial(gks_ctx *ctx, double *sum, double *volume) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!sum) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "sum is NULL");
  if (ctx->bulk_axis < 0) return gks_set_err(ctx, GKS_ERR_STATE, "no bulk-flux forcing set");
  if (ctx->mid_step != 2) return gks_set_err(ctx, GKS_ERR_STATE, "gks_bulk_partial belongs between gks_step_finish and gks_step_force");
  ctx->launches += gks_launch_bulk_reduce(ctx->g, ctx->Wn, ctx->bulk_axis, ctx->red, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  if (volume) *volume = ctx->total_volume;
  if (gks_is_device_ptr(sum)) {
    CUDA_TRY(ctx, cudaMemcpyAsync(sum, ctx->red + GKS_RED_BULK_SUM, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
  } else {
    CUDA_TRY(ctx, cudaMemcpyAsync(sum, ctx->red + GKS_RED_BULK_SUM, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  }
  return GKS_OK;
}

gks_status gks_bulk_set_global(gks_ctx *ctx, const double *sum, double volume) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!sum || !(volume > 0) || !std::isfinite(volume)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "sum is NULL or volume is not > 0");
  if (ctx->bulk_axis < 0) return gks_set_err(ctx, GKS_ERR_STATE, "no bulk-flux forcing set");
  if (ctx->mid_step != 2) return gks_set_err(ctx, GKS_ERR_STATE, "gks_bulk_set_global belongs between gks_step_finish and gks_step_force");
  const cudaMemcpyKind k = gks_is_device_ptr(sum) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->red + GKS_RED_BULK_SUM, sum, sizeof(double), k, ctx->stream));
  if (k == cudaMemcpyHostToDevice) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  ctx->bulk_external = 1;
  ctx->bulk_volume_ext = volume;
  return GKS_OK;
}

gks_status alm_set_points(gks_ctx *ctx, int n, const double *pos, const double *force, double eps) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (n < 0 || n > GKS_MAX_ALM_POINTS) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "n out of range");
  ctx->rotor_on = 0;   /* prescribed points replace an on-line rotor */
  ctx->rotor_external = 0;
  if (n == 0) {
    ctx->n_alm = 0;
    return GKS_OK;
  }
  if (!pos || !force) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "pos/force is NULL");
  if (!(eps > 0) || !std::isfinite(eps)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "eps must be > 0");
  std::vector<double> hp;
  if (gks_status st = fetch_host(ctx, pos, 3 * (size_t)n, hp)) return st;
  double pmin[3], pmax[3];
  for (int a = 0; a < 3; ++a) {
    pmin[a] = pmax[a] = hp[a];
    for (int p = 1; p < n; ++p) {
      pmin[a] = fmin(pmin[a], hp[3 * p + a]);
      pmax[a] = fmax(pmax[a], hp[3 * p + a]);
    }
  }
  int lo[3], cnt[3];
  if (gks_status st = alm_bbox(ctx, pmin, pmax, eps, lo, cnt)) return st;
  const cudaMemcpyKind kind = gks_is_device_ptr(pos) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  const cudaMemcpyKind kindf = gks_is_device_ptr(force) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->alm_pos, pos, 3 * (size_t)n * sizeof(double), kind, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->alm_force, force, 3 * (size_t)n * sizeof(double), kindf, ctx->stream));
  if (kind == cudaMemcpyHostToDevice || kindf == cudaMemcpyHostToDevice)
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream)); /* caller may reuse its arrays at once */
  for (int a = 0; a < 3; ++a) {
    ctx->alm_lo[a] = lo[a];
    ctx->alm_cnt[a] = cnt[a];
  }
  ctx->n_alm = n;
  ctx->alm_eps = eps;
  return GKS_OK;
}

namespace {
/* validate a rotor description, copy its tables to the device and fill the kernel's view of it */
gks_status upload_rotor(gks_ctx *ctx, const alm_rotor *r, GksRotor &R) {
  const int ns = r->nsections > 1 ? r->nsections : 1;
  if (r->nblades < 1 || r->npts < 1 || r->npts > GKS_MAX_ROTOR_STATIONS || r->npolar < 2 || r->npolar > GKS_MAX_POLAR ||
      (long long)r->nblades * r->npts > GKS_MAX_ALM_POINTS || ns > GKS_MAX_SECTIONS ||
      (long long)ns * r->npolar > 4 * GKS_MAX_POLAR)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: sizes out of range");
  if (!r->chord || !r->twist || !r->alpha || !r->cl || !r->cd) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: NULL table");
  if (!(r->R > r->r_hub) || !(r->r_hub >= 0) || !(r->eps > 0) || !std::isfinite(r->R) || !std::isfinite(r->eps) ||
      !std::isfinite(r->omega) || !std::isfinite(r->theta0))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: need R > r_hub >= 0, eps > 0 and finite parameters");
  if (r->tip_correction && !(r->u_ref > 0))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: the tip correction needs u_ref > 0 (tip speed ratio)");
  if ((r->radius == nullptr) != (r->width == nullptr))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: radius and width come together");
  if (ns > 1 && !r->section_r) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: section radii missing");
  /* tables on the host: chord, twist, radius, width, alpha, cl, cd, section radii */
  enum { CHORD, TWIST, RADIUS, WIDTH, ALPHA, CL, CD, SECR, NT };
  std::vector<double> t[NT];
  const double *src[NT] = {r->chord, r->twist, r->radius, r->width, r->alpha, r->cl, r->cd, ns > 1 ? r->section_r : nullptr};
  const size_t cnt[NT] = {(size_t)r->npts, (size_t)r->npts, (size_t)r->npts, (size_t)r->npts, (size_t)r->npolar,
                          (size_t)ns * r->npolar, (size_t)ns * r->npolar, ns > 1 ? (size_t)ns : 0};
  for (int q = 0; q < NT; ++q)
    if (src[q])
      if (gks_status st = fetch_host(ctx, src[q], cnt[q], t[q])) return st;
  if (!r->radius) { /* the default stations: r_hub + (k + 1/2) w, w = (R - r_hub) / npts */
    const double w = (r->R - r->r_hub) / r->npts;
    t[RADIUS].resize(r->npts);
    t[WIDTH].assign(r->npts, w);
    for (int k = 0; k < r->npts; ++k) t[RADIUS][k] = r->r_hub + (k + 0.5) * w;
  }
  for (int k = 0; k < r->npts; ++k)
    if (!(t[RADIUS][k] > 0) || !(t[RADIUS][k] <= r->R) || !(t[WIDTH][k] > 0))
      return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: need 0 < radius <= R and width > 0 at every station");
  for (int m = 1; m < r->npolar; ++m)
    if (!(t[ALPHA][m] > t[ALPHA][m - 1])) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: polar angles must increase");
  for (int m = 1; m < ns; ++m)
    if (!(t[SECR][m] > t[SECR][m - 1])) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: section radii must increase");
  const size_t S = GKS_MAX_ROTOR_STATIONS, P = GKS_MAX_POLAR;
  const size_t off[NT] = {0, S, 2 * S, 3 * S, 4 * S, 4 * S + P, 4 * S + 5 * P, 4 * S + 9 * P};
  for (int q = 0; q < NT; ++q)
    if (!t[q].empty())
      CUDA_TRY(ctx, cudaMemcpyAsync(ctx->rotor_tab + off[q], t[q].data(), t[q].size() * sizeof(double),
                                    cudaMemcpyHostToDevice, ctx->stream));
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));   /* the staging vectors go out of scope */
  R.nb = r->nblades; R.np = r->npts; R.npolar = r->npolar; R.nsec = ns;
  R.fs_corr = r->freestream_correction != 0; R.tip_corr = r->tip_correction != 0;
  for (int a = 0; a < 3; ++a) R.hub[a] = r->hub[a];
  R.R = r->R; R.rhub = r->r_hub; R.omega = r->omega; R.theta0 = r->theta0; R.uref = r->u_ref;
  R.chord = ctx->rotor_tab + off[CHORD]; R.twist = ctx->rotor_tab + off[TWIST];
  R.radius = ctx->rotor_tab + off[RADIUS]; R.width = ctx->rotor_tab + off[WIDTH];
  R.alpha = ctx->rotor_tab + off[ALPHA]; R.cl = ctx->rotor_tab + off[CL]; R.cd = ctx->rotor_tab + off[CD];
  R.sec_r = ctx->rotor_tab + off[SECR];
  return GKS_OK;
}
} /* namespace */

gks_status alm_set_rotor(gks_ctx *ctx, const alm_rotor *r) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!r) {
    ctx->rotor_on = 0;
    ctx->n_alm = 0;
    return GKS_OK;
  }
  /* the blades sweep the disc of radius R about the hub in the plane x = hub[0]: its bounding box is constant */
  const double pmin[3] = {r->hub[0], r->hub[1] - r->R, r->hub[2] - r->R};
  const double pmax[3] = {r->hub[0], r->hub[1] + r->R, r->hub[2] + r->R};
  int lo[3], cnt[3];
  if (!(r->eps > 0) || !std::isfinite(r->R)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor: need eps > 0 and a finite R");
  if (gks_status st = alm_bbox(ctx, pmin, pmax, r->eps, lo, cnt)) return st;
  GksRotor R;
  if (gks_status st = upload_rotor(ctx, r, R)) return st;
  ctx->rotor = R;
  for (int a = 0; a < 3; ++a) {
    ctx->alm_lo[a] = lo[a];
    ctx->alm_cnt[a] = cnt[a];
  }
  ctx->alm_eps = r->eps;
  ctx->n_alm = 0;
  ctx->rotor_on = 1;
  ctx->rotor_external = 0;
  ctx->rotor_time = 0.0;
  return GKS_OK;
}

gks_status alm_rotor_supply(gks_ctx *ctx, const double *pos, const double *force, double x_shift) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!pos || !force || !std::isfinite(x_shift)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "pos/force is NULL or x_shift is not finite");
  if (!ctx->rotor_on) return gks_set_err(ctx, GKS_ERR_STATE, "no rotor set");
  if (ctx->mid_step != 2) return gks_set_err(ctx, GKS_ERR_STATE, "alm_rotor_supply belongs between gks_step_finish and gks_step_force");
  /* the gather box of the disc as this sub-domain meets it (beyond the seam of a periodic x axis: its image) */
  const GksRotor &R = ctx->rotor;
  const double pmin[3] = {R.hub[0] + x_shift, R.hub[1] - R.R, R.hub[2] - R.R};
  const double pmax[3] = {R.hub[0] + x_shift, R.hub[1] + R.R, R.hub[2] + R.R};
  int lo[3], cnt[3];
  if (gks_status st = alm_bbox(ctx, pmin, pmax, ctx->alm_eps, lo, cnt)) return st;
  const size_t bytes = 3 * (size_t)R.nb * R.np * sizeof(double);
  const cudaMemcpyKind kp = gks_is_device_ptr(pos) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  const cudaMemcpyKind kf = gks_is_device_ptr(force) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->alm_pos, pos, bytes, kp, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->alm_force, force, bytes, kf, ctx->stream));
  if (x_shift != 0.0) ctx->launches += gks_launch_shift_x(ctx->alm_pos, R.nb * R.np, x_shift, ctx->stream);
  if (kp == cudaMemcpyHostToDevice || kf == cudaMemcpyHostToDevice) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  CUDA_TRY(ctx, cudaGetLastError());
  for (int a = 0; a < 3; ++a) {
    ctx->alm_lo[a] = lo[a];
    ctx->alm_cnt[a] = cnt[a];
  }
  ctx->rotor_external = 1;
  return GKS_OK;
}

gks_status alm_rotor_points(gks_ctx *ctx, const alm_rotor *r, double t, double *pos, double *force) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!r || !pos || !force) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "rotor/pos/force is NULL");
  if (!std::isfinite(t)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "t must be finite");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "alm_rotor_points before gks_set_state");
  if (ctx->rotor_on) return gks_set_err(ctx, GKS_ERR_STATE, "a rotor is set with alm_set_rotor: clear it first");
  GksRotor R;
  if (gks_status st = upload_rotor(ctx, r, R)) return st;
  const size_t n3 = 3 * (size_t)R.nb * R.np;
  double *dp = gks_is_device_ptr(pos) ? pos : ctx->rotor_out, *df = gks_is_device_ptr(force) ? force : ctx->rotor_out + n3;
  ctx->launches += gks_launch_rotor_forces(ctx->g, ctx->Wn, R, t, r->eps, dp, df, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  if (dp != pos) CUDA_TRY(ctx, cudaMemcpyAsync(pos, dp, n3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  if (df != force) CUDA_TRY(ctx, cudaMemcpyAsync(force, df, n3 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  if (dp != pos || df != force) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  return GKS_OK;
}

gks_status alm_rotor_eval(gks_ctx *ctx, double *pos, double *force) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!pos || !force) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "pos/force is NULL");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "alm_rotor_eval before gks_set_state");
  if (!ctx->rotor_on) return gks_set_err(ctx, GKS_ERR_STATE, "no rotor set");
  const int n = ctx->rotor.nb * ctx->rotor.np;
  ctx->launches += gks_launch_rotor_forces(ctx->g, ctx->Wn, ctx->rotor, ctx->rotor_time, ctx->alm_eps, ctx->alm_pos,
                                           ctx->alm_force, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  const cudaMemcpyKind kp = gks_is_device_ptr(pos) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  const cudaMemcpyKind kf = gks_is_device_ptr(force) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  CUDA_TRY(ctx, cudaMemcpyAsync(pos, ctx->alm_pos, 3 * (size_t)n * sizeof(double), kp, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(force, ctx->alm_force, 3 * (size_t)n * sizeof(double), kf, ctx->stream));
  if (kp == cudaMemcpyDeviceToHost || kf == cudaMemcpyDeviceToHost) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  return GKS_OK;
}

gks_status ibm_set_points(gks_ctx *ctx, int n, const double *pos, const double *weights) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (n < 0 || n > ctx->ibm_capacity)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "n out of range (capacity of this context: %d)", ctx->ibm_capacity);
  if (n == 0) {
    ctx->n_ibm = 0;
    return GKS_OK;
  }
  if (!pos || !weights) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "pos/weights is NULL");
  std::vector<double> hp;
  if (gks_status st = fetch_host(ctx, pos, 3 * (size_t)n, hp)) return st;
  for (int p = 0; p < n; ++p)
    for (int a = 0; a < 3; ++a) {
      const int c0 = gks_host_find_cell(ctx, a, hp[3 * p + a]);
      if (c0 < 0) {
        /* a point of the neighbouring sub-domain, at most 2 cells beyond a HALO face (uniform axis): its
           support reaches cells owned here and reads the HALO ghosts */
        const double *xf = ctx->h_xf[a] + GKS_NG;
        const double x = hp[3 * p + a], h = ctx->g.dx[a];
        const int nn = ctx->g.n[a];
        if ((ctx->g.halo[2 * a] && x < xf[0] && x >= xf[0] - 2.0 * h) ||
            (ctx->g.halo[2 * a + 1] && x > xf[nn] && x <= xf[nn] + 2.0 * h))
          continue;
        return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "ibm: point %d lies outside the domain", p);
      }
      const double *w = ctx->h_w[a] + GKS_NG;
      if (fabs(w[c0 - 1] - w[c0]) > 1e-9 * w[c0] || fabs(w[c0 + 1] - w[c0]) > 1e-9 * w[c0])
        return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "ibm: grid not locally uniform over the support of point %d", p);
    }
  const cudaMemcpyKind kp = gks_is_device_ptr(pos) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  const cudaMemcpyKind kw = gks_is_device_ptr(weights) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->ibm_pos, pos, 3 * (size_t)n * sizeof(double), kp, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->ibm_vol, weights, (size_t)n * sizeof(double), kw, ctx->stream));
  CUDA_TRY(ctx, cudaMemsetAsync(ctx->ibm_vel, 0, 3 * (size_t)n * sizeof(double), ctx->stream));
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  ctx->n_ibm = n;
  return GKS_OK;
}

gks_status gks_set_reconstruction(gks_ctx *ctx, int tangential_linear) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (tangential_linear != 0 && tangential_linear != 1)
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "tangential_linear must be 0 or 1");
  ctx->ph.tang_linear = tangential_linear;
  return GKS_OK;
}

gks_status ibm_set_iterations(gks_ctx *ctx, int max_iter, double tol) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (max_iter < 1 || max_iter > GKS_IBM_MAX_PASSES || !(tol >= 0.0) || !std::isfinite(tol))
    return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "ibm: max_iter must be in 1..%d and tol finite and >= 0", GKS_IBM_MAX_PASSES);
  ctx->ibm_maxit = max_iter;
  ctx->ibm_tol = tol;
  return GKS_OK;
}

gks_status ibm_set_velocities(gks_ctx *ctx, const double *vel) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  const size_t bytes = 3 * (size_t)ctx->n_ibm * sizeof(double);
  if (bytes == 0) return GKS_OK;
  if (!vel) {
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->ibm_vel, 0, bytes, ctx->stream));
    return GKS_OK;
  }
  const cudaMemcpyKind k = gks_is_device_ptr(vel) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->ibm_vel, vel, bytes, k, ctx->stream));
  if (k == cudaMemcpyHostToDevice) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  return GKS_OK;
}

gks_status gks_debug_eval_flux(gks_ctx *ctx, int dir, double *F, double *dFdt) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (dir < 0 || dir > 2 || !F || !dFdt) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "bad dir or NULL output");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "gks_debug_eval_flux before gks_set_state");
  if (ctx->mid_step) return gks_set_err(ctx, GKS_ERR_STATE, "gks_debug_eval_flux inside an unfinished step (it refills ghosts and flux buffers)");
  if (gks_status st = gks_check_device(ctx)) return st;
  const GksGrid &g = ctx->g;
  ctx->launches += gks_launch_ghost_fill(g, ctx->ph, ctx->Wn, ctx->Wn, ctx->stream);
#ifdef GKS_DEBUG
  if (ctx->sweep_mode == 1)
    ctx->launches += gks_launch_sweep_unfused(g, ctx->ph, dir, ctx->Wn, ctx->tmpN, ctx->tmpT, ctx->flux[dir], true,
                                              ctx->stream);
  else
#endif
    ctx->launches += gks_launch_sweep_fused(ctx, dir, 0, ctx->flux[dir], true);
  const size_t nf = 4 * (size_t)(g.n[0] + (dir == 0)) * (g.n[1] + (dir == 1)) * (g.n[2] + (dir == 2));
  double *outs[2] = {F, dFdt};
  for (int h = 0; h < 2; ++h) {
    const double *src = ctx->flux[dir] + (size_t)h * 4 * g.FS;
    if (gks_is_device_ptr(outs[h])) {
      ctx->launches += gks_launch_unpack_faces(g, dir, src, outs[h], ctx->stream);
    } else {
      ctx->launches += gks_launch_unpack_faces(g, dir, src, ctx->Pbuf, ctx->stream);
      CUDA_TRY(ctx, cudaMemcpyAsync(outs[h], ctx->Pbuf, nf * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
      CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    }
  }
  CUDA_TRY(ctx, cudaGetLastError());
  return GKS_OK;
}

gks_status gks_cfl_dt(gks_ctx *ctx, double cfl, double *dt) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!dt) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "dt is NULL");
  if (!(cfl > 0) || !std::isfinite(cfl)) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "cfl must be > 0");
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "gks_cfl_dt before gks_set_state");
  double *scr = ctx->red + GKS_RED_CFL;
  CUDA_TRY(ctx, cudaMemsetAsync(scr, 0, 2 * sizeof(double), ctx->stream));
  ctx->launches += gks_launch_cfl_dt(ctx->g, ctx->Wn, cfl, ctx->dmin, sqrt(ctx->ph.RT), scr, ctx->stream);
  CUDA_TRY(ctx, cudaGetLastError());
  if (gks_is_device_ptr(dt)) {
    CUDA_TRY(ctx, cudaMemcpyAsync(dt, scr + 1, sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
  } else {
    CUDA_TRY(ctx, cudaMemcpyAsync(dt, scr + 1, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  }
  return GKS_OK;
}

#ifdef GKS_DEBUG
gks_status gks_debug_set_sweep(gks_ctx *ctx, int mode) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (mode != 0 && mode != 1) return gks_set_err(ctx, GKS_ERR_INVALID_ARG, "mode must be 0 or 1");
  if (ctx->mid_step) return gks_set_err(ctx, GKS_ERR_STATE, "gks_debug_set_sweep inside an unfinished step");
  ctx->sweep_mode = mode;
  return GKS_OK;
}
#endif

gks_status gks_check_finite(gks_ctx *ctx) {
  if (!ctx) return GKS_ERR_INVALID_ARG;
  if (!ctx->have_state) return gks_set_err(ctx, GKS_ERR_STATE, "no state set");
  int *flag = (int *)(ctx->red + 1536);
  int h = 0;
  CUDA_TRY(ctx, cudaMemsetAsync(flag, 0, sizeof(int), ctx->stream));
  ctx->launches += gks_launch_check_finite(ctx->g, ctx->Wn, flag, ctx->stream);
  CUDA_TRY(ctx, cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  if (h) return gks_set_err(ctx, GKS_ERR_NONFINITE, "state holds a NaN or Inf");
  return GKS_OK;
}

} /* extern "C" */
