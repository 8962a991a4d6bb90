/*
 * gks_ghost.cu — ghost-cell fill for the six boundary kinds (formulas
 * DESIGN.md S17-S21), convective-outflow ghost state (S20), pack/unpack between the C-ABI interior
 * layout and the padded HBM layout.
 *
 * Pass order x, y, z; pass y also covers the i-ghosts, pass z covers i- and j-ghosts, so edges and
 * corners are defined.  One thread fills the 3 ghosts x 4 components of one line end.
 * The convective-outflow ghosts of an axis are state on EVERY line its pass covers (also the lines through
 * the ghosts of the lower axes): initialised and advanced per axis, with the passes of the lower axes run in
 * between, so that a periodic / mirrored tangential ghost line carries the image of the ghost state.
 */
#include <cstdlib>

#include "gks_internal.h"

namespace {

enum { BC_PERIODIC = 0, BC_NOSLIP = 1, BC_SLIP = 2, BC_INFLOW = 3, BC_OUTFLOW = 4, BC_EXTRAP = 5, BC_HALO = 6 };

/* AX = axis being filled; (u,v) run over the two other axes: u the lower one.  One thread fills the 3 ghosts of
 * ONE component of one line end: its (at most 3) source values are all loaded before the first store, so a thread
 * pays one memory latency, and the pass has four times as many threads to hide it (the ghost passes are pure
 * latency: a few MB per pass). */
template <int AX>
__global__ void __launch_bounds__(128) k_ghost(GksGrid g, GksPhys ph, double *W,
                                               const double *Wstate /* may alias W */, int ulo, int ucnt, int vlo,
                                               int vcnt) {
  gks_pdl_enter();
  constexpr int UA = AX == 0 ? 1 : 0, VA = AX == 2 ? 1 : 2;
  const int iu = blockIdx.x * blockDim.x + threadIdx.x;
  const int iv = blockIdx.y;
  const int side = blockIdx.z & 1, c = blockIdx.z >> 1;
  if (iu >= ucnt || iv >= vcnt) return;
  int p[3];
  p[UA] = ulo + iu;
  p[VA] = vlo + iv;
  p[AX] = 0;
  const long long base = g.idx(p[0], p[1], p[2]); /* cell 0 of the line */
  const long long sa = g.st[AX];
  const int n = g.n[AX];
  const int kind = ph.bc[2 * AX + side];
  if (kind == BC_HALO) return;   /* ghosts of a cut face come from the neighbouring sub-domain */
  const int first = side == 0 ? 0 : n - 1;
  double *w = W + c * g.FS + base;
  double q[GKS_NG];
  if (kind == BC_INFLOW) {
    const double sign = side == 0 ? -1.0 : 1.0;
    const double rhoI = W[base + first * sa];
    const double UnI = sign * W[(1 + AX) * g.FS + base + first * sa] / rhoI;
    const double Unb = sign * ph.inflow[1 + AX];
    const double rhob = rhoI * exp((UnI - Unb) / sqrt(ph.RT));
    const double qin = c == 0 ? rhob : rhob * ph.inflow[c];
#pragma unroll
    for (int gi = 1; gi <= GKS_NG; ++gi) q[gi - 1] = qin;
  } else {
#pragma unroll
    for (int gi = 1; gi <= GKS_NG; ++gi) {
      const int ghost = side == 0 ? -gi : n - 1 + gi;
      const int mirror = side == 0 ? gi - 1 : n - gi;
      const int image = side == 0 ? n - gi : gi - 1;
      switch (kind) {
        case BC_PERIODIC: q[gi - 1] = w[image * sa]; break;
        case BC_NOSLIP: q[gi - 1] = c == 0 ? w[mirror * sa] : -w[mirror * sa]; break;
        case BC_SLIP: q[gi - 1] = c == 1 + AX ? -w[mirror * sa] : w[mirror * sa]; break;
        case BC_OUTFLOW: q[gi - 1] = Wstate[c * g.FS + base + ghost * sa]; break;
        default: q[gi - 1] = w[first * sa]; break;
      }
    }
  }
#pragma unroll
  for (int gi = 1; gi <= GKS_NG; ++gi) w[(side == 0 ? -gi : n - 1 + gi) * sa] = q[gi - 1];
}

/* The passes of several axes in ONE kernel, for the boundary kinds whose ghost is a signed copy of one cell (periodic
 * image, wall mirrors, zero-gradient extrapolation): a ghost cell of the pass order x, y, z is then the signed copy of
 * the interior cell that the per-axis index maps lead to, the sign being the product of the mirrors' - the value the
 * three passes produce, bit for bit, without their launch-to-launch dependencies (a step of a small grid is a chain of
 * short kernels).  WITH_X: x, y and z (x faces of those kinds or GKS_BC_HALO, whose ghosts are left alone and serve as
 * sources of the y and z maps); otherwise y and z only, behind an x pass of the general kernel (inflow / outflow on x).
 * Regions (blockIdx.y): 0 = the k-ghost planes, 1 = j-ghost rows of interior planes, 2 = i-ghost cells of interior rows. */
__device__ __forceinline__ int ghost_map(int idx, int n, int kind_lo, int kind_hi, int axis, int c, double &sign) {
  if (idx >= 0 && idx < n) return idx;
  const int kind = idx < 0 ? kind_lo : kind_hi;
  switch (kind) {
    case BC_PERIODIC: return idx < 0 ? idx + n : idx - n;
    case BC_NOSLIP:
      if (c != 0) sign = -sign;
      return idx < 0 ? -1 - idx : 2 * n - 1 - idx;
    case BC_SLIP:
      if (c == 1 + axis) sign = -sign;
      return idx < 0 ? -1 - idx : 2 * n - 1 - idx;
    case BC_EXTRAP: return idx < 0 ? 0 : n - 1;
    default: return idx;   /* HALO (x only): the ghost holds the neighbouring sub-domain's cell */
  }
}

template <bool WITH_X>
__global__ void __launch_bounds__(256) k_ghost_fused(GksGrid g, GksPhys ph, double *W) {
  gks_pdl_enter();
  const int region = blockIdx.y, c = blockIdx.z;
  const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
  const int PXn = n0 + 2 * GKS_NG, PYn = n1 + 2 * GKS_NG;
  const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
  int i, j, k;
  if (region == 0) {
    const long long per = (long long)PXn * PYn;
    if (t >= 2 * GKS_NG * per) return;
    const int l = (int)(t / per), r = (int)(t - l * per);
    k = l < GKS_NG ? l - GKS_NG : n2 + l - GKS_NG;
    j = r / PXn - GKS_NG;
    i = r % PXn - GKS_NG;
  } else if (region == 1) {
    const long long per = (long long)PXn * 2 * GKS_NG;
    if (t >= per * n2) return;
    k = (int)(t / per);
    const int r = (int)(t - k * per), l = r / PXn;
    j = l < GKS_NG ? l - GKS_NG : n1 + l - GKS_NG;
    i = r % PXn - GKS_NG;
  } else {
    const long long per = (long long)2 * GKS_NG * n1;
    if (!WITH_X || t >= per * n2) return;
    k = (int)(t / per);
    const int r = (int)(t - k * per), l = r % (2 * GKS_NG);
    j = r / (2 * GKS_NG);
    i = l < GKS_NG ? l - GKS_NG : n0 + l - GKS_NG;
    if (ph.bc[i < 0 ? 0 : 1] == BC_HALO) return;
  }
  double sign = 1.0;
  const int is = WITH_X ? ghost_map(i, n0, ph.bc[0], ph.bc[1], 0, c, sign) : i;
  const int js = ghost_map(j, n1, ph.bc[2], ph.bc[3], 1, c, sign);
  const int ks = ghost_map(k, n2, ph.bc[4], ph.bc[5], 2, c, sign);
  double *w = W + c * g.FS;
  w[g.idx(i, j, k)] = sign * w[g.idx(is, js, ks)];
}

/* S20: initialise (dt < 0) or advance (dt >= 0) the convective-outflow ghost state of axis AX */
template <int AX>
__global__ void __launch_bounds__(128) k_outflow(GksGrid g, GksPhys ph, double *__restrict__ W, double dt, int ulo,
                                                 int ucnt, int vlo, int vcnt) {
  gks_pdl_enter();
  constexpr int UA = AX == 0 ? 1 : 0, VA = AX == 2 ? 1 : 2;
  const int iu = blockIdx.x * blockDim.x + threadIdx.x;
  const int iv = blockIdx.y;
  const int side = blockIdx.z & 1;
  const int c = blockIdx.z >> 1;
  if (iu >= ucnt || iv >= vcnt) return;
  if (ph.bc[2 * AX + side] != BC_OUTFLOW) return;
  int p[3];
  p[UA] = ulo + iu;
  p[VA] = vlo + iv;
  p[AX] = 0;
  double *w = W + c * g.FS + g.idx(p[0], p[1], p[2]);
  const long long sa = g.st[AX];
  const int n = g.n[AX];
  const double *xc = g.xc[AX] + GKS_NG;
  const double Uc = fabs(ph.inflow[1 + AX]);
  double prev = w[(side == 0 ? 0 : n - 1) * sa];
  for (int gi = 1; gi <= GKS_NG; ++gi) {
    const int ghost = side == 0 ? -gi : n - 1 + gi;
    const int inner = side == 0 ? -gi + 1 : n - 2 + gi;
    double phi;
    if (dt < 0) {
      phi = prev; /* start from the last interior value */
    } else {
      const double C = Uc * dt / fabs(xc[ghost] - xc[inner]);
      phi = w[ghost * sa];
      phi = phi - C * (phi - prev);
      prev = phi;
    }
    w[ghost * sa] = phi;
  }
}

/* the 3 interior planes next to a face (pack) or the 3 ghost planes beyond it (unpack) <-> buf[c][layer][v][u] */
template <int AX>
__global__ void __launch_bounds__(128) k_halo(GksGrid g, double *__restrict__ W, double *__restrict__ buf, int side,
                                              int unpack) {
  gks_pdl_enter();
  constexpr int UA = AX == 0 ? 1 : 0, VA = AX == 2 ? 1 : 2;
  const int iu = blockIdx.x * blockDim.x + threadIdx.x;
  const int iv = blockIdx.y;
  const int layer = blockIdx.z % GKS_NG, c = blockIdx.z / GKS_NG;
  if (iu >= g.n[UA] || iv >= g.n[VA]) return;
  const int n = g.n[AX];
  int p[3];
  p[UA] = iu;
  p[VA] = iv;
  p[AX] = unpack ? (side == 0 ? -GKS_NG + layer : n + layer) : (side == 0 ? layer : n - GKS_NG + layer);
  const long long id = c * g.FS + g.idx(p[0], p[1], p[2]);
  const long long b = (((long long)c * GKS_NG + layer) * g.n[VA] + iv) * g.n[UA] + iu;
  if (unpack) W[id] = buf[b];
  else buf[b] = W[id];
}

/* the 3 interior planes next to an x face of THIS context straight into the ghost planes beyond the opposite x face of
 * a NEIGHBOUR's padded state (its window: base pointer, pitches, nx): pack, transfer and unpack in one kernel - the
 * stores travel peer-to-peer when the window lives on another GPU of the NVSwitch domain */
__global__ void __launch_bounds__(128) k_halo_push(GksGrid g, const double *__restrict__ W, int side, double *__restrict__ dstW,
                                                   int dnx, int dPX, int dPY, long long dFS) {
  gks_pdl_enter();
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y;
  const int layer = blockIdx.z % GKS_NG, c = blockIdx.z / GKS_NG;
  if (j >= g.n[1] || k >= g.n[2]) return;
  const int isrc = side == 0 ? layer : g.n[0] - GKS_NG + layer;
  const int idst = side == 0 ? dnx + layer : -GKS_NG + layer;      /* my low face feeds the neighbour's HIGH ghosts */
  const long long d = c * dFS + ((long long)(k + GKS_NG) * dPY + (j + GKS_NG)) * dPX + (idst + GKS_NG);
  dstW[d] = W[c * g.FS + g.idx(isrc, j, k)];
}

__global__ void __launch_bounds__(256) k_pack(GksGrid g, double *__restrict__ Wint, double *__restrict__ Wpad,
                                              int to_padded, int ex, int ey, int ez) {
  gks_pdl_enter();
  /* interior box (n + e) per axis; e = 1 along the sweep direction for face arrays */
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const int nx = g.n[0] + ex, ny = g.n[1] + ey, nz = g.n[2] + ez;
  if (i >= nx || j >= ny || k >= nz) return;
  /* face arrays: on a periodic axis face n is stored as face 0 */
  const long long ip = g.idx((ex && g.wrapf[0] && i == g.n[0]) ? 0 : i, (ey && g.wrapf[1] && j == g.n[1]) ? 0 : j,
                             (ez && g.wrapf[2] && k == g.n[2]) ? 0 : k);
  const long long ii = ((long long)k * ny + j) * nx + i;
  const long long N = (long long)nx * ny * nz;
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (to_padded) Wpad[c * g.FS + ip] = Wint[c * N + ii];
    else Wint[c * N + ii] = Wpad[c * g.FS + ip];
  }
}

__global__ void __launch_bounds__(256) k_check_finite(GksGrid g, const double *__restrict__ W, int *flag) {
  gks_pdl_enter();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= g.n[0] || j >= g.n[1] || k >= g.n[2]) return;
  const long long ip = g.idx(i, j, k);
  bool bad = false;
#pragma unroll
  for (int c = 0; c < 4; ++c) bad |= !isfinite(W[c * g.FS + ip]);
  if (bad) atomicOr(flag, 1);
}

/* lines of pass AX: x pass: interior (j,k); y pass: all i, interior k; z pass: all i, all j */
template <int AX>
struct PassLines {
  static constexpr int UA = AX == 0 ? 1 : 0, VA = AX == 2 ? 1 : 2;
  int ulo, ucnt, vlo, vcnt;
  explicit PassLines(const GksGrid &g)
      : ulo(AX == 0 ? 0 : -GKS_NG), ucnt(AX == 0 ? g.n[UA] : g.n[UA] + 2 * GKS_NG), vlo(AX == 2 ? -GKS_NG : 0),
        vcnt(AX == 2 ? g.n[VA] + 2 * GKS_NG : g.n[VA]) {}
};

template <int AX>
void launch_ghost_axis(const GksGrid &g, const GksPhys &ph, double *W, const double *Wstate, cudaStream_t s) {
  const PassLines<AX> L(g);
  dim3 grid((L.ucnt + 127) / 128, L.vcnt, 8);       /* z: (side, component) */
  gks_launch(k_ghost<AX>, grid, dim3(128), 0, s, g, ph, W, Wstate, L.ulo, L.ucnt, L.vlo, L.vcnt);
}

static bool outflow_on(const GksPhys &ph, int ax) {
  return ph.bc[2 * ax] == BC_OUTFLOW || ph.bc[2 * ax + 1] == BC_OUTFLOW;
}

template <int AX>
int launch_outflow_axis(const GksGrid &g, const GksPhys &ph, double *W, double dt, cudaStream_t s) {
  if (!outflow_on(ph, AX)) return 0;
  const PassLines<AX> L(g);
  dim3 grid((L.ucnt + 127) / 128, L.vcnt, 8);
  gks_launch(k_outflow<AX>, grid, dim3(128), 0, s, g, ph, W, dt, L.ulo, L.ucnt, L.vlo, L.vcnt);
  return 1;
}

/* initialise (dt < 0) or advance the outflow ghost state of every axis that has some.  The state of the y (z)
 * axis also lives on the lines through the x (x and y) ghosts: those must be current first, so the passes of
 * the lower axes run in between - only when there IS an outflow face on y or z (the paper's cases have theirs on x) */
int outflow_state(const GksGrid &g, const GksPhys &ph, double *W, double dt, cudaStream_t s) {
  int n = launch_outflow_axis<0>(g, ph, W, dt, s);
  if (!outflow_on(ph, 1) && !outflow_on(ph, 2)) return n;
  launch_ghost_axis<0>(g, ph, W, W, s);
  n += 1 + launch_outflow_axis<1>(g, ph, W, dt, s);
  if (!outflow_on(ph, 2)) return n;
  launch_ghost_axis<1>(g, ph, W, W, s);
  n += 1 + launch_outflow_axis<2>(g, ph, W, dt, s);
  return n;
}

} /* namespace */

static bool copy_kind(int kind) { return kind == BC_PERIODIC || kind == BC_NOSLIP || kind == BC_SLIP || kind == BC_EXTRAP; }

int gks_launch_ghost_fill(const GksGrid &g, const GksPhys &ph, double *W, const double *Wstate, cudaStream_t s) {
  static const bool fused_on = [] {
    const char *e = getenv("GKS_GHOST_FUSED");        /* GKS_GHOST_FUSED=0: always the three passes */
    return !(e && e[0] == '0');
  }();
  const bool yz = copy_kind(ph.bc[2]) && copy_kind(ph.bc[3]) && copy_kind(ph.bc[4]) && copy_kind(ph.bc[5]);
  const bool x = (copy_kind(ph.bc[0]) || ph.bc[0] == BC_HALO) && (copy_kind(ph.bc[1]) || ph.bc[1] == BC_HALO);
  if (fused_on && yz) {
    const long long PXn = g.n[0] + 2 * GKS_NG, PYn = g.n[1] + 2 * GKS_NG;
    long long most = 2 * GKS_NG * PXn * PYn;                                        /* region 0 */
    if (2 * GKS_NG * PXn * g.n[2] > most) most = 2 * GKS_NG * PXn * g.n[2];         /* region 1 */
    if (x && (long long)2 * GKS_NG * g.n[1] * g.n[2] > most) most = (long long)2 * GKS_NG * g.n[1] * g.n[2];
    const dim3 grid((unsigned)((most + 255) / 256), x ? 3 : 2, 4);
    if (x) {
      gks_launch(k_ghost_fused<true>, grid, dim3(256), 0, s, g, ph, W);
      return 1;
    }
    launch_ghost_axis<0>(g, ph, W, Wstate, s);
    gks_launch(k_ghost_fused<false>, grid, dim3(256), 0, s, g, ph, W);
    return 2;
  }
  launch_ghost_axis<0>(g, ph, W, Wstate, s);
  launch_ghost_axis<1>(g, ph, W, Wstate, s);
  launch_ghost_axis<2>(g, ph, W, Wstate, s);
  return 3;
}

int gks_launch_ghost_fill_xcols(const GksGrid &g, const GksPhys &ph, double *W, const double *Wstate, cudaStream_t s) {
  int n = 0;
  for (int side = 0; side < 2; ++side) {
    if (!g.halo[side]) continue;
    const int ulo = side == 0 ? -GKS_NG : g.n[0];
    const PassLines<1> Ly(g);
    const PassLines<2> Lz(g);
    gks_launch(k_ghost<1>, dim3(1, Ly.vcnt, 8), dim3(128), 0, s, g, ph, W, Wstate, ulo, GKS_NG, Ly.vlo, Ly.vcnt);
    gks_launch(k_ghost<2>, dim3(1, Lz.vcnt, 8), dim3(128), 0, s, g, ph, W, Wstate, ulo, GKS_NG, Lz.vlo, Lz.vcnt);
    n += 2;
  }
  return n;
}

int gks_launch_outflow_init(const GksGrid &g, const GksPhys &ph, double *W, cudaStream_t s) {
  return outflow_state(g, ph, W, -1.0, s);
}

int gks_launch_outflow_advance(const GksGrid &g, const GksPhys &ph, double *W, double dt, cudaStream_t s) {
  return outflow_state(g, ph, W, dt, s);
}

static dim3 grid2d(int nx, int ny, int nz) { return dim3((nx + 63) / 64, (ny + 3) / 4, nz); }

int gks_launch_pack(const GksGrid &g, const double *Wint, double *Wpad, cudaStream_t s) {
  gks_launch(k_pack, dim3(grid2d(g.n[0], g.n[1], g.n[2])), dim3(64, 4), 0, s, g, const_cast<double *>(Wint), Wpad, 1, 0, 0, 0);
  return 1;
}

int gks_launch_unpack(const GksGrid &g, const double *Wpad, double *Wint, cudaStream_t s) {
  gks_launch(k_pack, dim3(grid2d(g.n[0], g.n[1], g.n[2])), dim3(64, 4), 0, s, g, Wint, const_cast<double *>(Wpad), 0, 0, 0, 0);
  return 1;
}

int gks_launch_halo(const GksGrid &g, double *W, double *buf, int face, int unpack, cudaStream_t s) {
  const int ax = face >> 1, side = face & 1;
  const int ua = ax == 0 ? 1 : 0, va = ax == 2 ? 1 : 2;
  dim3 grid((g.n[ua] + 127) / 128, g.n[va], 4 * GKS_NG);
  if (ax == 0) gks_launch(k_halo<0>, grid, dim3(128), 0, s, g, W, buf, side, unpack);
  else if (ax == 1) gks_launch(k_halo<1>, grid, dim3(128), 0, s, g, W, buf, side, unpack);
  else gks_launch(k_halo<2>, grid, dim3(128), 0, s, g, W, buf, side, unpack);
  return 1;
}

int gks_launch_halo_push(const GksGrid &g, const double *W, int side, double *dstW, int dnx, int dPX, int dPY,
                         long long dFS, cudaStream_t s) {
  dim3 grid((g.n[1] + 127) / 128, g.n[2], 4 * GKS_NG);
  gks_launch(k_halo_push, grid, dim3(128), 0, s, g, W, side, dstW, dnx, dPX, dPY, dFS);
  return 1;
}

int gks_launch_unpack_faces(const GksGrid &g, int dir, const double *Fpad, double *Fout, cudaStream_t s) {
  const int ex = dir == 0, ey = dir == 1, ez = dir == 2;
  gks_launch(k_pack, dim3(grid2d(g.n[0] + ex, g.n[1] + ey, g.n[2] + ez)), dim3(64, 4), 0, s, 
      g, Fout, const_cast<double *>(Fpad), 0, ex, ey, ez);
  return 1;
}

int gks_launch_check_finite(const GksGrid &g, const double *W, int *flag, cudaStream_t s) {
  gks_launch(k_check_finite, dim3(grid2d(g.n[0], g.n[1], g.n[2])), dim3(64, 4), 0, s, g, W, flag);
  return 1;
}
