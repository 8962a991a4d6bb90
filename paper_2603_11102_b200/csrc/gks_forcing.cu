/*
 * gks_forcing.cu — the body-force term of Eq. 13: uniform / bulk-flux term
 * (PAPER.md:237), IBM direct forcing (Eq. 11-12; Lagrangian-centred form,
 * DESIGN.md S13-S15), ALM Gaussian projection (Eq. 10, cut at 3 eps :293; S22-S23).
 *
 * Every increment is computed from the un-forced W^{n+1} (S12): the bulk reduction and the IBM
 * interpolation run first and only read; the three adding kernels run afterwards and touch only
 * momentum (IBM spreading reads rho, which no forcing term changes).
 */
#include "gks_internal.h"
#include "gks_math.cuh"

namespace {

constexpr int RED_BLOCKS = GKS_RED_BULK_SUM;

/* ---- bulk momentum: deterministic two-level sum of m_axis * |Omega| over the interior ---- */
__global__ void __launch_bounds__(256) k_bulk_partial(GksGrid g, const double *__restrict__ W, int axis,
                                                      double *__restrict__ red) {
  gks_pdl_enter();
  __shared__ double sh[256];
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  const long long per = (N + RED_BLOCKS - 1) / RED_BLOCKS;
  const long long beg = blockIdx.x * per, end = min(N, beg + per);
  double acc = 0.0;
  for (long long t = beg + threadIdx.x; t < end; t += 256) {
    const int i = (int)(t % g.n[0]);
    const int j = (int)((t / g.n[0]) % g.n[1]);
    const int k = (int)(t / ((long long)g.n[0] * g.n[1]));
    const double vol = g.w[0][i + GKS_NG] * g.w[1][j + GKS_NG] * g.w[2][k + GKS_NG];
    acc += W[(1 + axis) * g.FS + g.idx(i, j, k)] * vol;
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) red[blockIdx.x] = sh[0];
}

__global__ void __launch_bounds__(256) k_bulk_final(double *__restrict__ red) {
  gks_pdl_enter();
  __shared__ double sh[256];
  double acc = 0.0;
  for (int t = threadIdx.x; t < RED_BLOCKS; t += 256) acc += red[t];
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) red[RED_BLOCKS] = sh[0];
}

/* ---- CFL time step: |U|_max over the interior, then dt = CFL dmin / (|U|_max + sqrt(RT)) ---- */
__global__ void __launch_bounds__(256) k_umax(GksGrid g, const double *__restrict__ W, unsigned long long *__restrict__ out) {
  gks_pdl_enter();
  __shared__ double sh[256];
  const long long N = (long long)g.n[0] * g.n[1] * g.n[2];
  double acc = 0.0;
  for (long long t = (long long)blockIdx.x * 256 + threadIdx.x; t < N; t += (long long)gridDim.x * 256) {
    const int i = (int)(t % g.n[0]);
    const int j = (int)((t / g.n[0]) % g.n[1]);
    const int k = (int)(t / ((long long)g.n[0] * g.n[1]));
    const long long id = g.idx(i, j, k);
    const double mx = W[g.FS + id], my = W[2 * g.FS + id], mz = W[3 * g.FS + id];
    acc = fmax(acc, sqrt(mx * mx + my * my + mz * mz) / W[id]);
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sh[threadIdx.x] = fmax(sh[threadIdx.x], sh[threadIdx.x + s]);
    __syncthreads();
  }
  /* non-negative doubles order like their bit patterns */
  if (threadIdx.x == 0) atomicMax(out, (unsigned long long)__double_as_longlong(sh[0]));
}

__global__ void k_cfl_final(const unsigned long long *__restrict__ umax_bits, double cfl, double dmin, double cs,
                            double *__restrict__ dt) {
  gks_pdl_enter();
  *dt = cfl * dmin / (__longlong_as_double((long long)*umax_bits) + cs);
}

/* m += dt rho g ;  m_axis += target - sum(m_axis |Omega|)/sum|Omega|   (S16) */
__global__ void __launch_bounds__(256) k_uniform_force(GksGrid g, double *__restrict__ W, double dt, double gx,
                                                       double gy, double gz, int bulk_axis, double target,
                                                       double total_volume, const double *__restrict__ red) {
  gks_pdl_enter();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= g.n[0] || j >= g.n[1]) return;
  const long long id = g.idx(i, j, k);
  const double rho = W[id];
  double inc[3] = {dt * rho * gx, dt * rho * gy, dt * rho * gz};
  if (bulk_axis >= 0) inc[bulk_axis] += target - red[RED_BLOCKS] / total_volume;
#pragma unroll
  for (int c = 0; c < 3; ++c)
    if (inc[c] != 0.0) W[(1 + c) * g.FS + id] += inc[c];
}

/* ---- IBM ---- */
/* cell containing x on axis a (caller guarantees lo <= x <= hi; beyond a HALO face, which needs a uniform axis,
 * the two nearest ghost cells count as well: a Lagrangian point of the neighbouring sub-domain) */
constexpr int IBM_DROP = -2147483647 - 1;   /* support cell outside the domain: no weight */
__device__ __forceinline__ int find_cell(const GksGrid &g, int a, double x) {
  const int n = g.n[a];
  if (g.uniform[a]) {
    int c = (int)floor((x - g.x0[a]) / g.dx[a]);
    return max(g.halo[2 * a] ? -2 : 0, min(g.halo[2 * a + 1] ? n + 1 : n - 1, c));
  }
  const double *xf = g.xf[a] + GKS_NG;
  int lo = 0, hi = n;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (x >= xf[mid]) lo = mid; else hi = mid;
  }
  return lo;
}

struct Support {
  int idx[3][3];
  double phi[3][3];
};

__device__ __forceinline__ void ibm_support(const GksGrid &g, const double *X, Support &sp) {
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int c0 = find_cell(g, a, X[a]);
    const double ih = g.inv_w[a][c0 + GKS_NG];
    const double *xc = g.xc[a] + GKS_NG;
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      const int i = c0 - 1 + m;
      sp.phi[a][m] = gksd::delta3((xc[i] - X[a]) * ih);
      int w = i;   /* ghost cells of a HALO face keep their index: readable, but owned by the neighbour */
      if (i < 0) w = g.periodic[a] ? i + g.n[a] : (g.halo[2 * a] ? i : IBM_DROP);
      else if (i >= g.n[a]) w = g.periodic[a] ? i - g.n[a] : (g.halo[2 * a + 1] ? i : IBM_DROP);
      sp.idx[a][m] = w;
    }
  }
}

/* Stop rule of the multi-direct-forcing passes (S25), evaluated on the device so
 * that gks_step stays asynchronous: res[k] holds max_p |v_p - U_p| seen by pass k >= 1 as the bit pattern of
 * a non-negative double (ordered like an unsigned integer), zeroed at the start of every step.  Pass k is
 * skipped when pass k or any earlier pass found a slip below tol; a skipped pass leaves res[k] = 0 < tol,
 * which carries the decision forward. */
__device__ __forceinline__ bool ibm_below_tol(const unsigned long long *res, int k, double tol) {
  return __longlong_as_double((long long)res[k]) < tol;
}

/* U_p = sum phi phi phi (m/rho);  coef_p = (v_p - U_p) V_p */
__global__ void __launch_bounds__(128) k_ibm_interp(GksGrid g, const double *__restrict__ W, int n,
                                                    const double *__restrict__ pos, const double *__restrict__ vol,
                                                    const double *__restrict__ vel, double *__restrict__ coef,
                                                    int pass, double tol, unsigned long long *__restrict__ res) {
  gks_pdl_enter();
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  if (pass >= 2 && ibm_below_tol(res, pass - 1, tol)) return;
  const double X[3] = {pos[3 * p], pos[3 * p + 1], pos[3 * p + 2]};
  Support sp;
  ibm_support(g, X, sp);
  double U[3] = {0, 0, 0};
  for (int mk = 0; mk < 3; ++mk)
    for (int mj = 0; mj < 3; ++mj)
      for (int mi = 0; mi < 3; ++mi) {
        const int i = sp.idx[0][mi], j = sp.idx[1][mj], k = sp.idx[2][mk];
        if (i == IBM_DROP || j == IBM_DROP || k == IBM_DROP) continue;
        const double wgt = sp.phi[0][mi] * sp.phi[1][mj] * sp.phi[2][mk];
        const long long id = g.idx(i, j, k);
        const double ir = 1.0 / W[id];
#pragma unroll
        for (int c = 0; c < 3; ++c) U[c] += wgt * (W[(1 + c) * g.FS + id] * ir);
      }
  double r2 = 0.0;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double d = vel[3 * p + c] - U[c];
    r2 += d * d;
    coef[3 * p + c] = d * vol[p];
  }
  if (pass >= 1) atomicMax(&res[pass], (unsigned long long)__double_as_longlong(sqrt(r2)));
}

/* one thread per (point, support cell): m_ijk += rho_ijk coef_p phi phi phi / |Omega_ijk| */
__global__ void __launch_bounds__(128) k_ibm_spread(GksGrid g, double *__restrict__ W, int n,
                                                    const double *__restrict__ pos, const double *__restrict__ coef,
                                                    int pass, double tol, const unsigned long long *__restrict__ res) {
  gks_pdl_enter();
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int p = (int)(t / 27);
  if (p >= n) return;
  if (pass >= 1 && ibm_below_tol(res, pass, tol)) return;
  const int m = (int)(t % 27), mi = m % 3, mj = (m / 3) % 3, mk = m / 9;
  const double X[3] = {pos[3 * p], pos[3 * p + 1], pos[3 * p + 2]};
  Support sp;
  ibm_support(g, X, sp);
  const int i = sp.idx[0][mi], j = sp.idx[1][mj], k = sp.idx[2][mk];
  /* only cells this sub-domain owns (dropped cells and HALO ghosts fall outside [0, n)) */
  if (i < 0 || j < 0 || k < 0 || i >= g.n[0] || j >= g.n[1] || k >= g.n[2]) return;
  const double wgt = sp.phi[0][mi] * sp.phi[1][mj] * sp.phi[2][mk];
  if (wgt == 0.0) return;
  const long long id = g.idx(i, j, k);
  const double ivol = g.inv_w[0][i + GKS_NG] * g.inv_w[1][j + GKS_NG] * g.inv_w[2][k + GKS_NG];
  const double f = W[id] * wgt * ivol;
#pragma unroll
  for (int c = 0; c < 3; ++c) atomicAdd(&W[(1 + c) * g.FS + id], f * coef[3 * p + c]);
}

/* ---- ALM: gather over the bounding box of the support; deterministic, no atomics.
 * One thread per cell of the box (indices are unwrapped: a periodic axis maps them back), points
 * staged through shared memory in chunks; contributions are added in point order. ---- */
constexpr int ALM_CHUNK = 256;

__global__ void __launch_bounds__(128) k_alm(GksGrid g, double *__restrict__ W, int n, const double *__restrict__ pos,
                                             const double *__restrict__ force, double eps, double dt, int lo0,
                                             int lo1, int lo2, int c0, int c1, int c2) {
  gks_pdl_enter();
  __shared__ double sp[ALM_CHUNK * 3], sf[ALM_CHUNK * 3];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)c0 * c1 * c2;
  const bool active = t < total;
  int iu[3] = {0, 0, 0};
  double xc[3] = {0, 0, 0};
  long long id = 0;
  /* a box that covers a whole periodic axis (point cloud + support wider than the axis) visits every cell once and
     takes the nearest image of each point along that axis; 6 eps < L (checked by the host) leaves only one in range */
  double Lmi[3];
  {
    const int cc[3] = {c0, c1, c2};
#pragma unroll
    for (int a = 0; a < 3; ++a)
      Lmi[a] = (g.periodic[a] && cc[a] == g.n[a]) ? g.xf[a][g.n[a] + GKS_NG] - g.xf[a][GKS_NG] : 0.0;
  }
  if (active) {
    iu[0] = lo0 + (int)(t % c0);
    iu[1] = lo1 + (int)((t / c0) % c1);
    iu[2] = lo2 + (int)(t / ((long long)c0 * c1));
    int iw[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { /* unwrapped centre: xc[r] + m L */
      const int nn = g.n[a];
      int m = iu[a] / nn, r = iu[a] - m * nn;
      if (r < 0) { r += nn; m -= 1; }
      iw[a] = r;
      const double L = g.xf[a][nn + GKS_NG] - g.xf[a][GKS_NG];
      xc[a] = g.xc[a][r + GKS_NG] + m * L;
    }
    id = g.idx(iw[0], iw[1], iw[2]);
  }
  const double R2 = 9.0 * eps * eps;
  const double ie2 = 1.0 / (eps * eps);
  const double norm = dt / (eps * eps * eps * 5.5683279968317078453); /* pi^1.5 */
  double acc[3] = {0, 0, 0};
  for (int base = 0; base < n; base += ALM_CHUNK) {
    const int cnt = min(ALM_CHUNK, n - base);
    __syncthreads();
    for (int q = threadIdx.x; q < cnt * 3; q += blockDim.x) {
      sp[q] = pos[3 * base + q];
      sf[q] = force[3 * base + q];
    }
    __syncthreads();
    if (active) {
      for (int q = 0; q < cnt; ++q) {
        double rx = xc[0] - sp[3 * q], ry = xc[1] - sp[3 * q + 1], rz = xc[2] - sp[3 * q + 2];
        if (Lmi[0] > 0.0) rx -= Lmi[0] * rint(rx / Lmi[0]);
        if (Lmi[1] > 0.0) ry -= Lmi[1] * rint(ry / Lmi[1]);
        if (Lmi[2] > 0.0) rz -= Lmi[2] * rint(rz / Lmi[2]);
        const double r2 = rx * rx + ry * ry + rz * rz;
        if (r2 <= R2) {
          const double kern = norm * exp(-r2 * ie2);
          acc[0] += sf[3 * q] * kern;
          acc[1] += sf[3 * q + 1] * kern;
          acc[2] += sf[3 * q + 2] * kern;
        }
      }
    }
  }
  if (active) {
#pragma unroll
    for (int c = 0; c < 3; ++c)
      if (acc[c] != 0.0) W[(1 + c) * g.FS + id] += acc[c];
  }
}

} /* namespace */

int gks_launch_bulk_reduce(const GksGrid &g, const double *W, int axis, double *red, cudaStream_t s) {
  gks_launch(k_bulk_partial, RED_BLOCKS, dim3(256), 0, s, g, W, axis, red);
  gks_launch(k_bulk_final, dim3(1), dim3(256), 0, s, red);
  return 2;
}

int gks_launch_cfl_dt(const GksGrid &g, const double *W, double cfl, double dmin, double cs, double *scratch,
                      cudaStream_t s) {
  /* scratch[0]: bit pattern of |U|_max (zeroed by the caller), scratch[1]: dt */
  gks_launch(k_umax, RED_BLOCKS, dim3(256), 0, s, g, W, reinterpret_cast<unsigned long long *>(scratch));
  gks_launch(k_cfl_final, dim3(1), dim3(1), 0, s, reinterpret_cast<const unsigned long long *>(scratch), cfl, dmin, cs, scratch + 1);
  return 2;
}

int gks_launch_uniform_force(const GksGrid &g, double *W, double dt, const double gacc[3], int bulk_axis,
                             double bulk_target, double total_volume, const double *red, cudaStream_t s) {
  dim3 blk(64, 4), grid((g.n[0] + 63) / 64, (g.n[1] + 3) / 4, g.n[2]);
  gks_launch(k_uniform_force, grid, blk, 0, s, g, W, dt, gacc[0], gacc[1], gacc[2], bulk_axis, bulk_target, total_volume, red);
  return 1;
}

int gks_launch_ibm_interp(const GksGrid &g, const double *W, int n, const double *pos, const double *vol,
                          const double *vel, double *coef, int pass, double tol, unsigned long long *res,
                          cudaStream_t s) {
  gks_launch(k_ibm_interp, dim3((n + 127) / 128), dim3(128), 0, s, g, W, n, pos, vol, vel, coef, pass, tol, res);
  return 1;
}

int gks_launch_ibm_spread(const GksGrid &g, double *W, int n, const double *pos, const double *coef, int pass,
                          double tol, const unsigned long long *res, cudaStream_t s) {
  const long long t = (long long)n * 27;
  gks_launch(k_ibm_spread, dim3((unsigned)((t + 127) / 128)), dim3(128), 0, s, g, W, n, pos, coef, pass, tol, res);
  return 1;
}

int gks_launch_alm(const GksGrid &g, double *W, int n, const double *pos, const double *force, double eps,
                   double dt, const int lo[3], const int cnt[3], cudaStream_t s) {
  const long long t = (long long)cnt[0] * cnt[1] * cnt[2];
  if (t <= 0) return 0;
  gks_launch(k_alm, dim3((unsigned)((t + 127) / 128)), dim3(128), 0, s, g, W, n, pos, force, eps, dt, lo[0], lo[1], lo[2], cnt[0], cnt[1],
                                                    cnt[2]);
  return 1;
}
