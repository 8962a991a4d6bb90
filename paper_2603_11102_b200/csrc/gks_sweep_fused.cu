/*
 * gks_sweep_fused.cu — the production sweep: reconstruction + collision + tangential passes +
 * Gauss-point flux of one direction fused in ONE kernel (Eq. 6-8, Appendix :501-558;
 * DESIGN.md readings S1-S11).  No intermediate leaves the SM.
 *
 * Decomposition.  A CTA owns a TA x TB tile of faces in the plane spanned by the memory-fastest
 * axis a (= x) and a second axis b, and MARCHES along the remaining axis, which is always the
 * second tangential direction t2 of the sweep (S9: lower tangential axis first):
 *     DIR 0 (x-faces): a = x = normal, b = y = t1, march z = t2
 *     DIR 1 (y-faces): a = x = t1,     b = y = normal, march z = t2
 *     DIR 2 (z-faces): a = x = t1,     b = z = normal, march y = t2
 * Per marched plane p the CTA
 *   A  reconstructs both edge values of every cell (one smoothness-indicator set per cell serves
 *      the face on either side) from the W halo slab that TMA staged in shared memory,
 *   B  evaluates the collision factors (erfc/exp) once per face,
 *   C  forms Q0 and the normal slope Dn on the TN x (T1+4) halo faces,
 *   D  runs tangential pass 1 (along t1) and pushes 24 doubles per face into a 5-plane ring in
 *      shared memory,
 *   E  runs tangential pass 2 (along t2) for plane p-2 out of the ring,
 *   F  evaluates the four Gauss-point fluxes and writes the face average F, dF/dt to HBM.
 * Thread mapping: 4 threads per face.  In A-E thread (face, c) owns component c (WENO is
 * component-wise); in F thread (face, g) owns Gauss point g (the flux couples all components);
 * the 4x4 transpose goes through shared memory and needs only __syncwarp.
 * The W slab of plane p+2 is fetched by TMA (cp.async.bulk.tensor, mbarrier completion) while plane
 * p is processed: 2-stage pipeline, one elected thread issues.
 *
 * Roofline: fp64-ALU bound (about 4.7 kflop per face against 32 B read + 64 B written per face).
 */
#include <cuda.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "gks_internal.h"
#include "gks_math.cuh"

namespace {

/* ---------------- PTX helpers: mbarrier + TMA ---------------- */
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

/* ---------------- compile-time geometry of a tile ---------------- */
template <int DIR, int TA, int TB>
struct Tile {
  static constexpr bool NA = (DIR == 0);            /* normal along a */
  static constexpr int TN = NA ? TA : TB;           /* faces along the normal */
  static constexpr int T1 = NA ? TB : TA;           /* faces along t1 */
  static constexpr int NF = TA * TB;                /* faces per CTA and plane */
  static constexpr int NT = NF * 4;                 /* threads */
  static constexpr int CA = NA ? TN + 5 : T1 + 5;   /* cells of the W slab along a / b; the slab always starts at
                                                       cell a0-3: TMA needs a 16-byte aligned box start (even index) */
  static constexpr int CB = NA ? T1 + 4 : TN + 5;
  static constexpr int EA = (CA + 1) & ~1;          /* TMA box: inner extent even (16-byte rows) */
  static constexpr int EB = CB;
  static constexpr int HA = NA ? TN : T1 + 4;       /* halo-face box (faces needed by pass 1) */
  static constexpr int HB = NA ? T1 + 4 : TN;
  static constexpr int FH = HA * HB;
  static constexpr int NCA = NA ? TN + 1 : T1 + 4;  /* cells reconstructed in phase A */
  static constexpr int NCB = NA ? T1 + 4 : TN + 1;
  static constexpr int AXB = DIR == 2 ? 2 : 1;      /* global axis of b */
  static constexpr int AXM = DIR == 2 ? 1 : 2;      /* global axis marched (= t2) */
  static constexpr int AXT1 = DIR == 0 ? 1 : 0;
  static constexpr int WSLAB = 4 * EB * EA;         /* doubles per staged slab */
  static constexpr int WSLAB_PAD = (WSLAB + 15) & ~15;
  static constexpr int XBS = 68;                    /* padded per-face stride of the transpose buffer */
  /* shared memory carve (doubles) */
  static constexpr int OFF_W = 0;
  static constexpr int OFF_Q = OFF_W + 2 * WSLAB_PAD;      /* QL|QR (then Q0|Dn), [2][FH][4] */
  static constexpr int OFF_CF = OFF_Q + 2 * FH * 4;        /* collision factors [FH][4] */
  static constexpr int OFF_XB = OFF_Q;                     /* transpose buffer aliases Q|CF (phases E,F) */
  static constexpr int QCF = 3 * FH * 4;
  static constexpr int XB = NF * XBS;
  static constexpr int OFF_RING = OFF_Q + (QCF > XB ? QCF : XB);
  static constexpr int RING = 5 * 6 * NF * 4;
  static constexpr int OFF_BAR = OFF_RING + RING;
  static constexpr size_t SMEM_BYTES = (size_t)(OFF_BAR + 2) * 8;
};

template <int DIR, bool NEED_F, int TA, int TB>
__global__ void __launch_bounds__(TA *TB * 4, 2)
    k_sweep_fused(const __grid_constant__ CUtensorMap tmap, GksGrid g, GksPhys ph, double *__restrict__ flux, int MC, int dbg) {
  using T = Tile<DIR, TA, TB>;
  constexpr int TN = T::TN, T1 = T::T1, NF = T::NF, NT = T::NT, EA = T::EA, EB = T::EB, HA = T::HA, FH = T::FH;
  extern __shared__ __align__(128) double sm[];
  double *const Wp = sm + T::OFF_W;
  double *const QL = sm + T::OFF_Q;            /* [FH][4] */
  double *const QR = QL + FH * 4;              /* [FH][4] */
  double *const CF = sm + T::OFF_CF;           /* [FH][4]: el, rho_l*xl, er, rho_r*xr */
  double *const XBuf = sm + T::OFF_XB;
  double *const ring = sm + T::OFF_RING;       /* [5][6][NF][4] */
  uint64_t *const bar = reinterpret_cast<uint64_t *>(sm + T::OFF_BAR);

  const int tid = threadIdx.x;
  const int a0 = blockIdx.x * TA, b0 = blockIdx.y * TB;
  const int m0 = blockIdx.z * MC;
  const int m1 = min(m0 + MC, g.n[T::AXM]);
  const int p0 = m0 - 2, np = (m1 - m0) + 4;   /* planes p0 .. p0+np-1 */
  const double eps = ph.weno_eps;

  /* face owned in phases D-F */
  const int c = tid & 3, fid = tid >> 2;
  const int fa = fid % TA, fb = fid / TA;       /* a fastest: coalesced output */
  const int ga = a0 + fa, gb = b0 + fb;         /* global indices along a and b */
  const int n_a = g.n[0] + (T::NA ? 1 : 0), n_b = g.n[T::AXB] + (T::NA ? 0 : 1);
  const bool face_ok = ga < n_a && gb < n_b;
  const int t1_local = T::NA ? fb : fa, t1_glob = T::NA ? gb : ga;
  const double iw1 = g.inv_w[T::AXT1][min(t1_glob, g.n[T::AXT1] - 1) + GKS_NG];

  /* TMA coordinates (padded index space: cell -3 <-> 0) */
  const int ca0 = a0, cb0 = T::NA ? b0 + 1 : b0;
  auto issue = [&](int it) {
    uint64_t *b = &bar[it & 1];
    double *dst = Wp + (it & 1) * T::WSLAB_PAD;
    const int pm = p0 + it + GKS_NG;
    mbar_expect_tx(b, T::WSLAB * 8);
    if (DIR == 2) tma_load_4d(dst, &tmap, b, ca0, pm, cb0, 0);
    else tma_load_4d(dst, &tmap, b, ca0, cb0, pm, 0);
  };
  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    fence_barrier_init();
  }
  __syncthreads();
  if (dbg == 1) return;
  if (tid == 0) {
    issue(0);
    if (np > 1) issue(1);
  }
  if (dbg == 2) { mbar_wait(&bar[0], 0); mbar_wait(&bar[1], 0); return; }

  for (int it = 0; it < np; ++it) {
    const double *W = Wp + (it & 1) * T::WSLAB_PAD;
    mbar_wait(&bar[it & 1], (it >> 1) & 1);
    if (dbg == 3) { __syncthreads(); if (tid == 0 && it + 2 < np) issue(it + 2); continue; }

    /* ---- A: both edge values of each cell, per component; two cells per thread at a time ---- */
    {
      constexpr int NITEM = T::NCA * T::NCB * 4;
      constexpr int sn = T::NA ? 1 : EA;
      for (int item0 = tid; item0 < NITEM; item0 += 2 * NT) {
        double q[5][2], vl[2], vr[2];
        int cnv[2], ctv[2], ccv[2];
        bool ok[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const int item = item0 + u * NT;
          ok[u] = item < NITEM;
          const int it2 = ok[u] ? item : item0;
          const int cc = it2 & 3, cell = it2 >> 2;
          const int xa = cell % T::NCA, xb = cell / T::NCA;
          const int sa = T::NA ? xa + 2 : xa + 1, sb = T::NA ? xb : xb + 2;
          const double *w = W + (cc * EB + sb) * EA + sa;
#pragma unroll
          for (int k = 0; k < 5; ++k) q[k][u] = w[(k - 2) * sn];
          cnv[u] = T::NA ? xa : xb; /* cell along the normal: global f0-1+cn */
          ctv[u] = T::NA ? xb : xa; /* halo index along t1 */
          ccv[u] = cc;
        }
        gksd::weno5_edges_v<2>(q, eps, vl, vr);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          if (!ok[u]) continue;
          const int cn = cnv[u], ct = ctv[u];
          if (cn >= 1) { /* left edge = face cn-1: Qr */
            const int fh = T::NA ? ct * HA + (cn - 1) : (cn - 1) * HA + ct;
            QR[fh * 4 + ccv[u]] = vl[u];
          }
          if (cn < TN) { /* right edge = face cn: Ql */
            const int fh = T::NA ? ct * HA + cn : cn * HA + ct;
            QL[fh * 4 + ccv[u]] = vr[u];
          }
        }
      }
    }
    __syncthreads();
    if (dbg == 4) { __syncthreads(); if (tid == 0 && it + 2 < np) issue(it + 2); continue; }

    /* ---- B: collision factors, one thread per (face, side) ---- */
    for (int item = tid; item < FH * 2; item += NT) {
      const int side = item & 1, fh = item >> 1;
      const double *q = (side ? QR : QL) + fh * 4;
      const double rho = q[0], U = q[1 + DIR] * gksd::fast_rcp(rho);
      double erfz, ex;
      gksd::erf_expm2(ph.theta * U, erfz, ex);
      const double e = side ? 0.5 - 0.5 * erfz : 0.5 + 0.5 * erfz; /* erfc(+z)/2 right, erfc(-z)/2 left */
      const double x = ph.cx * ex;
      CF[fh * 4 + 2 * side] = e;
      CF[fh * 4 + 2 * side + 1] = rho * x;
    }
    __syncthreads();

    /* ---- C: Q0 and Dn on the halo faces, in place of Ql / Qr ---- */
    for (int item = tid; item < FH * 4; item += NT) {
      const int cc = item & 3, fh = item >> 2;
      const int ha = fh % HA, hb = fh / HA;
      const double el = CF[fh * 4], er = CF[fh * 4 + 2];
      double q0 = QL[item] * el + QR[item] * er;
      if (cc == 1 + DIR) q0 += CF[fh * 4 + 1] - CF[fh * 4 + 3];
      /* normal slope from the 4 cells around the face; face nf sits between slab cells nf+2, nf+3 */
      const int sa = T::NA ? ha + 3 : ha + 1, sb = T::NA ? hb : hb + 3;
      const double *w = W + (cc * EB + sb) * EA + sa;
      constexpr int sn = T::NA ? 1 : EA;
      const int nf_glob = (T::NA ? a0 + ha : b0 + hb);
      const double ihn = g.inv_hn[DIR][min(nf_glob, g.n[DIR]) + GKS_NG];
      const double dn = gksd::normal_slope(w[-2 * sn], w[-sn], w[0], w[sn]) * ihn;
      QL[item] = q0;
      QR[item] = dn;
    }
    __syncthreads();
    if (tid == 0 && it + 2 < np) issue(it + 2);   /* slab buffer (it&1) is free again */
    if (dbg == 5) continue;

    /* ---- D: tangential pass 1 -> ring slot ---- */
    {
      const int slot = it % 5;
      double *r = ring + (size_t)slot * 6 * NF * 4 + fid * 4 + c;
      constexpr int s1 = T::NA ? HA : 1;                         /* halo-face stride along t1 */
      const int fh = T::NA ? (t1_local + 2) * HA + fa : fb * HA + (t1_local + 2);
      const double *q = QL + fh * 4 + c; /* Q0 */
      const double *d = QR + fh * 4 + c; /* Dn */
      double qq[5][2], vm[2], vp[2], sm_[2], sp_[2];
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        qq[k][0] = q[(k - 2) * s1 * 4];
        qq[k][1] = d[(k - 2) * s1 * 4];
      }
      gksd::weno5_gauss_v<2>(qq, eps, vm, vp, sm_, sp_);
      r[0 * NF * 4] = vm[0];
      r[1 * NF * 4] = vp[0];
      r[2 * NF * 4] = vm[1];
      r[3 * NF * 4] = vp[1];
      r[4 * NF * 4] = sm_[0] * iw1;
      r[5 * NF * 4] = sp_[0] * iw1;
    }
    __syncthreads();
    if (dbg == 6) continue;

    if (it >= 4) {
      /* ---- E: tangential pass 2 for plane m = p-2 (ring holds planes p-4 .. p) ---- */
      const int m = p0 + it - 2;
      const double iw2 = g.inv_w[T::AXM][m + GKS_NG];
      const double *rs[5];
#pragma unroll
      for (int k = 0; k < 5; ++k) rs[k] = ring + (size_t)((it + 1 + k) % 5) * 6 * NF * 4 + fid * 4 + c;
      double *xb = XBuf + fid * T::XBS + c * 4;     /* [fld][c][g], g = 2*g1 + g2 */
#pragma unroll
      for (int fld = 0; fld < 3; ++fld) { /* Q0, Dn, Dt1: the two g1 instances of a field go together */
        double qq[5][2], vm[2], vp[2], sm_[2], sp_[2];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          qq[k][0] = rs[k][(2 * fld) * NF * 4];
          qq[k][1] = rs[k][(2 * fld + 1) * NF * 4];
        }
        gksd::weno5_gauss_v<2>(qq, eps, vm, vp, sm_, sp_);
#pragma unroll
        for (int g1 = 0; g1 < 2; ++g1) {
          xb[fld * 16 + 2 * g1] = vm[g1];
          xb[fld * 16 + 2 * g1 + 1] = vp[g1];
          if (fld == 0) {
            xb[3 * 16 + 2 * g1] = sm_[g1] * iw2;
            xb[3 * 16 + 2 * g1 + 1] = sp_[g1] * iw2;
          }
        }
      }
      __syncwarp();
      /* ---- F: flux at Gauss point gp = c of this face; sum over the 4 lanes; write ---- */
      {
        const int gp = c;
        const double *x = XBuf + fid * T::XBS + gp;
        double Q0[4], dQ[3][4], F[4], dF[4];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          Q0[cc] = x[0 * 16 + cc * 4];
          dQ[DIR][cc] = x[1 * 16 + cc * 4];
          dQ[T::AXT1][cc] = x[2 * 16 + cc * 4];
          dQ[T::AXM][cc] = x[3 * 16 + cc * 4];
        }
        gksd::gauss_point_flux<DIR, NEED_F>(Q0, dQ, ph.RT, ph.mu, F, dF);
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          if (NEED_F) {
            F[cc] += __shfl_xor_sync(0xffffffffu, F[cc], 1);
            F[cc] += __shfl_xor_sync(0xffffffffu, F[cc], 2);
          }
          dF[cc] += __shfl_xor_sync(0xffffffffu, dF[cc], 1);
          dF[cc] += __shfl_xor_sync(0xffffffffu, dF[cc], 2);
        }
        if (face_ok) {
          int pidx[3];
          pidx[0] = ga;
          pidx[T::AXB] = gb;
          pidx[T::AXM] = m;
          const long long id = g.idx(pidx[0], pidx[1], pidx[2]);
          double fsel = 0.0, dsel = 0.0;
#pragma unroll
          for (int cc = 0; cc < 4; ++cc)
            if (cc == c) {
              if (NEED_F) fsel = F[cc];
              dsel = dF[cc];
            }
          if (NEED_F) flux[c * g.FS + id] = 0.25 * fsel;
          flux[(4 + c) * g.FS + id] = 0.25 * dsel;
        }
      }
      __syncthreads();   /* the transpose buffer aliases QL/QR/CF of the next plane */
    }
  }
}

} /* namespace */

/* ---------------- host side: tensor maps and launch ---------------- */
namespace {

typedef CUresult (*encode_fn_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

/* tile shapes: x-faces 8x8 (normal along a), y/z-faces 16x4 (t1 along a, 4 faces along the normal) */
template <int DIR> struct Shape { static constexpr int TA = DIR == 0 ? 8 : 16, TB = DIR == 0 ? 8 : 4; };

template <int DIR>
bool encode_dir(encode_fn_t enc, const GksGrid &g, double *base, CUtensorMap *out) {
  using T = Tile<DIR, Shape<DIR>::TA, Shape<DIR>::TB>;
  const cuuint64_t dims[4] = {(cuuint64_t)g.P[0], (cuuint64_t)g.P[1], (cuuint64_t)g.P[2], 4};
  const cuuint64_t strides[3] = {(cuuint64_t)g.P[0] * 8, (cuuint64_t)g.P[0] * g.P[1] * 8, (cuuint64_t)g.FS * 8};
  cuuint32_t box[4] = {(cuuint32_t)T::EA, 1, 1, 4};
  box[T::AXB] = T::EB;
  const cuuint32_t es[4] = {1, 1, 1, 1};
  return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int DIR, bool NEED_F>
int launch_dir(gks_ctx *ctx, const CUtensorMap &map, double *flux) {
  constexpr int TA = Shape<DIR>::TA, TB = Shape<DIR>::TB;
  using T = Tile<DIR, TA, TB>;
  const GksGrid &g = ctx->g;
  auto kern = k_sweep_fused<DIR, NEED_F, TA, TB>;
  static bool attr_done = false;
  if (!attr_done) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES);
    attr_done = true;
  }
  const int ext_a = g.n[0] + (T::NA ? 1 : 0), ext_b = g.n[T::AXB] + (T::NA ? 0 : 1), n2 = g.n[T::AXM];
  const int ga = (ext_a + TA - 1) / TA, gb = (ext_b + TB - 1) / TB;
  /* chunks along the marched axis: enough CTAs for ~6 waves of 2 CTAs/SM, each at least 32 planes */
  long long cols = (long long)ga * gb;
  int nch = (int)((1776 + cols - 1) / cols);
  const int maxch = n2 / 32 > 1 ? n2 / 32 : 1;
  if (nch > maxch) nch = maxch;
  if (nch < 1) nch = 1;
  const int MC = (n2 + nch - 1) / nch;
  nch = (n2 + MC - 1) / MC;
  kern<<<dim3(ga, gb, nch), T::NT, T::SMEM_BYTES, ctx->stream>>>(map, g, ctx->ph, flux, MC, getenv("GKS_DBG") ? atoi(getenv("GKS_DBG")) : 0);
  return 1;
}

} /* namespace */

bool gks_fused_init(gks_ctx *ctx) {
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn ||
      q != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  encode_fn_t enc = (encode_fn_t)fn;
  double *bases[2] = {ctx->Wn, ctx->Ws};
  for (int b = 0; b < 2; ++b) {
    CUtensorMap *m = reinterpret_cast<CUtensorMap *>(ctx->tmaps[b][0]);
    if (!encode_dir<0>(enc, ctx->g, bases[b], m)) return false;
    if (!encode_dir<1>(enc, ctx->g, bases[b], reinterpret_cast<CUtensorMap *>(ctx->tmaps[b][1]))) return false;
    if (!encode_dir<2>(enc, ctx->g, bases[b], reinterpret_cast<CUtensorMap *>(ctx->tmaps[b][2]))) return false;
  }
  return true;
}

int gks_launch_sweep_fused(gks_ctx *ctx, int dir, int which, double *flux, bool need_F) {
  const CUtensorMap &m = *reinterpret_cast<const CUtensorMap *>(ctx->tmaps[which][dir]);
  switch (dir) {
    case 0: return need_F ? launch_dir<0, true>(ctx, m, flux) : launch_dir<0, false>(ctx, m, flux);
    case 1: return need_F ? launch_dir<1, true>(ctx, m, flux) : launch_dir<1, false>(ctx, m, flux);
    default: return need_F ? launch_dir<2, true>(ctx, m, flux) : launch_dir<2, false>(ctx, m, flux);
  }
}
