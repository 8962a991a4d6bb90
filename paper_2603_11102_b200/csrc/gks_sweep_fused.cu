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

/* named barriers (bar.sync / bar.arrive with a thread count): producer <-> consumer hand-over */
__device__ __forceinline__ void bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
enum { BAR_PROD = 1, BAR_FULL0 = 2, BAR_EMPTY0 = 4 }; /* FULL0/FULL1 = 2,3; EMPTY0/EMPTY1 = 4,5; 0 = __syncthreads */

/* ---------------- compile-time geometry of a tile ---------------- */
template <int DIR, int TA, int TB>
struct Tile {
  static constexpr bool NA = (DIR == 0);            /* normal along a */
  static constexpr int TN = NA ? TA : TB;           /* faces along the normal */
  static constexpr int T1 = NA ? TB : TA;           /* faces along t1 */
  static constexpr int NF = TA * TB;                /* faces per CTA and plane */
  static constexpr int NC = NF * 4;                 /* consumer threads (4 per face) */
  static constexpr int NP = NC / 2;                 /* producer threads */
  static constexpr int NT = NC + NP;                /* threads per CTA */
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
  /* shared memory carve (doubles) */
  static constexpr int OFF_W = 0;                          /* 2 slabs (TMA destinations) */
  static constexpr int OFF_S = OFF_W + 2 * WSLAB_PAD;      /* producer staging: QL|QR [2][FH][4] */
  static constexpr int OFF_CF = OFF_S + 2 * FH * 4;        /* collision factors [FH][4] */
  static constexpr int OFF_Q = OFF_CF + FH * 4;            /* 2 hand-over buffers, each Q0|Dn [2][FH][4] */
  static constexpr int OFF_XB = OFF_Q + 2 * 2 * FH * 4;    /* transpose buffer, 64 doubles per face, XOR-swizzled */
  static constexpr int OFF_RING = OFF_XB + NF * 64;        /* 4-plane ring of pass-1 results [4][6][NF][4] */
  static constexpr int RING = 4 * 6 * NF * 4;
  static constexpr int OFF_BAR = OFF_RING + RING;
  static constexpr size_t SMEM_BYTES = (size_t)(OFF_BAR + 2) * 8;
  static constexpr int CTAS_PER_SM = (2 * (SMEM_BYTES + 1024) <= 233472 && 2 * NT <= 1024) ? 2 : 1;
  static_assert(SMEM_BYTES + 1024 <= 233472, "the CTA must fit in shared memory");
  static_assert(NC % 32 == 0 && NP % 32 == 0, "whole warps per role");
};

/* one contiguous run of marched planes of one tile column: output planes [mb, mb+len) */
struct Seg {
  int a0, b0, p0, np;   /* tile origin; first staged plane (mb-2); planes to stage (len+4) */
};

/*
 * Persistent and warp-specialised.  The work of one launch is the list of (tile column, marched plane)
 * pairs in column-major order; CTA b owns the contiguous range [b*PPC, (b+1)*PPC) of it, i.e. a few
 * column segments, so that all CTAs finish together (no wave quantisation).  Threads [0, NC) are
 * CONSUMERS (4 per face: tangential passes + flux), threads [NC, NC+NP) are PRODUCERS (normal
 * reconstruction + collision on the halo faces, one to two planes ahead).  The two groups meet only at
 * the named barriers FULL/EMPTY of the double-buffered Q0|Dn hand-over.
 */
template <int DIR, bool NEED_F, int TA, int TB>
__global__ void __launch_bounds__(Tile<DIR, TA, TB>::NT, Tile<DIR, TA, TB>::CTAS_PER_SM)
    k_sweep_fused(const __grid_constant__ CUtensorMap tmap, GksGrid g, GksPhys ph, double *__restrict__ flux,
                  int ncol_a, long long total, long long PPC) {
  using T = Tile<DIR, TA, TB>;
  constexpr int TN = T::TN, NF = T::NF, NC = T::NC, NP = T::NP, NT = T::NT, EA = T::EA, EB = T::EB, HA = T::HA,
                FH = T::FH;
  extern __shared__ __align__(128) double sm[];
  double *const Wp = sm + T::OFF_W;
  double *const QLs = sm + T::OFF_S;           /* [FH][4] */
  double *const QRs = QLs + FH * 4;            /* [FH][4] */
  double *const CF = sm + T::OFF_CF;           /* [FH][4]: el, rho_l*xl, er, rho_r*xr */
  double *const Qb = sm + T::OFF_Q;            /* [2][2][FH][4] */
  double *const XBuf = sm + T::OFF_XB;
  double *const ring = sm + T::OFF_RING;       /* [4][6][NF][4] */
  uint64_t *const bar = reinterpret_cast<uint64_t *>(sm + T::OFF_BAR);

  const int tid = threadIdx.x;
  const int n2 = g.n[T::AXM];
  const double eps = ph.weno_eps;
  long long L0 = (long long)blockIdx.x * PPC, L1 = L0 + PPC;
  if (L0 > total) L0 = total;
  if (L1 > total) L1 = total;
  auto seg_at = [&](long long l) {
    const int col = (int)(l / n2), mb = (int)(l - (long long)col * n2);
    const long long left = L1 - l;
    const int len = (int)(left < (long long)(n2 - mb) ? left : (long long)(n2 - mb));
    Seg s;
    s.a0 = (col % ncol_a) * TA;
    s.b0 = (col / ncol_a) * TB;
    s.p0 = mb - 2;
    s.np = len + 4;
    return s;
  };
  int planes_total = 0;                        /* staged planes of this CTA over all its segments */
  for (long long l = L0; l < L1;) {
    const Seg s = seg_at(l);
    planes_total += s.np;
    l += s.np - 4;
  }

  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    fence_barrier_init();
  }
  __syncthreads();

  if (tid >= NC) {
    /* ======================= PRODUCER ======================= */
    const int pt = tid - NC;
    /* TMA prefetch cursor (used by pt == 0 only): next plane to request and its running number */
    long long lpf = L0;
    Seg spf = seg_at(L0 < L1 ? L0 : 0);
    int itpf = 0, gpf = 0;
    auto issue_next = [&]() {
      if (lpf >= L1) return;
      uint64_t *b = &bar[gpf & 1];
      double *dst = Wp + (gpf & 1) * T::WSLAB_PAD;
      const int pm = spf.p0 + itpf + GKS_NG;   /* padded index space: cell -3 <-> 0 */
      const int ca0 = spf.a0, cb0 = T::NA ? spf.b0 + 1 : spf.b0;
      mbar_expect_tx(b, T::WSLAB * 8);
      if (DIR == 2) tma_load_4d(dst, &tmap, b, ca0, pm, cb0, 0);
      else tma_load_4d(dst, &tmap, b, ca0, cb0, pm, 0);
      ++gpf;
      if (++itpf == spf.np) {
        lpf += spf.np - 4;
        itpf = 0;
        if (lpf < L1) spf = seg_at(lpf);
      }
    };
    if (pt == 0) {
      issue_next();
      issue_next();
    }
    constexpr int sn = T::NA ? 1 : EA;         /* slab stride along the normal */
    int gi = 0;                                /* running plane number: selects slab, hand-over buffer, parities */
    for (long long l = L0; l < L1;) {
      const Seg s = seg_at(l);
      l += s.np - 4;
      for (int it = 0; it < s.np; ++it, ++gi) {
        const double *W = Wp + (gi & 1) * T::WSLAB_PAD;
        mbar_wait(&bar[gi & 1], (gi >> 1) & 1);

        /* ---- A: both edge values of each cell, per component (one smoothness-indicator set serves the
         *         face on either side); two cells per thread at a time, a single one in the ragged tail ---- */
        {
          constexpr int NITEM = T::NCA * T::NCB * 4;
          auto locate = [&](int item, const double *&w, int &cn, int &ct, int &cc) {
            cc = item & 3;
            const int cell = item >> 2;
            const int xa = cell % T::NCA, xb = cell / T::NCA;
            const int sa = T::NA ? xa + 2 : xa + 1, sb = T::NA ? xb : xb + 2;
            w = W + (cc * EB + sb) * EA + sa;
            cn = T::NA ? xa : xb; /* cell along the normal: global f0-1+cn */
            ct = T::NA ? xb : xa; /* halo index along t1 */
          };
          auto store = [&](int cn, int ct, int cc, double vl, double vr) {
            if (cn >= 1) { /* left edge = face cn-1: Qr */
              const int fh = T::NA ? ct * HA + (cn - 1) : (cn - 1) * HA + ct;
              QRs[fh * 4 + cc] = vl;
            }
            if (cn < TN) { /* right edge = face cn: Ql */
              const int fh = T::NA ? ct * HA + cn : cn * HA + ct;
              QLs[fh * 4 + cc] = vr;
            }
          };
          int item0 = pt;
          for (; item0 + NP < NITEM; item0 += 2 * NP) {
            double q[5][2], vl[2], vr[2];
            int cnv[2], ctv[2], ccv[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              const double *w;
              locate(item0 + u * NP, w, cnv[u], ctv[u], ccv[u]);
#pragma unroll
              for (int k = 0; k < 5; ++k) q[k][u] = w[(k - 2) * sn];
            }
            gksd::weno5_edges_v<2>(q, eps, vl, vr);
#pragma unroll
            for (int u = 0; u < 2; ++u) store(cnv[u], ctv[u], ccv[u], vl[u], vr[u]);
          }
          if (item0 < NITEM) {
            double q[5][1], vl[1], vr[1];
            int cn, ct, cc;
            const double *w;
            locate(item0, w, cn, ct, cc);
#pragma unroll
            for (int k = 0; k < 5; ++k) q[k][0] = w[(k - 2) * sn];
            gksd::weno5_edges_v<1>(q, eps, vl, vr);
            store(cn, ct, cc, vl[0], vr[0]);
          }
        }
        bar_sync(BAR_PROD, NP);

        /* ---- B: collision factors (S4), one thread per (face, side), two independent chains at a time ---- */
        for (int item0 = pt; item0 < FH * 2; item0 += 2 * NP) {
          double z[2], rho[2], erfz[2], ex[2], ir[2];
          int at[2];
          bool ok[2];
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            const int item = item0 + u * NP;
            ok[u] = item < FH * 2;
            const int it2 = ok[u] ? item : item0;
            const int side = it2 & 1, fh = it2 >> 1;
            const double *q = (side ? QRs : QLs) + fh * 4;
            rho[u] = q[0];
            z[u] = q[1 + DIR];
            at[u] = fh * 4 + 2 * side;
          }
          gksd::fast_rcp_v<2>(rho, ir);
#pragma unroll
          for (int u = 0; u < 2; ++u) z[u] = ph.theta * (z[u] * ir[u]);
          gksd::erf_expm2_v<2>(z, erfz, ex);
#pragma unroll
          for (int u = 0; u < 2; ++u) {
            if (!ok[u]) continue;
            const double h = (at[u] & 2) ? -0.5 : 0.5;   /* erfc(+z)/2 right, erfc(-z)/2 left */
            CF[at[u]] = fma(h, erfz[u], 0.5);
            CF[at[u] + 1] = rho[u] * (ph.cx * ex[u]);
          }
        }
        bar_sync(BAR_PROD, NP);

        /* the hand-over buffer (gi & 1) was last read by pass 1 of plane gi-2 */
        if (gi >= 2) bar_sync(BAR_EMPTY0 + (gi & 1), NT);

        /* ---- C: Q0 and Dn on the halo faces -> hand-over buffer ---- */
        {
          double *const Q0o = Qb + (gi & 1) * (2 * FH * 4);
          double *const Dno = Q0o + FH * 4;
#pragma unroll 2
          for (int item = pt; item < FH * 4; item += NP) {
            const int cc = item & 3, fh = item >> 2;
            const int ha = fh % HA, hb = fh / HA;
            const double el = CF[fh * 4], er = CF[fh * 4 + 2];
            double q0 = QLs[item] * el + QRs[item] * er;
            if (cc == 1 + DIR) q0 += CF[fh * 4 + 1] - CF[fh * 4 + 3];
            /* normal slope from the 4 cells around the face; face nf sits between slab cells nf+2, nf+3 */
            const int sa = T::NA ? ha + 3 : ha + 1, sb = T::NA ? hb : hb + 3;
            const double *w = W + (cc * EB + sb) * EA + sa;
            const int nf_glob = (T::NA ? s.a0 + ha : s.b0 + hb);
            const double ihn = g.inv_hn[DIR][min(nf_glob, g.n[DIR]) + GKS_NG];
            Q0o[item] = q0;
            Dno[item] = gksd::normal_slope(w[-2 * sn], w[-sn], w[0], w[sn]) * ihn;
          }
        }
        __threadfence_block();
        bar_arrive(BAR_FULL0 + (gi & 1), NT);
        bar_sync(BAR_PROD, NP);                        /* slab (gi & 1) and the staging arrays are free again */
        if (pt == 0) issue_next();                     /* plane gi+2 (possibly of the next segment) */
      }
    }
    return;
  }

  /* ======================= CONSUMER ======================= */
  const int c = tid & 3, fid = tid >> 2;
  const int fa = fid % TA, fb = fid / TA;       /* a fastest: coalesced output */
  const int n_a = g.n[0] + (T::NA ? 1 : 0), n_b = g.n[T::AXB] + (T::NA ? 0 : 1);
  const int t1_local = T::NA ? fb : fa;
  constexpr int s1 = T::NA ? HA : 1;                         /* halo-face stride along t1 */
  const int fh0 = T::NA ? (t1_local + 2) * HA + fa : fb * HA + (t1_local + 2);
  double *const rg = ring + fid * 4 + c;        /* this thread's private column of the ring */
  constexpr int RS = 6 * NF * 4, RF = NF * 4;   /* ring strides: plane slot, field */
  /* transpose buffer: element (field, component cc, Gauss point gq) of face fid lives at
   * fid*64 + field*16 + 4*(cc ^ (fid&3)) + (gq ^ cc): conflict-free for the component-major writes
   * and for the Gauss-point-major reads of a half warp */
  double *const xw = XBuf + fid * 64 + 4 * (c ^ (fid & 3));                /* writes: + field*16 + (gq ^ c) */
  const double *const xr = XBuf + fid * 64;                                 /* reads:  + field*16 + ro[cc] */
  int ro[4];
#pragma unroll
  for (int cc = 0; cc < 4; ++cc) ro[cc] = 4 * (cc ^ (fid & 3)) + (c ^ cc);

  int gi = 0;
  for (long long l = L0; l < L1;) {
    const Seg s = seg_at(l);
    l += s.np - 4;
    const int ga = s.a0 + fa, gb = s.b0 + fb;     /* global indices along a and b */
    const bool face_ok = ga < n_a && gb < n_b;
    const int t1_glob = T::NA ? gb : ga;
    const double iw1 = g.inv_w[T::AXT1][min(t1_glob, g.n[T::AXT1] - 1) + GKS_NG];
    for (int it = 0; it < s.np; ++it, ++gi) {
      bar_sync(BAR_FULL0 + (gi & 1), NT);
      /* ---- D: tangential pass 1 (along t1) on Q0 and Dn of plane it ---- */
      double d6[6];
      {
        const double *q = Qb + (gi & 1) * (2 * FH * 4) + fh0 * 4 + c; /* Q0 */
        const double *d = q + FH * 4;                                 /* Dn */
        double qq[5][2], vm[2], vp[2], sm_[2], sp_[2];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          qq[k][0] = q[(k - 2) * s1 * 4];
          qq[k][1] = d[(k - 2) * s1 * 4];
        }
        gksd::weno5_gauss_v<2>(qq, eps, vm, vp, sm_, sp_);
        d6[0] = vm[0];
        d6[1] = vp[0];
        d6[2] = vm[1];
        d6[3] = vp[1];
        d6[4] = sm_[0] * iw1;
        d6[5] = sp_[0] * iw1;
      }
      /* the loaded values have been consumed: the hand-over buffer may be refilled (plane gi+2) */
      if (gi + 2 < planes_total) bar_arrive(BAR_EMPTY0 + (gi & 1), NT);

    double *const rnew = rg + (it & 3) * RS;     /* slot of plane it-4, dead once pass 2 below has read it */
    if (it < 4) {
#pragma unroll
      for (int v = 0; v < 6; ++v) rnew[v * RF] = d6[v];
      continue;
    }
    /* ---- E: tangential pass 2 (along t2, the marched axis) for plane m = it-2; the ring holds planes
     *         it-4 .. it-1 (plane it-4+k in slot (it+k)&3), plane it comes straight from d6 ---- */
    const int m = s.p0 + it - 2;
    const double iw2 = g.inv_w[T::AXM][m + GKS_NG];
    const double *rs[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) rs[k] = rg + ((it + k) & 3) * RS;
#pragma unroll
    for (int fld = 0; fld < 3; ++fld) { /* Q0, Dn, Dt1: the two g1 instances of a field go together */
      double qq[5][2], vm[2], vp[2], sm_[2], sp_[2];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        qq[k][0] = rs[k][(2 * fld) * RF];
        qq[k][1] = rs[k][(2 * fld + 1) * RF];
      }
      qq[4][0] = d6[2 * fld];
      qq[4][1] = d6[2 * fld + 1];
      rnew[(2 * fld) * RF] = d6[2 * fld];          /* rs[0] aliases rnew: stored after the loads above */
      rnew[(2 * fld + 1) * RF] = d6[2 * fld + 1];
      gksd::weno5_gauss_v<2>(qq, eps, vm, vp, sm_, sp_);
#pragma unroll
      for (int g1 = 0; g1 < 2; ++g1) {            /* Gauss point gq = 2*g1 + g2 */
        xw[fld * 16 + ((2 * g1) ^ c)] = vm[g1];
        xw[fld * 16 + ((2 * g1 + 1) ^ c)] = vp[g1];
        if (fld == 0) {
          xw[3 * 16 + ((2 * g1) ^ c)] = sm_[g1] * iw2;
          xw[3 * 16 + ((2 * g1 + 1) ^ c)] = sp_[g1] * iw2;
        }
      }
    }
    __syncwarp();
    /* ---- F: flux at Gauss point gp = c of this face; sum over the 4 lanes; write ---- */
    {
      double Q0[4], dQ[3][4], F[4], dF[4];
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {
        Q0[cc] = xr[0 * 16 + ro[cc]];
        dQ[DIR][cc] = xr[1 * 16 + ro[cc]];
        dQ[T::AXT1][cc] = xr[2 * 16 + ro[cc]];
        dQ[T::AXM][cc] = xr[3 * 16 + ro[cc]];
      }
      gksd::gauss_point_flux<DIR, NEED_F>(Q0, dQ, ph.RT, ph.mu, F, dF);
      __syncwarp();                               /* every lane has consumed its reads: the buffer is reusable */
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
  }
  }
}

} /* namespace */

/* ---------------- host side: tensor maps and launch ---------------- */
namespace {

typedef CUresult (*encode_fn_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

/* tile shapes: 128 faces per CTA; x-faces 8 (normal, along a) x 16 (t1), y/z-faces 16 (t1, along a) x 8 (normal) */
template <int DIR> struct Shape { static constexpr int TA = DIR == 0 ? 8 : 16, TB = DIR == 0 ? 16 : 8; };

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
  /* persistent CTAs: the (column, plane) list is cut into equal contiguous ranges, one per resident CTA;
     a range shorter than 8 planes is not worth its 4 priming planes */
  const long long total = (long long)ga * gb * n2;
  const long long slots = (long long)ctx->num_sms * T::CTAS_PER_SM;
  long long PPC = (total + slots - 1) / slots;
  if (PPC < 8) PPC = 8;
  const int nblk = (int)((total + PPC - 1) / PPC);
  kern<<<nblk, T::NT, T::SMEM_BYTES, ctx->stream>>>(map, g, ctx->ph, flux, ga, total, PPC);
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
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
    cudaGetLastError();
    return false;
  }
  ctx->num_sms = nsm;
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
