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
 * Per marched plane the CTA runs the stages
 *   A   both WENO5 edge values of every cell (one smoothness-indicator set per cell serves the face on
 *       either side) and the normal slope Dn, from the W halo slab that TMA staged in shared memory,
 *   BC  the collision Q0(QL, QR) on the TN x (T1+4) halo faces (four lanes per face split sides and series),
 *   D   tangential pass 1 (along t1): 6 values per (face, component),
 *   EF  tangential pass 2 (along t2) for the plane two behind, out of a thread-private 4-plane ring in shared
 *       memory (the newest plane comes from D's registers), the four Gauss-point fluxes, the face average
 *       F, dF/dt to HBM,
 * software-pipelined over three planes per iteration (k_sweep_fused's comment has the schedule, the
 * persistent wave-major work distribution and the single split mbarrier hand-over per iteration).
 * Thread mapping: 4 threads per face.  In A-E thread (face, c) owns component c (WENO is component-wise);
 * in F thread (face, g) owns Gauss point g (the flux couples all components); the 4x4 transpose goes
 * through a swizzled warp-private buffer and needs only __syncwarp.
 * The W slab of the next plane is fetched by TMA (cp.async.bulk.tensor) one iteration ahead: 2 slab buffers,
 * one elected thread issues, the bytes are expected on the iteration barrier itself (one wait per iteration);
 * cells beyond the padded array (overhanging tiles) are filled with NaN, which takes the short path
 * everywhere and is never stored.
 *
 * Roofline: fp64-ALU bound (about 4.7 kflop per face against 32 B read + 64 B written per face).
 */
#include <cuda.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "gks_internal.h"
#include "gks_math.cuh"

#ifndef GKS_MIN_PPC
#define GKS_MIN_PPC 2   /* remainder columns: fewest output planes per CTA (idle SMs are free; measured on C1-C3) */
#endif
#ifndef GKS_NF
#define GKS_NF 128      /* faces per CTA tile: 128 = one CTA of 512 threads per SM; 64 = two CTAs of 256 threads per SM */
#endif
#define GKS_CTAS_PER_SM (128 / GKS_NF)
#ifndef GKS_XHALF
#define GKS_XHALF 1   /* 1: the 4x4 transposes go through the warp-private buffer two fields at a time (32 doubles per face) */
#endif
#ifndef GKS_E_WIDTH
#define GKS_E_WIDTH 3   /* pass-2 evaluations written side by side: 2, 3 or 6 (measured: 3 is best for all three tile shapes) */
#endif

/* Phase timeline (build with -DGKS_TRACE, `python -m paper_2603_11102_b200.trace`): every warp of CTA 0 accumulates the
 * clock64 ticks it spends in each phase of the plane loop; gks_debug_trace reads them back.  Off in the product. */
#ifdef GKS_TRACE
__device__ unsigned long long gks_trace_buf[32 * 8];   /* [warp][phase] */
#define TR_DECL unsigned long long tr_[8] = {0, 0, 0, 0, 0, 0, 0, 0}; long long tr_t = clock64();
#define TR(k) { const long long n_ = clock64(); tr_[k] += n_ - tr_t; tr_t = n_; }
#define TR_DUMP if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) { for (int q_ = 0; q_ < 8; ++q_) gks_trace_buf[(threadIdx.x >> 5) * 8 + q_] = tr_[q_]; }
#else
#define TR_DECL
#define TR(k)
#define TR_DUMP
#endif

namespace {

#ifndef GKS_FUSE_BCD
#define GKS_FUSE_BCD 1   /* 0: stages separate; 1: BC + D one straight-line block; 2: that for y- and z-faces only;
                            3: A + BC + D one block */
#endif

/* ---------------- PTX helpers: mbarrier + TMA ---------------- */
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
/* raises the transaction count of the current phase without arriving */
__device__ __forceinline__ void mbar_expect_tx_only(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  /* try_wait suspends the warp in hardware up to the time hint (ns) instead of spinning on issue slots */
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n"
      "@P1 bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity), "r"(0x989680)
      : "memory");
}
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

/* one arrival per warp, by lane 0, predicated inside the instruction (no divergent branch around it) */
__device__ __forceinline__ void mbar_arrive_lane0(uint64_t *bar, int lane) {
  asm volatile(
      "{\n"
      ".reg .pred P2;\n"
      "setp.eq.s32 P2, %1, 0;\n"
      "@P2 mbarrier.arrive.shared::cta.b64 _, [%0];\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(lane)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

/* ---------------- compile-time geometry of a tile ---------------- */
template <int DIR, int TA, int TB>
struct Tile {
  static constexpr bool NA = (DIR == 0);            /* normal along a */
  static constexpr int TN = NA ? TA : TB;           /* faces along the normal */
  static constexpr int T1 = NA ? TB : TA;           /* faces along t1 */
  static constexpr int NF = TA * TB;                /* faces per CTA and plane */
  static constexpr int NT = NF * 4;                 /* threads per CTA (4 per face) */
  static constexpr int NW = NT / 32;                /* warps */
  static constexpr int CA = NA ? TN + 5 : T1 + 5;   /* cells of the W slab along a / b; the slab always starts at
                                                       cell a0-3: TMA needs a 16-byte aligned box start (even index) */
  static constexpr int CB = NA ? T1 + 4 : TN + 5;
  static constexpr int EA = (CA + 1) & ~1;          /* TMA box: inner extent even (16-byte rows) */
  /* rows of the box: padded until the component stride EB*EA is 4 or 12 (mod 16 doubles), which makes the
     (component, cell) lanes of stage A hit 16 different bank pairs */
  static constexpr int eb_pad(int cb, int ea) {
    int eb = cb;
    while ((eb * ea) % 16 != 4 && (eb * ea) % 16 != 12) ++eb;
    return eb;
  }
  static constexpr int EB = eb_pad(CB, EA);
  static constexpr int HA = NA ? TN : T1 + 4;       /* halo-face box (faces needed by pass 1) */
  static constexpr int HB = NA ? T1 + 4 : TN;
  static constexpr int FH = HA * HB;
  static constexpr int NCA = NA ? TN + 1 : T1 + 4;  /* cells reconstructed in stage A */
  static constexpr int NCB = NA ? T1 + 4 : TN + 1;
  static constexpr int AXB = DIR == 2 ? 2 : 1;      /* global axis of b */
  static constexpr int AXM = DIR == 2 ? 1 : 2;      /* global axis marched (= t2) */
  static constexpr int AXT1 = DIR == 0 ? 1 : 0;
  static constexpr int WSLAB = 4 * EB * EA;         /* doubles per staged slab */
  static constexpr int WSLAB_PAD = (WSLAB + 15) & ~15;
  /* shared memory carve (doubles) */
  static constexpr int OFF_W = 0;                          /* 2 slabs (TMA destinations) */
  static constexpr int SBUF = 3 * FH * 4 + 8;              /* one stage buffer: QL->Q0 | QR | Dn, each [FH][4]; QR and Dn
                                                              are shifted by 2 and 4 doubles against bank conflicts
                                                              between the QL and QR rows of a face (stage BC) */
  static constexpr int OFF_S = OFF_W + 2 * WSLAB_PAD;      /* 3 stage buffers (plane j lives in buffer j % 3) */
  static constexpr int OFF_XB = OFF_S + 3 * SBUF;          /* transpose buffer, 64 doubles per face, XOR-swizzled */
  static constexpr int XF = GKS_XHALF ? 32 : 64;           /* doubles of the transpose buffer per face */
  static constexpr int OFF_RING = OFF_XB + NF * XF;        /* 4-plane ring of pass-1 results [4][6][NF][4] */
  static constexpr int RING = 4 * 6 * NF * 4;
  static constexpr int OFF_BAR = OFF_RING + RING;          /* mbarriers: [0] first slab, [2] iteration barrier */
  static constexpr int OFF_CF = OFF_BAR + 4;               /* series coefficients of the collision stage [2][8] */
  static constexpr size_t SMEM_BYTES = (size_t)(OFF_CF + 16) * 8;
  static_assert((SMEM_BYTES + 1024) * GKS_CTAS_PER_SM <= 233472, "the CTA(s) must fit in shared memory");
  static_assert(NT <= 1024 && NT % 32 == 0 && (NT & (NT - 1)) == 0, "whole warps, power of two");
};

/* one contiguous run of marched planes of one tile column: output planes [mb, mb+len) */
struct Seg {
  int a0, b0, p0, np;   /* tile origin; first staged plane (mb-2); planes to stage (len+4) */
};

/*
 * Persistent, symmetric and software-pipelined.  The work of one launch is the list of (tile column,
 * marched plane) pairs.  With G CTAs and C columns, every CTA first marches floor(C/G) whole columns
 * (CTA b: columns b, b+G, ...: neighbouring columns move through the same planes together, so the halo
 * of a slab is read from L2, not from HBM); the planes of the remaining C mod G columns are cut into G
 * equal contiguous ranges (a few column segments per CTA, each costs 4 priming planes), so that all
 * CTAs finish together.
 *
 * Every warp runs the same program.  Iteration i works on three different staged planes at once:
 *     stage A  on plane i    : normal WENO edge values QL, QR and the normal slope Dn      -> S[i % 3]
 *     stage BC on plane i-1  : collision Q0(QL, QR), in place                              -> S[(i-1) % 3]
 *     stage D  on plane i-2  : tangential pass 1 (reads Q0, Dn of the t1 neighbours)       <- S[(i-2) % 3]
 *     stage EF on plane i-2  : tangential pass 2 out of the thread-private ring, flux, store
 * A, BC and D touch three different buffers, so an iteration needs ONE CTA-wide hand-over, and that one
 * is split: a warp arrives on the iteration mbarrier after A, BC, D and waits for it only at the top of
 * the next iteration, after its EF (about half of the iteration's arithmetic) - warps may drift by half
 * an iteration without anyone waiting.  A thread's own BC item and its D item are written as one
 * straight-line block (GKS_FUSE_BCD): BC's serial chain issues in the shadow of D's arithmetic.
 */
template <int DIR, bool NEED_F, bool LIN, int TA, int TB, int UMASK>
__global__ void __launch_bounds__(Tile<DIR, TA, TB>::NT, GKS_CTAS_PER_SM)
    k_sweep_fused(const __grid_constant__ CUtensorMap tmap, GksGrid g, GksPhys ph, double *__restrict__ flux,
                  int ncol_a, int nfull, long long rem, long long PPC, int ta0, int tlen0, int ta1, int n_a, int n_b) {
  using T = Tile<DIR, TA, TB>;
  /* UMASK: bit a set = axis a is KNOWN to be uniform (its metric factors are kernel parameters, no table code); the
     instantiations are 7 (all three), 5 (x and z: the channel, stretched between its walls) and 0 (nothing known) */
  constexpr bool UN_N = (UMASK >> DIR) & 1, UN_T1 = (UMASK >> T::AXT1) & 1, UN_M = (UMASK >> T::AXM) & 1;
  constexpr int TN = T::TN, NF = T::NF, NT = T::NT, EA = T::EA, EB = T::EB, HA = T::HA, FH = T::FH;
  constexpr bool FUSE_BCD = GKS_FUSE_BCD == 1 || GKS_FUSE_BCD == 3 || (GKS_FUSE_BCD == 2 && DIR != 0);
  constexpr bool FUSE_A = GKS_FUSE_BCD == 3;
  constexpr bool D_FIRST = DIR == 0;   /* source order of D and BC inside the fused block: measured, x-faces 0.7 % */
  extern __shared__ __align__(128) double sm[];
  double *const Wp = sm + T::OFF_W;
  double *const Sb = sm + T::OFF_S;            /* [3][3][FH][4] */
  double *const XBuf = sm + T::OFF_XB;
  double *const ring = sm + T::OFF_RING;       /* [4][6][NF][4] */
  uint64_t *const bar = reinterpret_cast<uint64_t *>(sm + T::OFF_BAR);   /* [0] slab of plane 0; [2] iteration hand-over + slabs */

  const int tid = threadIdx.x;
  const int n2 = g.n[T::AXM];
  const double eps = ph.weno_eps4;   /* 4 x the WENO epsilon (gks_math.cuh) */
  /* This CTA's plane list, addressed by a private index v in [0, L1):
   *   v <  nfull*n2 : whole columns blockIdx.x + gridDim.x*w, w = v / n2 - all CTAs march neighbouring
   *                   columns through the same planes at the same time (halo slabs are shared in L2);
   *   v >= nfull*n2 : this CTA's share [r0, r1) of the planes of the remaining columns, column-major. */
  const long long full = (long long)nfull * n2;
  const long long r0 = (long long)blockIdx.x * PPC < rem ? (long long)blockIdx.x * PPC : rem;
  const long long r1 = r0 + PPC < rem ? r0 + PPC : rem;
  const long long L0 = 0, L1 = full + (r1 - r0);
  if (L0 >= L1) return;
  auto seg_at = [&](long long v) {
    int col, mb, len;
    if (v < full) {
      const int w = (int)(v / n2);
      col = (int)blockIdx.x + (int)gridDim.x * w;
      mb = (int)(v - (long long)w * n2);
      len = n2 - mb;
    } else {
      const long long r = r0 + (v - full);
      const int cr = (int)(r / n2);
      col = nfull * (int)gridDim.x + cr;
      mb = (int)(r - (long long)cr * n2);
      const long long left = r1 - r;
      len = (int)(left < (long long)(n2 - mb) ? left : (long long)(n2 - mb));
    }
    Seg s;
    /* the launch covers the tiles [ta0, ta0 + tlen0) and [ta1, ta1 + ncol_a - tlen0) along a (all of them, or the
       interior, or the two rims next to cut faces: gks_step_begin_part) */
    const int ia = col % ncol_a;
    s.a0 = (ia + (ia < tlen0 ? ta0 : ta1)) * TA;      /* ta1: already less tlen0 */
    s.b0 = (col / ncol_a) * TB;
    s.p0 = mb - 2;
    s.np = len + 4;
    return s;
  };
  int J = 0;                                   /* staged planes of this CTA over all its segments */
  for (long long l = L0; l < L1;) {
    const Seg s = seg_at(l);
    J += s.np;
    l += s.np - 4;
  }
  /* three cursors walk the same plane list: TMA (plane i+1), stage A (plane i), stages D/EF (plane i-2) */
  struct Cur {
    long long l;
    Seg s;
    int it;
  };
  auto cur_next = [&](Cur &c) {
    if (++c.it == c.s.np) {
      c.l += c.s.np - 4;
      c.it = 0;
      if (c.l < L1) c.s = seg_at(c.l);
    }
  };
  Cur cT, cD;
  cT.l = L0; cT.s = seg_at(L0); cT.it = 0;
  cD = cT;
  int n0_next = T::NA ? cT.s.a0 : cT.s.b0;     /* stage A: normal face 0 of the tile of the plane it works on next */

  /* stage BC: the 8 Maclaurin coefficients of erf (lanes with func = 0) and of exp(-z^2) (func = 1) sit in shared memory;
     a lane reads its own set every plane (two addresses per warp: one wavefront) - cheaper than what the compiler makes
     of per-thread coefficients, 8 LDC.64 + 16 predicated LDC per plane (measured 890 -> 895) */
  if (tid < 16) {
    double tmp[8];
    gksd::series_coefficients(tid >> 3, tmp);
    double v = tmp[0];
#pragma unroll
    for (int n = 1; n < 8; ++n) v = (tid & 7) == n ? tmp[n] : v;
    sm[T::OFF_CF + tid] = v;
  }
  const double *const cfs = sm + T::OFF_CF + ((tid & 3) >> 1) * 8;   /* its items all have cc = tid & 3 */
  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[2], T::NW);
    fence_barrier_init();
  }
  /* everything above ran in the shadow of the previous kernel's tail; global memory from here on.  The next kernel
     is released when this CTA is done (end of the kernel): released at the start, its CTAs would queue for the whole
     sweep (measured: slower) */
  asm volatile("griddepcontrol.wait;" ::: "memory");
  __syncthreads();

  auto issue = [&](const Cur &c, int j) {       /* request staged plane j (described by cursor c) */
    uint64_t *b = j == 0 ? &bar[0] : &bar[2];     /* see the hand-over at the top of the loop */
    double *dst = Wp + (j & 1) * T::WSLAB_PAD;
    const int pm = c.s.p0 + c.it + GKS_NG;      /* padded index space: cell -3 <-> 0 */
    const int ca0 = c.s.a0, cb0 = T::NA ? c.s.b0 + 1 : c.s.b0;
    if (j == 0) mbar_expect_tx(b, T::WSLAB * 8);
    else mbar_expect_tx_only(b, T::WSLAB * 8);
    if (DIR == 2) tma_load_4d(dst, &tmap, b, ca0, pm, cb0, 0);
    else tma_load_4d(dst, &tmap, b, ca0, cb0, pm, 0);
  };
  if (tid == 0) issue(cT, 0);
  cur_next(cT);

  /* ---- static roles of this thread ---- */
  /* D / EF: face fid, component c (A-D) or Gauss point c (F) */
  const int c = tid & 3, fid = tid >> 2;
  const int fa = fid % TA, fb = fid / TA;       /* a fastest: coalesced output */
  /* faces to store: n+1 along the normal, n on a periodic axis (face n is face 0) */
  /* n_a, n_b (kernel parameters): n + 1 along the normal unless that axis wraps */
  const int t1_local = T::NA ? fb : fa;
  constexpr int s1 = T::NA ? HA : 1;            /* halo-face stride along t1 */
  const int fh0 = T::NA ? (t1_local + 2) * HA + fa : fb * HA + (t1_local + 2);
  double *const rg = ring + fid * 4 + c;        /* this thread's private column of the ring */
  constexpr int RS = 6 * NF * 4, RF = NF * 4;   /* ring strides: plane slot, field */
  /* transpose buffer: element (field, component cc, Gauss point gq) of face fid lives at
   * fid*64 + field*16 + 4*(cc ^ (fid&3)) + (gq ^ cc): conflict-free for the component-major writes
   * and for the Gauss-point-major reads of a half warp.
   * Both offsets are ONE xor of a per-thread constant with a compile-time one: a write of Gauss point gq goes to
   * Kw ^ gq, Kw = 4 (c ^ (fid&3)) + c; a read of component cc comes from Kr ^ 5 cc, Kr = 4 (fid&3) + c. */
  double *const xb = XBuf + fid * T::XF;
  double *const flux_d = flux + (4 + c) * g.FS;   /* this thread's output field: dF/dt of component c */
  int Kr = tid & 15, Kw = Kr ^ ((tid & 3) << 2);   /* fid = tid >> 2, c = tid & 3 */
  asm volatile("" : "+r"(Kr), "+r"(Kw));           /* kept in registers: otherwise re-derived from tid every plane */
#define XW(field, gq) xb[(field) * 16 + (Kw ^ (gq))]
#define XR(field, cc) xb[(field) * 16 + (Kr ^ (5 * (cc)))]
  constexpr int sn = T::NA ? 1 : EA;            /* slab stride along the normal */
  double bcf[8];                                /* the same coefficients per thread, for the out-of-line collision items
                                                   (extra halo faces, the long series): measured, handing those the
                                                   shared-memory table as well loses what the table gains (895 -> 888) */
  gksd::series_coefficients((tid & 3) >> 1, bcf);
  constexpr int QLo = 0, QRo = FH * 4 + 2, DNo = 2 * FH * 4 + 4;   /* offsets inside a stage buffer */

  /* offsets of the three stage buffers in turn, rotated once per iteration: plane i lives in buffer i % 3, so stage A
     works at (i % 3) SBUF, BC at ((i + 2) % 3) SBUF, D at ((i + 1) % 3) SBUF (three moves instead of three mod-3) */
  int sA = 0, sB = 2 * T::SBUF, sD = T::SBUF;
  int idseg = -1;                              /* stage F: cell index of this thread's face in marched plane 0 of the segment */
  const double *wA = Wp, *wB = Wp + T::WSLAB_PAD;
  /* slots of planes i-6 .. i-3 at i = 0, as pointers to this thread's column */
  double *rq0 = rg + 2 * (6 * NF * 4), *rq1 = rg + 3 * (6 * NF * 4), *rq2 = rg, *rq3 = rg + 6 * NF * 4;
  TR_DECL
  for (int i = 0; i < J + 2; ++i) {
    const int oA = sA, oB = sB, oD = sD;
    sA = oD;
    sB = oA;
    sD = oB;
    /* ring slots likewise: the plane that stage D produces in iteration i sits in slot (i - 2) & 3 (slots follow the
       iteration count, not the position in the column segment: a new segment primes 4 planes before pass 2 reads any) */
    double *const q0 = rq0, *const q1 = rq1, *const q2 = rq2, *const q3 = rq3;
    rq0 = q1;
    rq1 = q2;
    rq2 = q3;
    rq3 = q0;
    const double *const wcur = wA;                /* slab of plane i; the other one receives plane i + 1 */
    wA = wB;
    wB = wcur;
    /* cT describes plane i + 1 here: what stage A needs of it in the NEXT iteration */
    const int n0_A = n0_next;
    if (!UN_N) n0_next = T::NA ? cT.s.a0 : cT.s.b0;
    TR(0)   /* loop bookkeeping between two iterations */
    /* ONE hand-over per iteration: phase i-1 of the iteration barrier completes when every warp has finished
       A, BC, D of iteration i-1 AND the slab of plane i has landed - its TMA was issued at the top of iteration
       i-1, inside that phase, with its bytes expected on the same barrier (thread 0 arrives after it has issued,
       so the phase cannot complete before the expectation is registered).  Plane 0 has a barrier of its own. */
    if (i > 0) mbar_wait(&bar[2], (i - 1) & 1);
    else mbar_wait(&bar[0], 0);
    TR(1)   /* hand-over wait */
    if (i + 1 < J) {
      /* on a uniform grid only the issuing thread needs the TMA cursor: the other warps do not walk it */
      if (!UN_N || tid < 32) {
        if (tid == 0) issue(cT, i + 1);           /* slab (i+1)&1 was last read by stage A of iteration i-1 */
        cur_next(cT);
      }
    }
    TR(2)   /* TMA issue + cursor */

    /* ================= stage A: plane i =================
     * both WENO5 edge values of each cell, per component (one smoothness-indicator set serves the face on
     * either side), and the normal slope at the cell's right face.  Every thread owns item tid; the NITEM - NT
     * extra items go to a window of warps that rotates with the iteration, so that no warp is systematically
     * the slowest.  Without FUSE_A a thread with two items evaluates them together, statement-interleaved; with
     * FUSE_A the thread's own item is computed here unconditionally (stale slab in the draining iterations,
     * result dropped) as the head of the straight-line block that continues through BC and D below, and the
     * stores and the extra item follow that block. */
    const bool okA = i < J;
    const double *const W = wcur;
    double *const SA = Sb + oA;
    constexpr int NITEM = T::NCA * T::NCB * 4;
    const int n0 = n0_A;                          /* global index of normal face 0 of the tile */
    auto locate = [&](int item, const double *&w, int &cn, int &ct, int &cc) {
      cc = item & 3;
      const int cell = item >> 2;
      const int xa = cell % T::NCA, xb = cell / T::NCA;
      const int sa = T::NA ? xa + 2 : xa + 1, sb = T::NA ? xb : xb + 2;
      w = W + (cc * EB + sb) * EA + sa;
      cn = T::NA ? xa : xb; /* cell along the normal: global f0-1+cn */
      ct = T::NA ? xb : xa; /* halo index along t1 */
    };
    auto store = [&](int cn, int ct, int cc, double vl, double vr, double dn) {
      if (cn >= 1) { /* left edge = face cn-1: Qr */
        const int fh = T::NA ? ct * HA + (cn - 1) : (cn - 1) * HA + ct;
        SA[QRo + fh * 4 + cc] = vl;
      }
      if (cn < TN) { /* right edge = face cn: Ql, and the slope at that face */
        const int fh = T::NA ? ct * HA + cn : cn * HA + ct;
        SA[QLo + fh * 4 + cc] = vr;
        double mf = g.inv_12hn_u[DIR];
        if (!UN_N && !g.uniform[DIR]) mf = g.inv_12hn[DIR][min(n0 + cn, g.n[DIR]) + GKS_NG];
        SA[DNo + fh * 4 + cc] = dn * mf;
      }
    };
    auto edges_of_one = [&](int item) {
      double q[5][1], vl[1], vr[1];
      int cn, ct, cc;
      const double *w;
      locate(item, w, cn, ct, cc);
#pragma unroll
      for (int k = 0; k < 5; ++k) q[k][0] = w[(k - 2) * sn];
      gksd::weno5_edges_v<1>(q, eps, vl, vr);
      store(cn, ct, cc, vl[0], vr[0], gksd::normal_slope12(q[1][0], q[2][0], q[3][0], q[4][0]));
    };
    constexpr int NXA = NITEM - NT;
    static_assert(NXA >= 0 && NXA <= NT, "stage A: at most two items per thread");
    const int xa_id = (tid - 160 * i) & (NT - 1);   /* = (tid - 32 ((5 i) mod NW)) mod NT: the window moves 5 warps per iteration */
    double a_vl[1], a_vr[1], a_dn = 0.0;
    int a_cn = 0, a_ct = 0, a_cc = 0;
    if (FUSE_A) {
      double q[5][1];
      const double *w;
      locate(tid, w, a_cn, a_ct, a_cc);
#pragma unroll
      for (int k = 0; k < 5; ++k) q[k][0] = w[(k - 2) * sn];
      gksd::weno5_edges_v<1>(q, eps, a_vl, a_vr);
      a_dn = gksd::normal_slope12(q[1][0], q[2][0], q[3][0], q[4][0]);
    } else if (okA) {
      if (xa_id < NXA) {
        double q[5][2], vl[2], vr[2];
        int cnv[2], ctv[2], ccv[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
          const double *w;
          locate(u ? NT + xa_id : tid, w, cnv[u], ctv[u], ccv[u]);
#pragma unroll
          for (int k = 0; k < 5; ++k) q[k][u] = w[(k - 2) * sn];
        }
        gksd::weno5_edges_v<2>(q, eps, vl, vr);
#pragma unroll
        for (int u = 0; u < 2; ++u)
          store(cnv[u], ctv[u], ccv[u], vl[u], vr[u], gksd::normal_slope12(q[1][u], q[2][u], q[3][u], q[4][u]));
      } else {
        edges_of_one(tid);
      }
    }

    TR(3)   /* stage A */
    /* ================= stages BC (plane i-1) and D (plane i-2) =================
     * BC, collision (S4): the 4 lanes of a halo face split the four half-Maxwellian factors (left / right side,
     * erf / exp series), exchange them by shuffle, and every lane forms its component of Q0 in place of QL.
     * D, tangential pass 1 (along t1) on Q0 and Dn of the plane before.
     * The two touch different stage buffers.  With FUSE_BCD every thread's own BC item and its D item form ONE
     * straight-line block - loads, the short series unconditionally, two WENO5 Gauss-point evaluations, shuffles -
     * so that BC's serial chain (reciprocal, Horner, shuffles) issues in the shadow of D's dense arithmetic; in
     * the priming / draining iterations a stage works on stale shared memory and its result is dropped; a warp
     * that needs the long series (rare: |z| > 1/8) redoes its item afterwards. */
    const bool okB = i >= 1 && i - 1 < J;
    const bool have = i >= 2;
    double d6[6];
    int ga = 0, gb = 0;
    {
      double *const S = Sb + oB;                                    /* plane i-1 */
      static_assert((FH * 4) % 32 == 0, "whole warps in the collision stage");
      const int gl = (tid & 31) & ~3;               /* first lane of this face group */
      constexpr int NXB = FH * 4 - NT;              /* extra items: a rotating window of whole warps, disjoint from A's */
      static_assert(NXB >= 0 && NXB <= NT / 2 && NXB % 32 == 0, "stage BC: extras on whole warps");
      const int xb_id = xa_id ^ (NT / 2);           /* the same window half the warps further on */
      auto collide = [&](int item) {
        const int cc = item & 3, fh = item >> 2, side = cc & 1, func = cc >> 1;
        const double *qs = S + (side ? QRo : QLo) + fh * 4;
        const double rho = qs[0];
        const double z = ph.theta * (qs[1 + DIR] * gksd::fast_rcp3(rho));
        /* lane (side, func): func 0 -> erfc(-+z)/2 of that side, func 1 -> rho exp(-z^2) / (2 sqrt(pi lambda)) */
        const double v = gksd::erf_or_expm2_warp(z, func, bcf);
        const double r = func ? rho * (ph.cx * v) : fma(side ? -0.5 : 0.5, v, 0.5);
        const double el = __shfl_sync(0xffffffffu, r, gl), er = __shfl_sync(0xffffffffu, r, gl + 1);
        const double xl = __shfl_sync(0xffffffffu, r, gl + 2), xr = __shfl_sync(0xffffffffu, r, gl + 3);
        double q0 = S[QLo + item] * el + S[QRo + item] * er;
        if (cc == 1 + DIR) q0 += xl - xr;
        S[QLo + item] = q0;
      };
      auto pass1 = [&]() {
        ga = cD.s.a0 + fa;
        gb = cD.s.b0 + fb;
        const int t1_glob = T::NA ? gb : ga;
        double iw1 = g.inv_w_u[T::AXT1];
        if (!UN_T1 && !g.uniform[T::AXT1]) iw1 = g.inv_w[T::AXT1][min(t1_glob, g.n[T::AXT1] - 1) + GKS_NG];
        const double *q = Sb + oD + QLo + fh0 * 4 + c;                      /* Q0 of plane i-2 */
        const double *d = q + DNo;                                          /* Dn */
        double qq[5][2], vm[2], vp[2], sm_[2], sp_[2];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          qq[k][0] = q[(k - 2) * s1 * 4];
          qq[k][1] = d[(k - 2) * s1 * 4];
        }
        gksd::weno5_gauss_v<2, LIN>(qq, eps, vm, vp, sm_, sp_);
        d6[0] = vm[0];
        d6[1] = vp[0];
        d6[2] = vm[1];
        d6[3] = vp[1];
        d6[4] = sm_[0] * iw1;
        d6[5] = sp_[0] * iw1;
      };
      if (FUSE_BCD) {
        if (D_FIRST) pass1();
        const int side = c & 1, func = c >> 1;
        const double *qs = S + (side ? QRo : QLo) + (tid & ~3);
        const double rho = qs[0], mn = qs[1 + DIR];
        const double ql = S[QLo + tid], qr = S[QRo + tid];
        const double z = ph.theta * (mn * gksd::fast_rcp3(rho));
        const double w = z * z;
        const bool all_small = __all_sync(0xffffffffu, !(w > 1.0 / 64.0));
        double p = cfs[7];
#pragma unroll
        for (int n = 6; n >= 0; --n) p = fma(p, w, cfs[n]);
        const double v = func ? p : p * z;
        const double r = func ? rho * (ph.cx * v) : fma(side ? -0.5 : 0.5, v, 0.5);
        const double el = __shfl_sync(0xffffffffu, r, gl), er = __shfl_sync(0xffffffffu, r, gl + 1);
        const double xl = __shfl_sync(0xffffffffu, r, gl + 2), xr = __shfl_sync(0xffffffffu, r, gl + 3);
        double q0 = ql * el + qr * er;
        if (c == 1 + DIR) q0 += xl - xr;
        if (!D_FIRST) pass1();
        if (okB) {
          if (all_small) S[QLo + tid] = q0;
          else collide(tid);
        }
      } else {
        if (okB) collide(tid);
        if (have) pass1();
      }
      if (okB && xb_id < NXB) collide(NT + xb_id);
    }
    if (FUSE_A && okA) {
      store(a_cn, a_ct, a_cc, a_vl[0], a_vr[0], a_dn);
      if (xa_id < NXA) edges_of_one(NT + xa_id);
    }
    /* this warp is done with the shared stage buffers of iteration i */
    __syncwarp();
    mbar_arrive_lane0(&bar[2], tid & 31);
    TR(4)   /* stages BC + D, arrival */
    if (!have) continue;

    /* ================= stage EF: plane i-2 ================= */
    const int it = cD.it;
    const int m = cD.s.p0 + it - 2;
    cur_next(cD);

    double *const rnew = q0;                     /* slot of the plane four back, dead once pass 2 below has read it */
    if (it < 4) {
#pragma unroll
      for (int v = 0; v < 6; ++v) rnew[v * RF] = d6[v];
      /* what the stores of this column segment need, once per segment (here, in the priming planes, it costs the plane loop
         nothing): the cell index of marched plane 0, or -1 for a face beyond the last one (overhanging tile) */
      int pidx[3];
      pidx[0] = ga;
      pidx[T::AXB] = gb;
      pidx[T::AXM] = 0;
      idseg = (ga < n_a && gb < n_b)
                  ? ((pidx[2] + GKS_NG) * g.P[1] + (pidx[1] + GKS_NG)) * g.P[0] + (pidx[0] + GKS_NG)
                  : -1;
      continue;
    }
    /* ---- E: tangential pass 2 (along t2, the marched axis) for plane m = it-2; the ring holds planes
     *         it-4 .. it-1 (plane it-4+k in slot (it+k)&3), plane it comes straight from d6 ---- */
    double iw2 = g.inv_w_u[T::AXM];
    if (!UN_M && !g.uniform[T::AXM]) iw2 = g.inv_w[T::AXM][m + GKS_NG];
    const double *const rs[4] = {q0, q1, q2, q3};
    /* the six evaluations (field Q0, Dn, Dt1) x (g1 = -, +) run EW at a time, statement-interleaved */
    constexpr int EW = GKS_E_WIDTH;
    static_assert(6 % EW == 0, "E width");
    double late[8];                               /* GKS_XHALF: Dn and Dt1 at the 4 Gauss points */
#pragma unroll
    for (int e0 = 0; e0 < 6; e0 += EW) {
      double qq[5][EW], vm[EW], vp[EW], sm_[EW], sp_[EW];
#pragma unroll
      for (int u = 0; u < EW; ++u) {
#pragma unroll
        for (int k = 0; k < 4; ++k) qq[k][u] = rs[k][(e0 + u) * RF];
        qq[4][u] = d6[e0 + u];
      }
#pragma unroll
      for (int u = 0; u < EW; ++u) rnew[(e0 + u) * RF] = d6[e0 + u];   /* rs[0] aliases rnew: stored after the loads */
      gksd::weno5_gauss_v<EW, LIN>(qq, eps, vm, vp, sm_, sp_);
#pragma unroll
      for (int u = 0; u < EW; ++u) {              /* evaluation e = 2*fld + g1; Gauss point gq = 2*g1 + g2 */
        const int fld = (e0 + u) >> 1, g1 = (e0 + u) & 1;
        if (GKS_XHALF && fld != 0) {              /* Dn and Dt1 wait in registers for the second round */
          late[(fld - 1) * 4 + 2 * g1] = vm[u];
          late[(fld - 1) * 4 + 2 * g1 + 1] = vp[u];
        } else {
          XW(fld, 2 * g1) = vm[u];
          XW(fld, 2 * g1 + 1) = vp[u];
        }
        if (fld == 0) {
          XW(GKS_XHALF ? 1 : 3, 2 * g1) = sm_[u] * iw2;
          XW(GKS_XHALF ? 1 : 3, 2 * g1 + 1) = sp_[u] * iw2;
        }
      }
    }
    __syncwarp();
    TR(5)   /* pass 2 (E) */
    /* ---- F: flux at Gauss point gp = c of this face; sum over the 4 lanes; write ---- */
    {
      double Q0[4], dQ[3][4], F[4], dF[4];
      if (GKS_XHALF) {
        /* two rounds through 32 doubles per face: Q0 and Dt2 (complete after the first three evaluations), then Dn
           and Dt1 */
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          Q0[cc] = XR(0, cc);
          dQ[T::AXM][cc] = XR(1, cc);
        }
        __syncwarp();
#pragma unroll
        for (int gq = 0; gq < 4; ++gq) {
          XW(0, gq) = late[gq];
          XW(1, gq) = late[4 + gq];
        }
        __syncwarp();
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          dQ[DIR][cc] = XR(0, cc);
          dQ[T::AXT1][cc] = XR(1, cc);
        }
      } else {
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          Q0[cc] = XR(0, cc);
          dQ[DIR][cc] = XR(1, cc);
          dQ[T::AXT1][cc] = XR(2, cc);
          dQ[T::AXM][cc] = XR(3, cc);
        }
      }
      gksd::gauss_point_flux<DIR, NEED_F>(Q0, dQ, ph.RT, ph.mu, F, dF);
      __syncwarp();                               /* every lane has consumed its reads: the buffer is reusable */
      /* face average: the 4 lanes of a face (one Gauss point each) leave their F, dF in the warp-private
         buffer, lane c sums component c in the order (g0+g1)+(g2+g3).  Row v of face fid sits at
         ((v ^ (fid&3)) * 4 + gp): conflict-free 64-bit stores and loads */
#pragma unroll
      for (int v = 0; v < 4; ++v) {               /* (v ^ (fid&3)) * 4 + c = Kr ^ 4 v */
        if (NEED_F) xb[Kr ^ (4 * v)] = F[v];
        xb[16 + (Kr ^ (4 * v))] = dF[v];
      }
      __syncwarp();
      double fsel = 0.0, dsel;
      {
        const double *r = xb + (Kw & 12);         /* (c ^ (fid&3)) * 4 */
        if (NEED_F) fsel = (r[0] + r[1]) + (r[2] + r[3]);
        dsel = (r[16] + r[17]) + (r[18] + r[19]);
      }
      __syncwarp();                               /* pass 2 of the next plane writes the buffer again */
      if (idseg >= 0) {
        /* a padded field holds fewer than 2^31 doubles (gks_create): the cell index is a 32-bit number */
        const int id = idseg + m * (T::AXM == 2 ? g.P[0] * g.P[1] : g.P[0]);
        double *const fd = flux_d + id;           /* dF/dt of component c; F sits 4 fields below */
        if (NEED_F) fd[-4 * g.FS] = 0.25 * fsel;
        fd[0] = 0.25 * dsel;
      }
    }
    TR(6)   /* transposes, flux, face average, store (F) */
  }
  TR_DUMP
}

} /* namespace */

/* ---------------- host side: tensor maps and launch ---------------- */
namespace {

typedef CUresult (*encode_fn_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

/* tile shapes: 128 faces per CTA.  y- and z-faces: 32 (t1, along a) x 4 (normal).  x-faces: 8 (normal, along a) x 16 (t1)
   on a periodic x axis, 4 x 32 where face n+1 exists (walls, inflow / outflow, cut faces of a sub-domain): the two are
   equally fast per tile, the narrow one wastes less of the tile that hangs over the last face (257 faces: 1.2 % instead
   of 2.7 %; 33 faces of a 32-cell slab: 9 % instead of 21 %) but stages 9 cells for 4 faces along x and re-reads more of
   the slab halo from DRAM (measured 1.39 GB instead of 0.91 GB read per launch at 256^3): chosen per context */
#ifndef GKS_TILE_YZ_A
#define GKS_TILE_YZ_A 32
#endif
template <int DIR, int XA> struct Shape {
  static constexpr int TA = DIR == 0 ? XA : GKS_TILE_YZ_A, TB = GKS_NF / TA;
};
inline int x_tile_a(const GksGrid &g) { return g.wrapf[0] ? 8 : 4; }

template <int DIR, int XA>
bool encode_dir(encode_fn_t enc, const GksGrid &g, double *base, CUtensorMap *out) {
  using T = Tile<DIR, Shape<DIR, XA>::TA, Shape<DIR, XA>::TB>;
  const cuuint64_t dims[4] = {(cuuint64_t)g.P[0], (cuuint64_t)g.P[1], (cuuint64_t)g.P[2], 4};
  const cuuint64_t strides[3] = {(cuuint64_t)g.P[0] * 8, (cuuint64_t)g.P[0] * g.P[1] * 8, (cuuint64_t)g.FS * 8};
  cuuint32_t box[4] = {(cuuint32_t)T::EA, 1, 1, 4};
  box[T::AXB] = T::EB;
  const cuuint32_t es[4] = {1, 1, 1, 1};
  return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NAN_REQUEST_ZERO_FMA) == CUDA_SUCCESS;
}

/* tiles along a of direction dir: all of them */
int tiles_a(const GksGrid &g, int dir) {
  const int TA = dir == 0 ? x_tile_a(g) : GKS_TILE_YZ_A;
  const int ext_a = g.n[0] + (dir == 0 && !g.wrapf[0] ? 1 : 0);
  return (ext_a + TA - 1) / TA;
}

/* launch over the a-tiles [ta0, ta0 + len0) and [ta1, ta1 + len1) (len1 may be 0); returns the launches made */
template <int DIR, bool NEED_F, bool LIN, int XA, int UMASK>
int launch_dir(gks_ctx *ctx, const CUtensorMap &map, double *flux, int ta0, int len0, int ta1, int len1) {
  constexpr int TA = Shape<DIR, XA>::TA, TB = Shape<DIR, XA>::TB;
  using T = Tile<DIR, TA, TB>;
  const GksGrid &g = ctx->g;
  auto kern = k_sweep_fused<DIR, NEED_F, LIN, TA, TB, UMASK>;
  static bool attr_done[64] = {};                /* the attribute is per device: one process may hold contexts on several */
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_done[dev]) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM_BYTES);
    if (dev >= 0 && dev < 64) attr_done[dev] = true;
  }
  const int ext_a = g.n[0] + (T::NA && !g.wrapf[0] ? 1 : 0), ext_b = g.n[T::AXB] + (!T::NA && !g.wrapf[T::AXB] ? 1 : 0);
  const int n2 = g.n[T::AXM];
  const int ga = len0 + len1, gb = (ext_b + TB - 1) / TB;
  if (ga <= 0) return 0;
  /* persistent CTAs: the (column, plane) list is cut into equal contiguous ranges, one per resident CTA;
     a range shorter than 8 planes is not worth its 4 priming planes */
  const int ncols = ga * gb;
  int grid = ctx->num_sms * GKS_CTAS_PER_SM, nfull = ncols / grid;
  long long rem = (long long)(ncols - nfull * grid) * n2;      /* planes of the columns that do not fill a wave */
  long long PPC = (rem + grid - 1) / grid;
  if (PPC < GKS_MIN_PPC) PPC = GKS_MIN_PPC;                    /* shortest range worth its 4 priming planes */
  if (nfull == 0) grid = (int)((rem + PPC - 1) / PPC);
  gks_launch(kern, grid, dim3(T::NT), T::SMEM_BYTES, ctx->stream, map, g, ctx->ph, flux, ga, nfull, rem, PPC, ta0, len0, ta1 - len0, ext_a, ext_b);
  return 1;
}

} /* namespace */

#ifdef GKS_DEBUG
extern "C" gks_status gks_debug_trace(gks_ctx *ctx, unsigned long long *ticks) {
  if (!ctx || !ticks) return GKS_ERR_INVALID_ARG;
#ifdef GKS_TRACE
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e == cudaSuccess) e = cudaMemcpyFromSymbol(ticks, gks_trace_buf, sizeof(gks_trace_buf));
  if (e != cudaSuccess) return gks_set_err(ctx, GKS_ERR_CUDA, "trace read-back: %s", cudaGetErrorString(e));
  return GKS_OK;
#else
  return gks_set_err(ctx, GKS_ERR_STATE, "this library was built without -DGKS_TRACE (python -m paper_2603_11102_b200.trace builds one)");
#endif
}
#endif

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
    if (!(x_tile_a(ctx->g) == 8 ? encode_dir<0, 8>(enc, ctx->g, bases[b], m) : encode_dir<0, 4>(enc, ctx->g, bases[b], m))) return false;
    if (!encode_dir<1, 8>(enc, ctx->g, bases[b], reinterpret_cast<CUtensorMap *>(ctx->tmaps[b][1]))) return false;
    if (!encode_dir<2, 8>(enc, ctx->g, bases[b], reinterpret_cast<CUtensorMap *>(ctx->tmaps[b][2]))) return false;
  }
  return true;
}

/* part: 0 = the whole direction, 1 = interior tiles only, 2 = rim tiles only (ctx->part_*: gks_step_begin_part) */
int gks_launch_sweep_fused(gks_ctx *ctx, int dir, int which, double *flux, bool need_F, int part) {
  const CUtensorMap &m = *reinterpret_cast<const CUtensorMap *>(ctx->tmaps[which][dir]);
  const bool lin = ctx->ph.tang_linear != 0;
  const int all = tiles_a(ctx->g, dir);
  int ta0 = 0, len0 = all, ta1 = 0, len1 = 0;
  if (part != 0) {
    const int t0 = ctx->part_t0[dir], t1 = ctx->part_t1[dir];   /* interior tiles [t0, t1) */
    if (part == 1) {
      ta0 = t0;
      len0 = t1 - t0;
    } else {
      ta0 = 0;
      len0 = t0;
      ta1 = t1;
      len1 = all - t1;
    }
  }
  const int ubits = (ctx->g.uniform[0] ? 1 : 0) | (ctx->g.uniform[1] ? 2 : 0) | (ctx->g.uniform[2] ? 4 : 0);
  const int umask = ubits == 7 ? 7 : ((ubits & 5) == 5 ? 5 : 0);
#define GKS_DISPATCH3(D, XA, NF_, LIN_)                                                                      \
  (umask == 7 ? launch_dir<D, NF_, LIN_, XA, 7>(ctx, m, flux, ta0, len0, ta1, len1)                          \
   : umask == 5 ? launch_dir<D, NF_, LIN_, XA, 5>(ctx, m, flux, ta0, len0, ta1, len1)                        \
                : launch_dir<D, NF_, LIN_, XA, 0>(ctx, m, flux, ta0, len0, ta1, len1))
#define GKS_DISPATCH(D, XA)                                                                                  \
  (need_F ? (lin ? GKS_DISPATCH3(D, XA, true, true) : GKS_DISPATCH3(D, XA, true, false))                     \
          : (lin ? GKS_DISPATCH3(D, XA, false, true) : GKS_DISPATCH3(D, XA, false, false)))
  switch (dir) {
    case 0: return x_tile_a(ctx->g) == 8 ? GKS_DISPATCH(0, 8) : GKS_DISPATCH(0, 4);
    case 1: return GKS_DISPATCH(1, 8);
    default: return GKS_DISPATCH(2, 8);
  }
#undef GKS_DISPATCH3
#undef GKS_DISPATCH
}

/* tile sizes along x of the three sweep directions (for the interior / rim split of a sub-domain) */
void gks_fused_tiles_x(const GksGrid &g, int ta[3]) {
  ta[0] = x_tile_a(g);
  ta[1] = GKS_TILE_YZ_A;
  ta[2] = GKS_TILE_YZ_A;
}
