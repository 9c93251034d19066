// chunk_dev.cuh -- per-chunk sequential kernels' building blocks (k_fold0, k_down0, k_query).
//
// Layout: a group of G lanes (8, 16 or 32 lanes of one warp) works on one chunk.  Every n x n state
// matrix (P, Lambda, C, A, J) lives in shared memory, row-major with an odd row stride ld >= n + 1
// (column n carries the companion vector: [P | m], [Lambda | lambda], [A | b], [J | eta]), and lane j
// OWNS column j: it computes whole columns, so a product with the transition needs no cross-lane
// reduction.  The transition of one step is never assembled: it is applied straight from the step's
// discretisation record (staged by a TMA bulk copy; block-diagonal Phi_b, integral rows Phi-bar_b), so a
// product F X costs sum_b (d_b^2 + d_b) + N_inst n_blk FMAs per column instead of n^2.
//
//   F  = R [Phi 0; Phi-bar I]  (Eq. 3.7, Eq. 3.17; R zeroes the z rows in `tz`,
//                               the reset of Eq. 3.11/3.18 folded into the step, reading R2/R6)
//   z_q row of [Phi-bar I]:  sum_b c_qb Phi-bar_b x_b + z_q   (c_qb = 0 if component b is not in
//                               instrument q's integrand, Eq. 3.2)
#pragma once
#ifndef SG_JIT
#include <string.h>

#include "common.h"
#endif
#include "dev_consts.h"
#include "grp_dev.cuh"

// Model tables of the chunk kernels.  Passed BY VALUE inside the kernel parameter struct: kernel
// parameters live in the constant bank, so every table look-up with a warp-uniform index is a
// uniform load and the block loop's bookkeeping and branches run on the uniform datapath.
struct Tab {
  int n, d, ninst, nblk, stride, ld;
  unsigned char bdim[SG_MAXBLK], boff[SG_MAXBLK];
  short roff[SG_MAXBLK];
  unsigned char blk_of[SG_NMAX];
  double cz[SG_MAXINST * SG_MAXBLK]; // [q * nblk + b]
  double tau[SG_MAXINST];
  double bsig[SG_MAXBLK];            // sigma_b
  unsigned bmask[SG_MAXBLK];         // inst_mask of block b's component (bits >= n_inst: virtual instruments, C13-C14)
};

// row stride of the chunk kernels' matrices: the smallest value = 1 (mod 4) that holds n + 1 columns
// (odd: conflict-free row reads; a multiple-of-4 family keeps the number of compiled variants small)
__host__ __device__ inline int chunk_ld(int n) { return ((n + 3) / 4) * 4 + 1; }

#ifndef SG_JIT
inline void tab_build(const ModelDev* M, Tab* T) {
  memset(T, 0, sizeof(Tab));
  const int n = M->n;
  T->n = n; T->d = M->d; T->ninst = M->n_inst; T->nblk = M->nblk; T->stride = M->disc_stride; T->ld = chunk_ld(n);
  for (int b = 0; b < M->nblk; ++b) {
    T->bdim[b] = (unsigned char)M->blk[b].dim; T->boff[b] = (unsigned char)M->blk[b].off; T->roff[b] = (short)M->disc_off[b];
    for (int i = 0; i < M->blk[b].dim; ++i) T->blk_of[M->blk[b].off + i] = (unsigned char)b;
    for (int q = 0; q < M->n_inst; ++q) T->cz[q * M->nblk + b] = M->cz[q][b];
    T->bsig[b] = M->bsig[b]; T->bmask[b] = M->bmask[b];
  }
  for (int q = 0; q < M->n_inst; ++q) T->tau[q] = M->tau[q];
}
#endif

// Table access.  Statically compiled kernels read the tables from the kernel parameters (`T`); the
// run-time specialised build (SG_JIT, jit.cu) replaces them by constants generated for one model, so
// every loop over blocks / instruments unrolls and the family switch disappears.
#ifdef SG_JIT
#define TN JT_N
#define TD JT_D
#define TNI JT_NI
#define TNB JT_NB
#define TSTRIDE JT_STRIDE
#define TBDIM(b) jt_bdim(b)
#define TBOFF(b) jt_boff(b)
#define TROFF(b) jt_roff(b)
#define TBLKOF(j) jt_blkof(j)
#define TCZ(i) (jt_czmask(i) ? T.cz[i] : 0.0) /* values stay run-time; the zero pattern is compile-time */
#define TTAU(q) (T.tau[q])
#define SG_UNROLL _Pragma("unroll")
#else
#define TN (T.n)
#define TD (T.d)
#define TNI (T.ninst)
#define TNB (T.nblk)
#define TSTRIDE (T.stride)
#define TBDIM(b) (T.bdim[b])
#define TBOFF(b) (T.boff[b])
#define TROFF(b) (T.roff[b])
#define TBLKOF(j) (T.blk_of[j])
#define TCZ(i) (T.cz[i])
#define TTAU(q) (T.tau[q])
#define SG_UNROLL
#endif

// ---- record staging: global -> shared with the TMA bulk copy (cp.async.bulk, UBLKCP) ----------------
// One lane of the group arms an mbarrier with the record's byte count and issues ONE bulk copy per
// event (records have an even number of doubles and start on 16-byte boundaries in both memories);
// every lane then waits on the barrier's phase.  Two buffers, two barriers: event k + 1 is in flight
// while event k is being used.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

struct RecStage {
  double* buf;               // 2 x stride doubles
  unsigned long long* bar;   // 2 mbarriers (right after the buffers)
  unsigned phase;            // bit b = parity to wait for on barrier b
  int stride;

  template <int G>
  __device__ __forceinline__ void init(const Grp<G>& g, double* recs, int stride_) {
    buf = recs; stride = stride_; phase = 0u;
    bar = reinterpret_cast<unsigned long long*>(recs + 2 * stride_);
    if (g.gl == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(bar)));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(smem_u32(bar + 1)));
      asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    g.sync();
  }
  // request the record at `src` into buffer b (all lanes call it; one issues)
  template <int G>
  __device__ __forceinline__ void issue(const Grp<G>& g, const double* __restrict__ src, int b) {
    if (g.gl == 0) {
      const unsigned bytes = (unsigned)stride * 8u, mb = smem_u32(bar + b);
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mb), "r"(bytes) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(buf + b * stride)),
                   "l"(src), "r"(bytes), "r"(mb)
                   : "memory");
    }
  }
  // wait until buffer b holds its record; returns it
  __device__ __forceinline__ const double* wait(int b) {
    const unsigned mb = smem_u32(bar + b), par = (phase >> b) & 1u;
    unsigned ok = 0;
    while (!ok) {
      asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(mb), "r"(par) : "memory");
    }
    phase ^= (1u << b);
    return buf + b * stride;
  }
};

// Phi_b (DB x DB, row-major) and Phi-bar_b (DB) of one block, contiguous in the staged record.  Records
// are laid out so that every block starts on a 16-byte boundary (even block sizes, even buffer offsets):
// for even DB the rows come in as 128-bit shared-memory loads -- all lanes read the same address, so a
// wider broadcast load halves the number of LSU wavefronts.
template <int DB>
__device__ __forceinline__ void load_block(const double* r, double (&m)[DB * DB + DB]) { // no __restrict__: a compiler fence between blocks must hold these loads back (chunk_reg.cuh)
  if constexpr (DB % 2 == 0) {
    const double2* r2 = reinterpret_cast<const double2*>(r);
#pragma unroll
    for (int k = 0; k < (DB * DB + DB) / 2; ++k) { const double2 t = r2[k]; m[2 * k] = t.x; m[2 * k + 1] = t.y; }
  } else {
#pragma unroll
    for (int k = 0; k < DB * DB + DB; ++k) m[k] = r[k];
  }
}

// ---- one block of out = F v ------------------------------------------------------------------------
template <int DB, int VS, int OS>
__device__ __forceinline__ double blk_F(const double* __restrict__ r, const double* vp, double* op, int off) {
  double w[DB], m[DB * DB + DB];
#pragma unroll
  for (int l = 0; l < DB; ++l) w[l] = vp[(off + l) * VS];
  load_block<DB>(r, m);
#pragma unroll
  for (int i = 0; i < DB; ++i) {
    double acc = 0.0;
#pragma unroll
    for (int l = 0; l < DB; ++l) acc = fma(m[i * DB + l], w[l], acc);
    op[(off + i) * OS] = acc;
  }
  double u = 0.0;
#pragma unroll
  for (int l = 0; l < DB; ++l) u = fma(m[DB * DB + l], w[l], u); // Phi-bar_b . v_b
  return u;
}

// out = F v for the calling lane's vector: v[i] = vp[i * vs], out[i] = op[i * os] (i < n).
// U: lane-private scratch of nblk doubles at stride G.  `rec` in shared memory.
template <int G, int VS, int OS>
__device__ __forceinline__ void apply_F(const Tab& T, const double* rec, unsigned tz, const double* vp, double* op, double* U) {
  const int nblk = TNB, d = TD;
#ifdef SG_JIT
  double ul[JT_NB]; // the specialised build unrolls the block loops: the per-block integrals stay in registers
#define SG_UREF(b) ul[b]
#else
#define SG_UREF(b) U[(b) * G]
#endif
  SG_UNROLL
  for (int b = 0; b < nblk; ++b) {
    const double* r = rec + TROFF(b);
    const int off = TBOFF(b);
    double u;
    switch (TBDIM(b)) {
      case 2: u = blk_F<2, VS, OS>(r, vp, op, off); break;
      case 3: u = blk_F<3, VS, OS>(r, vp, op, off); break;
      default: u = blk_F<4, VS, OS>(r, vp, op, off); break;
    }
    SG_UREF(b) = u;
  }
  SG_UNROLL
  for (int q = 0; q < TNI; ++q) {
    double acc = 0.0;
    if (!((tz >> q) & 1u)) {
      acc = vp[(d + q) * VS];
      SG_UNROLL
      for (int b = 0; b < nblk; ++b) acc = fma(TCZ(q * nblk + b), SG_UREF(b), acc);
    }
    op[(d + q) * OS] = acc;
  }
#undef SG_UREF
}

// ---- one block of out = F^T v ----------------------------------------------------------------------
template <int DB, int VS, int OS>
__device__ __forceinline__ void blk_Ft(const double* __restrict__ r, const double* vp, double* op, int off, double s) {
  double w[DB], m[DB * DB + DB];
#pragma unroll
  for (int i = 0; i < DB; ++i) w[i] = vp[(off + i) * VS];
  load_block<DB>(r, m);
#pragma unroll
  for (int l = 0; l < DB; ++l) {
    double acc = m[DB * DB + l] * s; // Phi-bar_b[l] * sum_q c_qb v_zq
#pragma unroll
    for (int i = 0; i < DB; ++i) acc = fma(m[i * DB + l], w[i], acc);
    op[(off + l) * OS] = acc;
  }
}

template <int G, int VS, int OS>
__device__ __forceinline__ void apply_Ft(const Tab& T, const double* rec, unsigned tz, const double* vp, double* op) {
  const int nblk = TNB, d = TD;
  SG_UNROLL
  for (int b = 0; b < nblk; ++b) {
    double s = 0.0;
    SG_UNROLL
    for (int q = 0; q < TNI; ++q)
      if (!((tz >> q) & 1u)) s = fma(TCZ(q * nblk + b), vp[(d + q) * VS], s);
    const double* r = rec + TROFF(b);
    const int off = TBOFF(b);
    switch (TBDIM(b)) {
      case 2: blk_Ft<2, VS, OS>(r, vp, op, off, s); break;
      case 3: blk_Ft<3, VS, OS>(r, vp, op, off, s); break;
      default: blk_Ft<4, VS, OS>(r, vp, op, off, s); break;
    }
  }
  SG_UNROLL
  for (int q = 0; q < TNI; ++q) op[(d + q) * OS] = ((tz >> q) & 1u) ? 0.0 : vp[(d + q) * VS];
}

// column j of X += column j of Q = R Q~ R^T (Eq. 3.10 P:403-405 per block; z rows through c_qb)
template <int LD>
__device__ __forceinline__ void add_Q_col(const Tab& T, const double* rec, unsigned tz, int j, double* X) {
  constexpr int ld = LD;
  const int d = TD, nblk = TNB;
  if (j < d) {
    // the block of column j is found by a loop over the blocks with compile-time bounds in the specialised
    // build (no table look-up with a lane-dependent index, which would live in local memory there)
    SG_UNROLL
    for (int b = 0; b < nblk; ++b) {
      const int db = TBDIM(b), off = TBOFF(b), jj = j - off;
      if (jj < 0 || jj >= db) continue;
      const double* r = rec + TROFF(b);
      const double* qxx = r + db * db + db;
      SG_UNROLL
      for (int i = 0; i < db; ++i) X[(off + i) * ld + j] += qxx[i * db + jj];
      const double q12 = r[2 * db * db + db + jj];
      SG_UNROLL
      for (int q = 0; q < TNI; ++q)
        if (!((tz >> q) & 1u)) X[(d + q) * ld + j] = fma(TCZ(q * nblk + b), q12, X[(d + q) * ld + j]);
    }
  } else if (j < TN) {
    SG_UNROLL
    for (int q = 0; q < TNI; ++q) { // the lane's own instrument, found with compile-time indices (see above)
      if (j != d + q || ((tz >> q) & 1u)) continue;
      SG_UNROLL
      for (int b = 0; b < nblk; ++b) {
        const int db = TBDIM(b), off = TBOFF(b);
        const double* r = rec + TROFF(b);
        const double c = TCZ(q * nblk + b);
        if (c == 0.0) continue;
        SG_UNROLL
        for (int l = 0; l < db; ++l) X[(off + l) * ld + j] = fma(c, r[2 * db * db + db + l], X[(off + l) * ld + j]);
        const double q22 = r[2 * db * db + 2 * db];
        SG_UNROLL
        for (int p = 0; p < TNI; ++p)
          if (!((tz >> p) & 1u)) X[(d + p) * ld + j] = fma(c * TCZ(p * nblk + b), q22, X[(d + p) * ld + j]);
      }
    }
  }
}

// X <- F X F^T (+ Q) for a symmetric X (columns 0..n-1) and x <- F x for the companion column n.
// Tm: scratch of the same shape.  Two column-owned products:  Tm = F [X | x];  X[:, j] = F (Tm[j, :])^T.
// One lane per column (the group has at least n + 1 lanes: pick_lanes).
template <int G, int LD, bool ADDQ>
__device__ __forceinline__ void sandwich_F(const Grp<G>& g, const Tab& T, const double* rec, unsigned tz, double* X, double* Tm, double* U) {
  constexpr int ld = LD;
  const int n = TN, j = g.gl;
  if (j <= n) apply_F<G, LD, LD>(T, rec, tz, X + j, Tm + j, U);
  g.sync();
  if (j < n) {
    apply_F<G, 1, LD>(T, rec, tz, Tm + j * ld, X + j, U);
    if (ADDQ) add_Q_col<LD>(T, rec, tz, j, X);
    X[j * ld + n] = Tm[j * ld + n]; // companion column: lane j moves entry j
  }
  g.sync();
}

// X <- F^T X F, x <- F^T x (the adjoint / information direction)
template <int G, int LD>
__device__ __forceinline__ void sandwich_Ft(const Grp<G>& g, const Tab& T, const double* rec, unsigned tz, double* X, double* Tm) {
  constexpr int ld = LD;
  const int n = TN, j = g.gl;
  if (j <= n) apply_Ft<G, LD, LD>(T, rec, tz, X + j, Tm + j);
  g.sync();
  if (j < n) {
    apply_Ft<G, 1, LD>(T, rec, tz, Tm + j * ld, X + j);
    X[j * ld + n] = Tm[j * ld + n];
  }
  g.sync();
}

// X <- (X + X^T) / 2 on columns 0..n-1: lane j pairs with the n/2 columns after it (cyclically), so
// every unordered pair is visited exactly once (the antipodal pairs of an even n by the lower lane only:
// no two lanes ever touch the same cells)
template <int G, int LD>
__device__ __forceinline__ void symmetrise(const Grp<G>& g, const Tab& T, double* X) {
  constexpr int ld = LD;
  const int n = TN, half = n >> 1, j = g.gl;
  if (j < n) {
#pragma unroll
    for (int s = 1; s <= (LD - 1) / 2; ++s) {
      if (s <= half && !(((n & 1) == 0) && s == half && j >= half)) {
        int i = j + s;
        if (i >= n) i -= n;
        const double w = 0.5 * (X[i * ld + j] + X[j * ld + i]);
        X[i * ld + j] = w;
        X[j * ld + i] = w;
      }
    }
  }
  g.sync();
}
