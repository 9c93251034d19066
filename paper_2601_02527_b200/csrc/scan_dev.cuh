// scan_dev.cuh -- group-cooperative small dense fp64 linear algebra in shared memory, used by the
// scan kernels of scan.cu.  A "group" is G lanes (8, 16 or 32) of one warp working on one chunk;
// all matrices are n x n (n <= 32, run time) row-major in shared memory.
#pragma once
#include "common.h"
#include "grp_dev.cuh"

// per-CTA tables derived from the model
struct Tables {
  int n, d, ninst, nblk, ntri, nent, stride;
  const unsigned char* tri_i; // [ntri] lower-triangle index -> row
  const unsigned char* tri_j; //                             -> column
  const unsigned char* lo;    // [n] column range of row i of F (x rows: own block; z rows: [0, d))
  const unsigned char* hi;
  const unsigned char* ent_r; // [nent] block entries: global row, column
  const unsigned char* ent_c;
  const short* ent_src;       // [nent] offset of the Phi entry inside an event record
  const short* ent_qsrc;      //        offset of the Qxx entry
  const short* x_pb;          // [d] offset of phibar entry for x index l
  const short* x_q12;         // [d] offset of q12 entry
  const short* b_q22;         // [nblk] offset of q22
  const double* czl;          // [ninst][d]  c_{q, blk(l)}
  const double* czb;          // [ninst][nblk]
  const double* tau;          // [ninst]
};

__host__ __device__ inline size_t tables_bytes(int n, int d, int ninst, int nblk, int nent) {
  size_t dbl = (size_t)ninst * d + (size_t)ninst * nblk + ninst;
  size_t sh = (size_t)2 * nent + 2 * d + nblk;
  size_t by = (size_t)n * (n + 1) + 2 * n + 2 * nent;
  size_t tot = dbl * 8 + ((sh * 2 + 7) / 8) * 8 + ((by + 7) / 8) * 8;
  return tot;
}

// builds the tables in shared memory (whole CTA participates; caller syncs afterwards)
__device__ inline void tables_build(const ModelDev* __restrict__ M, char* smem, Tables& T) {
  const int n = M->n, d = M->d, ninst = M->n_inst, nblk = M->nblk;
  int nent = 0;
  for (int b = 0; b < nblk; ++b) nent += M->blk[b].dim * M->blk[b].dim;
  T.n = n; T.d = d; T.ninst = ninst; T.nblk = nblk; T.ntri = n * (n + 1) / 2; T.nent = nent; T.stride = M->disc_stride;
  double* czl = (double*)smem;
  double* czb = czl + ninst * d;
  double* tau = czb + ninst * nblk;
  short* sh = (short*)(tau + ninst);
  short* ent_src = sh; short* ent_qsrc = ent_src + nent; short* x_pb = ent_qsrc + nent; short* x_q12 = x_pb + d; short* b_q22 = x_q12 + d;
  const size_t shn = (size_t)2 * nent + 2 * d + nblk;
  unsigned char* by = (unsigned char*)sh + ((shn * 2 + 7) / 8) * 8;
  unsigned char* tri_i = by; unsigned char* tri_j = tri_i + T.ntri; unsigned char* lo = tri_j + T.ntri; unsigned char* hi = lo + n;
  unsigned char* ent_r = hi + n; unsigned char* ent_c = ent_r + nent;
  if (threadIdx.x == 0) {
    int e = 0;
    for (int i = 0; i < n; ++i) for (int j = 0; j <= i; ++j) { tri_i[e] = (unsigned char)i; tri_j[e] = (unsigned char)j; ++e; }
    for (int i = 0; i < n; ++i) { lo[i] = (unsigned char)M->row_lo[i]; hi[i] = (unsigned char)M->row_hi[i]; }
    e = 0;
    for (int b = 0; b < nblk; ++b) {
      const int db = M->blk[b].dim, off = M->blk[b].off, ro = M->disc_off[b];
      for (int r = 0; r < db; ++r)
        for (int c = 0; c < db; ++c) {
          ent_r[e] = (unsigned char)(off + r); ent_c[e] = (unsigned char)(off + c);
          ent_src[e] = (short)(ro + r * db + c); ent_qsrc[e] = (short)(ro + db * db + db + r * db + c); ++e;
        }
      for (int c = 0; c < db; ++c) { x_pb[off + c] = (short)(ro + db * db + c); x_q12[off + c] = (short)(ro + 2 * db * db + db + c); }
      b_q22[b] = (short)(ro + 2 * db * db + 2 * db);
      for (int q = 0; q < ninst; ++q) {
        czb[q * nblk + b] = M->cz[q][b];
        for (int c = 0; c < db; ++c) czl[q * d + off + c] = M->cz[q][b];
      }
    }
    for (int q = 0; q < ninst; ++q) tau[q] = M->tau[q];
  }
  T.tri_i = tri_i; T.tri_j = tri_j; T.lo = lo; T.hi = hi; T.ent_r = ent_r; T.ent_c = ent_c;
  T.ent_src = ent_src; T.ent_qsrc = ent_qsrc; T.x_pb = x_pb; T.x_q12 = x_q12; T.b_q22 = b_q22;
  T.czl = czl; T.czb = czb; T.tau = tau;
}

// Assemble the dense transition Fs = R [Phi 0; Phi-bar I] and noise Qs = R Q~ R^T of one step in
// equilibrated units (Eq. 3.17 P:468-472 for the layout; Eq. 3.20 P:504 for the reset R folded into
// the step).  zm = set of instruments whose z row is zeroed by R.  Entries outside the block
// structure are zero and must have been zeroed once by the caller.  No sync inside.
template <int G>
__device__ __forceinline__ void assemble_step(const Grp<G>& g, const Tables& T, const double* __restrict__ rec,
                                              unsigned zm, double* Fs, double* Qs) {
  const int n = T.n, d = T.d;
  for (int e = g.gl; e < T.nent; e += G) {
    const int idx = T.ent_r[e] * n + T.ent_c[e];
    Fs[idx] = __ldg(rec + T.ent_src[e]);
    Qs[idx] = __ldg(rec + T.ent_qsrc[e]);
  }
  const int nz = T.ninst * d;
  const float rd = 1.0f / (float)d;
  for (int e = g.gl; e < nz; e += G) {
    int q, l;
    divmod_small(e, d, rd, q, l);
    const bool keep = !((zm >> q) & 1u);
    const double c = T.czl[e];
    const double f = keep ? c * __ldg(rec + T.x_pb[l]) : 0.0;
    const double qq = keep ? c * __ldg(rec + T.x_q12[l]) : 0.0;
    Fs[(d + q) * n + l] = f;
    Qs[(d + q) * n + l] = qq;
    Qs[l * n + d + q] = qq;
  }
  const int nzz = T.ninst * T.ninst;
  const float ri = 1.0f / (float)T.ninst;
  for (int e = g.gl; e < nzz; e += G) {
    int q, r;
    divmod_small(e, T.ninst, ri, q, r);
    const bool keep = !((zm >> q) & 1u) && !((zm >> r) & 1u);
    double s = 0.0;
    if (keep)
      for (int b = 0; b < T.nblk; ++b) s = fma(T.czb[q * T.nblk + b] * T.czb[r * T.nblk + b], __ldg(rec + T.b_q22[b]), s);
    Qs[(d + q) * n + d + r] = s;
    Fs[(d + q) * n + d + r] = (keep && q == r) ? 1.0 : 0.0;
  }
}

// dst[i, j] = sum_l Fs[i, l] src[l, j]   (i < n, j < nc), using the row ranges of Fs.
// src/dst addressed with (row stride, column stride).  No sync inside.
template <int G>
__device__ __forceinline__ void lmul_F(const Grp<G>& g, const Tables& T, const double* Fs, const double* src, int sr, int sc,
                                       double* dst, int dr, int dc, int nc) {
  const int n = T.n, d = T.d;
  const float rnc = 1.0f / (float)nc;
  for (int e = g.gl; e < n * nc; e += G) {
    int i, j;
    divmod_small(e, nc, rnc, i, j);
    const int lo = T.lo[i], hi = T.hi[i];
    double acc = 0.0;
    for (int l = lo; l < hi; ++l) acc = fma(Fs[i * n + l], src[l * sr + j * sc], acc);
    if (i >= d) acc = fma(Fs[i * n + i], src[i * sr + j * sc], acc);
    dst[i * dr + j * dc] = acc;
  }
}

// C[i, j] = C[j, i] = add[i, j] + sum_l Tm[i, l] Fs[j, l]   for i >= j   (the product X Fs^T)
template <int G>
__device__ __forceinline__ void rmul_Ft_sym(const Grp<G>& g, const Tables& T, const double* Fs, const double* Tm,
                                            const double* add, double* C) {
  const int n = T.n, d = T.d;
  for (int e = g.gl; e < T.ntri; e += G) {
    const int i = T.tri_i[e], j = T.tri_j[e];
    const int lo = T.lo[j], hi = T.hi[j];
    double acc = add ? add[i * n + j] : 0.0;
    for (int l = lo; l < hi; ++l) acc = fma(Tm[i * n + l], Fs[j * n + l], acc);
    if (j >= d) acc = fma(Tm[i * n + j], Fs[j * n + j], acc);
    C[i * n + j] = acc;
    C[j * n + i] = acc;
  }
}

// dst[i, j] = sum_l Fs[l, i] src[l, j]  (the product Fs^T X): column i of Fs is non-zero on its own
// block rows and on the z rows for i < d, and only on the diagonal for i >= d.
template <int G>
__device__ __forceinline__ void lmul_Ft(const Grp<G>& g, const Tables& T, const double* Fs, const double* src, int sr, int sc,
                                        double* dst, int dr, int dc, int nc) {
  const int n = T.n, d = T.d;
  const float rnc = 1.0f / (float)nc;
  for (int e = g.gl; e < n * nc; e += G) {
    int i, j;
    divmod_small(e, nc, rnc, i, j);
    double acc = 0.0;
    if (i < d) {
      const int lo = T.lo[i], hi = T.hi[i];
      for (int l = lo; l < hi; ++l) acc = fma(Fs[l * n + i], src[l * sr + j * sc], acc);
      for (int l = d; l < n; ++l) acc = fma(Fs[l * n + i], src[l * sr + j * sc], acc);
    } else {
      acc = Fs[i * n + i] * src[i * sr + j * sc];
    }
    dst[i * dr + j * dc] = acc;
  }
}

// general dense product  D[i,j] = (C ? C[i,j] : 0) + sum_l A[i,l] B[l,j],  strided operands
template <int G>
__device__ __forceinline__ void mm(const Grp<G>& g, int nr, int nc, int nk, const double* A, int ar, int ac,
                                   const double* B, int br, int bc, const double* C, int cr, int cc, double* D, int dr, int dc) {
  const float rnc = 1.0f / (float)nc;
  for (int e = g.gl; e < nr * nc; e += G) {
    int i, j;
    divmod_small(e, nc, rnc, i, j);
    double acc = C ? C[i * cr + j * cc] : 0.0;
    for (int l = 0; l < nk; ++l) acc = fma(A[i * ar + l * ac], B[l * br + j * bc], acc);
    D[i * dr + j * dc] = acc;
  }
}
// symmetric result: D[i,j] = D[j,i] = (C ? C[i,j] : 0) + sum_l A[i,l] B[l,j] for i >= j (n x n, row stride n)
template <int G>
__device__ __forceinline__ void mm_sym(const Grp<G>& g, const Tables& T, int nk, const double* A, int ar, int ac,
                                       const double* B, int br, int bc, const double* C, double* D) {
  const int n = T.n;
  for (int e = g.gl; e < T.ntri; e += G) {
    const int i = T.tri_i[e], j = T.tri_j[e];
    double acc = C ? C[i * n + j] : 0.0;
    for (int l = 0; l < nk; ++l) acc = fma(A[i * ar + l * ac], B[l * br + j * bc], acc);
    D[i * n + j] = acc;
    D[j * n + i] = acc;
  }
}

