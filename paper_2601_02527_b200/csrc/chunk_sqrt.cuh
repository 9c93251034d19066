// chunk_sqrt.cuh -- the per-chunk recursions of k_down0 in SQUARE-ROOT (Cholesky-factor) form: SURVEY 8(f) item 1,
// the paper's own remedy for the conditioning of the covariance recursions (Yaghoobi et al. 2025).
//
// Same two passes as down0_body (chunk_kernels.cuh), same inputs, outputs and kbuf records, but no covariance and no
// adjoint matrix is ever formed: the filter carries S with P = S S^T, the adjoint (modified Bryson-Frazier) recursion
// carries W with Lambda = W W^T, and every step is "put the factors side by side, re-triangularise":
//   predict   S <- tria([F S | G]),  G G^T = Q~: G is assembled from the blocks' own Cholesky factors, which k_disc
//             writes in place of (Qxx, q12, q22) when the model asks for them (Q~ itself is singular);
//   reset     zero row z_q of S;
//   update    scalar observation h = hs e_z: Carlson's triangular form (carlson_rows: column j of S becomes a
//             combination of itself and of the columns after it, so S STAYS lower triangular): no subtraction of
//             covariances, and the next [F S | G] is block lower triangular -- the triangularisation skips the zeros;
//   adjoint   end event:  W <- tria([W - h (W^T K)^T | h / sqrt s]),   step:  W <- F^T W;
//   smoothed  H~ P^ H~^T = hs^2 (p_z - |W^T p|^2),  p = P_f e_z (kept in kbuf by the forward pass, as in down0_body).
// tria(M) = lower-triangular L with L L^T = M M^T: Householder reflections from the right, LANE i OWNS ROW i of M
// (odd row stride: conflict-free), the reflector's row is read as a broadcast, so a reflection needs no cross-lane
// reduction; reflectors are applied in the scale-free form v / |u| (information factors span hundreds of orders).
// Generic (statically compiled) kernels, matrices in shared memory; one group of lanes per chunk.
// Chunked scan: k_fold0_sqrt folds a chunk into ONE element (A, b, U, eta, Z) with C = U U^T, J = Z Z^T (the recursion of
// fold0_body with C -> U by tria and the triangular update, J += a a^T / s as Z <- tria([Z | a / sqrt s])); the dense levels combine
// such elements in factor form (dense_sqrt.cuh); k_down0_sqrt starts from the chunk's prefix state [m | S] and from the
// chunk-end adjoint  W = Z T'^-T,  T' T'^T = I + (S^T Z)^T (S^T Z),  of the suffix information [eta | Z].
#pragma once
#include "chunk_kernels.cuh"

// row stride of the stacked matrix [S | G] (n + d + nblk <= 2.5 n columns) and [W | extra] (n + 1 columns): odd
__host__ __device__ constexpr int sqrt_ldm(int ld) { return ((5 * ld) / 2) | 1; }
__host__ __device__ inline int sqrt_group_doubles(int n, int ld, int stride, int nblk, int G) {
  return (2 * (ld - 1) * sqrt_ldm(ld) + 2 * stride + 2 + nblk * G + 7 * ld + 1) & ~1;
}
__host__ __device__ inline int fold0s_group_doubles(int n, int ld, int stride, int nblk, int G) {
  return ((ld - 1) * sqrt_ldm(ld) + 2 * (ld - 1) * ld + 2 * stride + 2 + nblk * G + 8 * ld + 1) & ~1;
}

// One reflection of tria, columns c0..m-1 of the reflector's row rj and of the lane's own row ri.  The loops are
// unrolled by hand with the loads ahead of the arithmetic: the trip count is a run-time value and ri / rj may alias as
// far as the compiler knows, so a plain loop runs one shared-memory round trip per column (measured: 3x slower).
__device__ __forceinline__ void hh_dots(const double* rj, const double* ri, int c0, int m, bool act, double& ss, double& dd) {
  double s0 = 0.0, s1 = 0.0, d0 = 0.0, d1 = 0.0;
  int c = c0;
  for (; c + 3 < m; c += 4) {
    const double u0 = rj[c], u1 = rj[c + 1], u2 = rj[c + 2], u3 = rj[c + 3];
    double x0 = 0.0, x1 = 0.0, x2 = 0.0, x3 = 0.0;
    if (act) { x0 = ri[c]; x1 = ri[c + 1]; x2 = ri[c + 2]; x3 = ri[c + 3]; }
    s0 = fma(u0, u0, s0); s1 = fma(u1, u1, s1); s0 = fma(u2, u2, s0); s1 = fma(u3, u3, s1);
    d0 = fma(x0, u0, d0); d1 = fma(x1, u1, d1); d0 = fma(x2, u2, d0); d1 = fma(x3, u3, d1);
  }
  for (; c < m; ++c) {
    const double u0 = rj[c];
    s0 = fma(u0, u0, s0);
    if (act) d0 = fma(ri[c], u0, d0);
  }
  ss += s0 + s1;
  dd += d0 + d1;
}
__device__ __forceinline__ void hh_axpy(const double* rj, double* ri, int c0, int m, double ws) {
  int c = c0;
  for (; c + 3 < m; c += 4) {
    const double u0 = rj[c], u1 = rj[c + 1], u2 = rj[c + 2], u3 = rj[c + 3];
    const double x0 = ri[c], x1 = ri[c + 1], x2 = ri[c + 2], x3 = ri[c + 3];
    ri[c] = fma(-ws, u0, x0); ri[c + 1] = fma(-ws, u1, x1); ri[c + 2] = fma(-ws, u2, x2); ri[c + 3] = fma(-ws, u3, x3);
  }
  for (; c < m; ++c) ri[c] = fma(-ws, rj[c], ri[c]);
}

// column sums  a = sum_r col[r * st] p[r],  b = sum_r col[r * st] k[r]  (same hand unrolling)
__device__ __forceinline__ void col_dots2(const double* col, int st, const double* p, const double* k, int n, double& a, double& b) {
  double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
  int r = 0;
  for (; r + 3 < n; r += 4) {
    const double x0 = col[r * st], x1 = col[(r + 1) * st], x2 = col[(r + 2) * st], x3 = col[(r + 3) * st];
    a0 = fma(x0, p[r], a0); a1 = fma(x1, p[r + 1], a1); a0 = fma(x2, p[r + 2], a0); a1 = fma(x3, p[r + 3], a1);
    b0 = fma(x0, k[r], b0); b1 = fma(x1, k[r + 1], b1); b0 = fma(x2, k[r + 2], b0); b1 = fma(x3, k[r + 3], b1);
  }
  for (; r < n; ++r) { const double x = col[r * st]; a0 = fma(x, p[r], a0); b0 = fma(x, k[r], b0); }
  a = a0 + a1; b = b0 + b1;
}
// col[r * st] += f v[r]
__device__ __forceinline__ void col_axpy(double* col, int st, const double* v, int n, double f) {
  int r = 0;
  for (; r + 3 < n; r += 4) {
    const double x0 = col[r * st], x1 = col[(r + 1) * st], x2 = col[(r + 2) * st], x3 = col[(r + 3) * st];
    const double v0 = v[r], v1 = v[r + 1], v2 = v[r + 2], v3 = v[r + 3];
    col[r * st] = fma(v0, f, x0); col[(r + 1) * st] = fma(v1, f, x1); col[(r + 2) * st] = fma(v2, f, x2); col[(r + 3) * st] = fma(v3, f, x3);
  }
  for (; r < n; ++r) col[r * st] = fma(v[r], f, col[r * st]);
}

// L L^T = M M^T in place: M = n rows x m columns at row stride LDM; on return the lower triangle of the first n
// columns holds L and the rest of those columns is zero.  All lanes of the group call it.
// e1t / g1t (optional): row j of M is known to be zero outside the columns [0, e1t[j]) and [n, g1t[j]), with both
// bounds non-decreasing in j (the stacked matrix [F S | G] of a predict step with S lower triangular: F is block
// diagonal over the components plus the dense integral rows, G has one group of columns per block); the reflections
// then touch those columns only, and the nesting of the supports keeps every later row inside its own.
template <int G, int LDM>
__device__ __forceinline__ void tria_rows(const Grp<G>& g, int n, int m, double* Mx, const short* e1t = nullptr, const short* g1t = nullptr) {
  const int i = g.gl;
  double* ri = Mx + (i < n ? i : 0) * LDM;
  for (int j = 0; j < n; ++j) {
    const double* rj = Mx + j * LDM;
    const bool act = (i > j) && (i < n);
    const double u0 = rj[j];
    double ss = u0 * u0, dd = 0.0;
    const int c1 = e1t ? (int)e1t[j] : m, c2 = e1t ? (int)g1t[j] : m;
    hh_dots(rj, ri, j + 1, c1, act, ss, dd);
    if (e1t) hh_dots(rj, ri, n, c2, act, ss, dd);
    const double sig = sqrt(ss);
    double alpha = 0.0;
    if (sig > 0.0) { // the same for every lane
      alpha = u0 > 0.0 ? -sig : sig;
      const double rsig = 1.0 / sig;                    // (sig > 0 in fp64 after a sum of squares: >= 1e-162, no overflow)
      const double v0 = (u0 - alpha) * rsig;            // reflector v = (u - alpha e_j) / |u|
      const double beta = 1.0 / (1.0 + fabs(u0) * rsig); // H = I - beta v v^T
      if (act) {
        const double w = beta * fma(ri[j], v0, dd * rsig);
        ri[j] = fma(-w, v0, ri[j]);
        hh_axpy(rj, ri, j + 1, c1, w * rsig);
        if (e1t) hh_axpy(rj, ri, n, c2, w * rsig);
      }
    }
    g.sync();
    if (i == j && sig > 0.0) ri[j] = alpha; // row j is final; its tail (the reflector) is cleared below
  }
  if (i < n)
    for (int c = i + 1; c < n; ++c) ri[c] = 0.0;
  g.sync();
}

// supports of the rows of [F S | G] for a lower-triangular S (see tria_rows): row j of block b is zero outside
// [0, off_b + d_b) and [n, n + off_b + b + d_b + 1) -- its own and the earlier blocks' columns of G; integral rows are full
template <int G>
__device__ __forceinline__ void sq_tables(const Grp<G>& g, const Tab& T, short* e1t, short* g1t) {
  const int n = TN, d = TD;
  for (int j = g.gl; j < n; j += G) {
    if (j < d) { const int b = T.blk_of[j]; e1t[j] = (short)(TBOFF(b) + TBDIM(b)); g1t[j] = (short)(n + TBOFF(b) + b + TBDIM(b) + 1); }
    else { e1t[j] = (short)n; g1t[j] = (short)(n + d + TNB); }
  }
  g.sync();
}
// row i of G (columns n..): cleared over the row's support, then its own entries -- row-owned, no other lane writes it.
// x row of block b: row (i - off_b) of L_xx in the block's columns; integral row p: c_pb (L_zx | L_zz) for every block.
__device__ __forceinline__ void sq_fill_G_row(const Tab& T, const double* rec, unsigned tz, int i, double* ri, int g1) {
  const int n = TN, d = TD, nblk = TNB;
  for (int c = n; c < g1; ++c) ri[c] = 0.0;
  if (i < d) {
    const int b = T.blk_of[i], db = TBDIM(b), off = TBOFF(b), lr = i - off;
    const double* r = rec + TROFF(b) + db * db + db + lr * db;
    double* o = ri + n + off + b;
    for (int l = 0; l <= lr; ++l) o[l] = r[l];
  } else if (!((tz >> (i - d)) & 1u)) {
    const int p = i - d;
    for (int b = 0; b < nblk; ++b) {
      const double c = TCZ(p * nblk + b);
      if (c == 0.0) continue;
      const int db = TBDIM(b);
      const double* r = rec + TROFF(b) + 2 * db * db + db;
      double* o = ri + n + TBOFF(b) + b;
      for (int l = 0; l <= db; ++l) o[l] = c * r[l];
    }
  }
}
// Scalar measurement update of a LOWER-TRIANGULAR factor that keeps it lower triangular (Carlson's form, columns
// taken from the last to the first): with f = S^T h, alpha_j = r + sum_{c > j} f_c^2,
//   S+[:, j] = sqrt(alpha_j / alpha'_j) S[:, j] - f_j / sqrt(alpha_j alpha'_j) e_j,   alpha'_j = alpha_j + f_j^2,
//   e_j = sum_{c > j} S[:, c] f_c;   at the end alpha' = s = h^T P h + r and e = P h.
// Row-owned (lane i updates row i, entries 0..i); the scalars are computed one column per lane first (bt, gm: n each).
// Returns s; a = (P h)_i.  Nothing is subtracted from a covariance.
template <int G>
__device__ __forceinline__ double carlson_rows(const Grp<G>& g, int n, double* ri, const double* f, double r, double* bt, double* gm, double& a) {
  const int i = g.gl;
  double tot = r;
  if (i < n) {
    double al = r;
    for (int c = n - 1; c > i; --c) al = fma(f[c], f[c], al);
    const double fi = f[i], al2 = fma(fi, fi, al);
    const double q = 1.0 / al2;
    bt[i] = sqrt(al * q);
    gm[i] = fi * q * sqrt(al2 / al);
  }
  for (int c = 0; c < n; ++c) tot = fma(f[c], f[c], tot);
  g.sync();
  double e = 0.0;
  if (i < n) {
    for (int j = i; j >= 0; --j) {
      const double x = ri[j];
      ri[j] = fma(bt[j], x, -gm[j] * e);
      e = fma(x, f[j], e);
    }
  }
  a = e;
  return tot;
}

// lower Cholesky factor of a positive SEMI-definite n x n matrix A (element (i, j) at A[i * lda + j]) into the first n
// columns of Mx (row stride LDM): a pivot that rounding has driven to <= 2^-44 of its diagonal entry gives a zero
// column (idle integral states have exact zero rows).  Once per chunk: done serially by one lane.
template <int G, int LDM>
__device__ __forceinline__ void chol_psd_rows(const Grp<G>& g, int n, const double* A, int lda, double* Mx) {
  if (g.gl == 0) {
    for (int j = 0; j < n; ++j) {
      for (int i = 0; i < j; ++i) Mx[i * LDM + j] = 0.0;
      double p = A[j * lda + j];
      for (int k = 0; k < j; ++k) p = fma(-Mx[j * LDM + k], Mx[j * LDM + k], p);
      if (!(p > A[j * lda + j] * 5.7e-14)) {
        for (int i = j; i < n; ++i) Mx[i * LDM + j] = 0.0;
        continue;
      }
      const double r = sqrt(p), rr = 1.0 / r;
      Mx[j * LDM + j] = r;
      for (int i = j + 1; i < n; ++i) {
        double a = A[i * lda + j];
        for (int k = 0; k < j; ++k) a = fma(-Mx[i * LDM + k], Mx[j * LDM + k], a);
        Mx[i * LDM + j] = a * rr;
      }
    }
  }
  g.sync();
}

template <int G, int LD>
__device__ __forceinline__ void down0_sqrt_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int LDM = sqrt_ldm(LD);
  constexpr int NR = LD - 1;
  const int n = TN, d = TD, nblk = TNB, nq = TD + TNB;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)smem + (size_t)(threadIdx.x / G) * sqrt_group_doubles(n, LD, TSTRIDE, TNB, G);
  double* Mx = base;                       // [S | G], later [W | extra column]
  double* Bx = Mx + NR * LDM;              // second stacked matrix: the chunk-end adjoint is built here
  double* recs = Bx + NR * LDM;            // 2 x stride + 2 mbarriers
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* mv = recs + 2 * TSTRIDE + 2 + TNB * G; // filtered mean, later lambda
  double* pv = mv + LD;
  double* kv = pv + LD;
  double* bv = kv + LD;
  double* av = bv + LD;
  short* e1t = (short*)(av + LD);          // supports of the rows of [F S | G] (sq_tables)
  short* g1t = e1t + 2 * LD;
  const int ks = kbuf_stride(n);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ampv = P.amp ? P.amp[series] : 1.0;
  const double ramp = 1.0 / ampv;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);
  const int i = g.gl;                      // the lane's row (tria, triangular update) and column (products with F)
  double* ri = Mx + (i < n ? i : 0) * LDM;

  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)TSTRIDE, 0);
  zero_fill(g, Mx, NR * LDM);
  zero_fill(g, mv, 5 * LD);
  sq_tables(g, T, e1t, g1t);
  if (P.PRE1) { // the chunk's prefix state [m | S] from the dense levels
    const double* sp = P.PRE1 + gid * (int64_t)state_size(n);
    for (int c = i; c <= n; c += G)
      for (int r = 0; r < n; ++r) { if (c < n) Mx[r * LDM + c] = sp[n + r * n + c]; else mv[r] = sp[r]; }
    g.sync();
  } else chol_psd_rows<G, LDM>(g, n, P.p0, n, Mx); // S0 S0^T = blkdiag(Pinf, 0)  (Eq. 3.19, reading R6)
  double ll = 0.0;
#ifdef SG_SQ_CLK
  long long c_prev = clock64();
#endif
  // ---- forward: square-root Kalman filter ----
  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const double* rec = rs.wait((int)((k - k0) & 1));
    g.sync();
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)TSTRIDE, (int)((k + 1 - k0) & 1));
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    // [F S | G]: lane c applies F to column c of S in place (a block is read before it is written, the z rows
    // last), lane n to the mean; then the lanes write G's columns
#ifdef SG_SQ_CLK
    const long long c_0 = clock64();
#endif
    if (i < n) apply_F<G, LDM, LDM>(T, rec, tz, Mx + i, Mx + i, U);
    else if (i == n) apply_F<G, 1, 1>(T, rec, tz, mv, mv, U);
#ifdef SG_SQ_CLK
    const long long c_1 = clock64();
#endif
    g.sync(); // F S complete: the rows are written next
    if (i < n) sq_fill_G_row(T, rec, tz, i, ri, g1t[i]);
    g.sync();
#ifdef SG_SQ_CLK
    const long long c_2 = clock64();
#endif
    tria_rows<G, LDM>(g, n, n + nq, Mx, e1t, g1t);
#ifdef SG_SQ_CLK
    const long long c_3 = clock64();
    if (gid == 0 && i == 0 && (k - k0) == 20) printf("down0_sqrt fwd event: applyF %lld  Gfill %lld  tria %lld  (prev event total %lld)\n", c_1 - c_0, c_2 - c_1, c_3 - c_2, c_0 - c_prev);
    c_prev = c_0;
#endif
    if (!kind) {
      const int zi = d + q;
      const double hs = TTAU(q) / dl_r;
      const double sg = sg_r * ramp;
      const double yy = y_r * ramp;
      if (i < n) pv[i] = hs * Mx[zi * LDM + i]; // phi = S^T h
      g.sync();
      const double v = yy - hs * mv[zi];
      if (!(sg_r > 0.0) || !isfinite(sg_r)) atomicOr(P.flags, NUMF_SIGMA);
      double a = 0.0;
      const double S = (sg > 0.0) ? carlson_rows(g, n, ri, pv, sg * sg, av, bv, a) : 0.0; // S stays lower triangular; a = (P h)_i
      if (!(S > 0.0) || !isfinite(S) || !isfinite(v)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      ll -= 0.5 * (log(6.283185307179586476925286766559 * S) + v * v * rS);
      g.sync(); // every lane has read m_z; the rows are updated
      if (i < n) {
        mv[i] = fma(a * rS, v, mv[i]);
        kv[i] = a * rS;
      }
      g.sync();
      if (P.want_smooth) {
        if (i < n) bv[i] = Mx[zi * LDM + i]; // row z of the updated factor
        g.sync();
        double* kb = P.kbuf + (series * P.N + ob) * (int64_t)ks;
        if (i < n) {
          double p = 0.0, dummy = 0.0;
          hh_dots(bv, ri, 0, n, true, dummy, p); // P_f e_z
          kb[i] = kv[i];
          kb[n + i] = p;
        }
        if (i == 0) { kb[2 * n] = S; kb[2 * n + 1] = v; kb[2 * n + 2] = mv[zi]; }
        g.sync();
      }
      // the instrument is idle after its end (reading R6)
      if (i == zi) { for (int c = 0; c < n; ++c) ri[c] = 0.0; mv[zi] = 0.0; }
      g.sync();
    }
    if (P.fstate) { // row a7: the post-event filtered state [m | S] of every event
      double* fs = P.fstate + (series * P.K + k) * (int64_t)state_size(n);
      for (int c = i; c <= n; c += G)
        for (int r = 0; r < n; ++r) { if (c < n) fs[n + r * n + c] = Mx[r * LDM + c]; else fs[r] = mv[r]; }
    }
  }
  if (g.gl == 0) P.llpart[gid] = ll;
  if (!P.want_smooth) return;

  // ---- backward: adjoint recursion with Lambda = W W^T (zero after the last event of the series) ----
  rs.issue(g, P.disc + (k1 - 1) * (int64_t)TSTRIDE, 0);
  if (P.SUF1 && chunk + 1 < P.c1) {
    // adjoint at the chunk's last event from the suffix information [eta | Z] about the state after the chunk and
    // the filtered state (m, S) there:  Lambda^ = (I + J P)^-1 J = W W^T with W = Z T'^-T, T' T'^T = I + V^T V,
    // V = S^T Z;  lambda^ = (I + J P)^-1 (J m - eta) = u - W W^T P u,  u = Z Z^T m - eta
    const double* sj = P.SUF1 + gid * (int64_t)state_size(n);
    for (int c = i; c <= n; c += G)
      for (int r = 0; r < n; ++r) { if (c < n) Bx[r * LDM + c] = sj[n + r * n + c]; else pv[r] = sj[r]; }
    g.sync();
    if (i < n) { double a = 0.0; for (int r = 0; r < n; ++r) a = fma(Bx[r * LDM + i], mv[r], a); kv[i] = a; }            // Z^T m
    g.sync();
    double* bi = Bx + (i < n ? i : 0) * LDM;
    if (i < n) { double a = -pv[i]; for (int c = 0; c < n; ++c) a = fma(bi[c], kv[c], a); bv[i] = a; }                     // u
    g.sync();
    if (i < n) { double a = 0.0; for (int r = 0; r < n; ++r) a = fma(Mx[r * LDM + i], bv[r], a); kv[i] = a; }            // S^T u
    g.sync();
    if (i < n) { double a = 0.0; for (int c = 0; c < n; ++c) a = fma(ri[c], kv[c], a); av[i] = a; }                        // P u
    if (i < n)                                                                                                             // column i of V^T = Z^T S
      for (int r2 = 0; r2 < n; ++r2) { double a = 0.0; for (int r = 0; r < n; ++r) a = fma(Bx[r * LDM + r2], Mx[r * LDM + i], a); Bx[r2 * LDM + n + i] = a; }
    g.sync();
    if (i < n)
      for (int c = 0; c < n; ++c) { ri[c] = (c == i) ? 1.0 : 0.0; ri[n + c] = bi[n + c]; }                                 // Mx = [I | V^T]
    g.sync();
    tria_rows<G, LDM>(g, n, 2 * n, Mx);                                                                                    // T'
    if (i < n)
      for (int c = 0; c < n; ++c) { double a = bi[c]; for (int k2 = 0; k2 < c; ++k2) a = fma(-Mx[c * LDM + k2], bi[k2], a); bi[c] = a / Mx[c * LDM + c]; } // row i of W
    g.sync();
    if (i < n) { double a = 0.0; for (int r = 0; r < n; ++r) a = fma(Bx[r * LDM + i], av[r], a); kv[i] = a; }            // W^T P u
    g.sync();
    if (i < n) {
      double a = bv[i];
      for (int c = 0; c < n; ++c) a = fma(-bi[c], kv[c], a);
      mv[i] = a;                                                                                                           // lambda^
      for (int c = 0; c < n; ++c) ri[c] = bi[c];
      ri[n] = 0.0;
    }
    g.sync();
  } else {
    zero_fill(g, Mx, NR * LDM);
    zero_fill(g, mv, LD);
    g.sync();
  }
  uint32_t meta_b = P.meta[k1 - 1];
  int32_t ob_b = P.obs[k1 - 1];
  for (int64_t k = k1 - 1; k >= k0; --k) {
    const double* rec = rs.wait((int)((k1 - 1 - k) & 1));
    g.sync();
    if (k > k0) rs.issue(g, P.disc + (k - 1) * (int64_t)TSTRIDE, (int)((k1 - k) & 1));
    const uint32_t meta = meta_b;
    const int32_t ob = ob_b;
    if (k > k0) { meta_b = P.meta[k - 1]; ob_b = P.obs[k - 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    // components zeroed after event k pass nothing backwards (adjoint of the zeroing)
    if (i >= d && i < n && ((zm >> (i - d)) & 1u)) { for (int c = 0; c < n; ++c) ri[c] = 0.0; mv[i] = 0.0; }
    g.sync();
    if (!kind) {
      const int zi = d + q;
      const double* kb = P.kbuf + (series * P.N + ob) * (int64_t)ks;
      const double S = kb[2 * n], v = kb[2 * n + 1], mfz = kb[2 * n + 2];
      const double hs = TTAU(q) / P.delta[k];
      if (i < n) { kv[i] = kb[i]; pv[i] = kb[n + i]; }
      const double rS = 1.0 / S;
      g.sync();
      double a = 0.0, b = 0.0, lp = 0.0, lk = 0.0;
      if (i < n) {
        col_dots2(Mx + i, LDM, pv, kv, n, a, b); // (W^T p)_i, (W^T K)_i
        lp = mv[i] * pv[i];
        lk = mv[i] * kv[i];
      }
      const double quad = group_sum(g, a * a);
      lp = group_sum(g, lp);
      lk = group_sum(g, lk);
      if (i == 0) {
        const double sm = mfz - lp, sv = pv[zi] - quad;
        if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
        P.mean[series * P.N + ob] = ampv * hs * sm;            // H~ m^
        P.var[series * P.N + ob] = ampv * ampv * hs * hs * sv; // H~ P^ H~^T
      }
      g.sync(); // pv[zi] has been read
      // W~ = [W - h (W^T K)^T | h / sqrt s],  lambda~ = lambda - h (K . lambda + v / s)
      if (i < n) {
        Mx[zi * LDM + i] = fma(-hs, b, Mx[zi * LDM + i]);
        Mx[i * LDM + n] = (i == zi) ? hs * sqrt(rS) : 0.0;
        if (i == zi) mv[zi] -= hs * (lk + v * rS);
      }
      g.sync();
      tria_rows<G, LDM>(g, n, n + 1, Mx);
    }
    if (P.binfo) { // row a7: the pre-update adjoint [lambda~ | W~] of every event
      double* bs = P.binfo + (series * P.K + k) * (int64_t)state_size(n);
      for (int c = i; c <= n; c += G)
        for (int r = 0; r < n; ++r) { if (c < n) bs[n + r * n + c] = Mx[r * LDM + c]; else bs[r] = mv[r]; }
    }
    if (k == k0) break;
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    if (i < n) apply_Ft<G, LDM, LDM>(T, rec, tz, Mx + i, Mx + i);
    else if (i == n) apply_Ft<G, 1, 1>(T, rec, tz, mv, mv);
    g.sync();
  }
}

// chunk -> one element in factor form
template <int G, int LD>
__device__ __forceinline__ void fold0_sqrt_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int LDM = sqrt_ldm(LD);
  constexpr int NR = LD - 1, ld = LD;
  const int n = TN, d = TD, nblk = TNB, nq = TD + TNB;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)smem + (size_t)(threadIdx.x / G) * fold0s_group_doubles(n, LD, TSTRIDE, TNB, G);
  double* Mx = base;                       // [U | G]
  double* AB = Mx + NR * LDM;              // [A | b], column-owned, row stride LD
  double* Bx = AB + NR * ld;               // [Z | extra column], row stride LD
  double* recs = Bx + NR * ld;
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* ev = recs + 2 * TSTRIDE + 2 + TNB * G; // eta
  double* pv = ev + LD;
  double* cv = pv + LD;
  double* av = cv + LD;                    // n + 1
  double* bt = av + LD;                    // scalars of the triangular update (carlson_rows)
  double* gm = bt + LD;
  short* e1t = (short*)(gm + LD);
  short* g1t = e1t + 2 * LD;
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ramp = P.amp ? 1.0 / P.amp[series] : 1.0;
  const int i = g.gl;
  double* ri = Mx + (i < n ? i : 0) * LDM;

  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)TSTRIDE, 0);
  zero_fill(g, Mx, NR * LDM + 2 * NR * ld);
  zero_fill(g, ev, 6 * LD);
  sq_tables(g, T, e1t, g1t);
  for (int r = i; r < n; r += G) AB[r * ld + r] = 1.0;
  g.sync();
  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const double* rec = rs.wait((int)((k - k0) & 1));
    g.sync();
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)TSTRIDE, (int)((k + 1 - k0) & 1));
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    // [A | b] <- F [A | b];  U <- tria([F U | G])
    if (i <= n) apply_F<G, LD, LD>(T, rec, tz, AB + i, AB + i, U);
    if (i < n) apply_F<G, LDM, LDM>(T, rec, tz, Mx + i, Mx + i, U);
    g.sync(); // F U complete: the rows are written next
    if (i < n) sq_fill_G_row(T, rec, tz, i, ri, g1t[i]);
    g.sync();
    tria_rows<G, LDM>(g, n, n + nq, Mx, e1t, g1t);
    if (!kind) {
      // fold the end event's primitive element onto the aggregate (SG21 Eq. 10, rank-one J_j: fold0_body), in factors
      const int zi = d + q;
      const double hs = TTAU(q) / dl_r;
      const double sg = sg_r * ramp;
      const double yy = y_r * ramp;
      if (i < n) pv[i] = hs * Mx[zi * LDM + i];       // phi = U^T h
      if (i <= n) av[i] = hs * AB[zi * ld + i];       // a = A^T h (entry n: h . b)
      g.sync();
      double a = 0.0;
      const double S = (sg > 0.0) ? carlson_rows(g, n, ri, pv, sg * sg, bt, gm, a) : 0.0; // C -= c c^T / s on the factor, kept lower triangular
      if (!(S > 0.0) || !isfinite(S)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S, resid = yy - av[n];
      if (i < n) {
        cv[i] = a;                                    // c = C h
        ev[i] = fma(av[i], resid * rS, ev[i]);        // eta += a resid / s
        Bx[i * ld + n] = av[i] * sqrt(rS);            // J += a a^T / s
      }
      g.sync();
      if (i <= n) { // column i of A -= c a_i / s;  b += c resid / s
        const double f = (i < n) ? -av[i] * rS : resid * rS;
        col_axpy(AB + i, ld, cv, n, f);
      }
      tria_rows<G, LD>(g, n, n + 1, Bx);
      // the instrument is idle after its end: zero z_q (reading R6)
      if (i <= n) AB[zi * ld + i] = 0.0;
      if (i == zi) for (int c = 0; c < n; ++c) ri[c] = 0.0;
      g.sync();
    }
  }
  double* out = P.E1 + gid * (int64_t)elem_size(n);
  const int n1 = n + 1;
  for (int j = i; j <= n; j += G)
    for (int r = 0; r < n; ++r) {
      out[r * n1 + j] = AB[r * ld + j];
      out[n * n1 + n * n + r * n1 + j] = (j < n) ? Bx[r * ld + j] : ev[r];
      if (j < n) out[n * n1 + r * n + j] = Mx[r * LDM + j];
    }
}

template <int G, int LD>
__global__ void __launch_bounds__(128) k_fold0_sqrt(const __grid_constant__ ScanDev P) { fold0_sqrt_body<G, LD>(P); }
template <int G, int LD>
__global__ void __launch_bounds__(128) k_down0_sqrt(const __grid_constant__ ScanDev P) { down0_sqrt_body<G, LD>(P); }

// ---------------------------------------------------------------------------------------------------
// Row a7 in factor form (query_body of chunk_kernels.cuh): the filtered factor after the last event at or before t*
// is predicted over Delta_1 (one triangularisation), the pre-update adjoint factor of the next event is stepped back
// over Delta_2 (W* = F_2^T W~: no triangularisation), and
//   H_q m^ = h . m* - lambda* . p,   H_q P^ H_q^T = |S*^T h|^2 - |W*^T p|^2,   p = P* h = S* (S*^T h).
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int querys_group_doubles(int n, int ld, int stride, int nblk, int G) {
  return ((ld - 1) * sqrt_ldm(ld) + (ld - 1) * ld + 2 * stride + 2 + nblk * G + 6 * ld + 1) & ~1;
}

template <int G, int LD>
__device__ __forceinline__ void query_sqrt_body(const QueryDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int LDM = sqrt_ldm(LD);
  constexpr int NR = LD - 1, ld = LD;
  const int n = TN, d = TD, nblk = TNB, nq = TD + TNB;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.Mq) return;
  double* base = (double*)smem + (size_t)(threadIdx.x / G) * querys_group_doubles(n, LD, TSTRIDE, TNB, G);
  double* Mx = base;                 // [S | G]
  double* Wx = Mx + NR * LDM;        // W, row stride LD
  double* recs = Wx + NR * ld;
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* mv = recs + 2 * TSTRIDE + 2 + TNB * G;
  double* lam = mv + LD;
  double* hv = lam + LD;
  double* t1 = hv + LD;
  double* ph = t1 + LD;
  short* e1t = (short*)(ph + LD);
  short* g1t = e1t + 2 * LD;
  const int ss = state_size(n);
  const int64_t series = gid / P.Mq, q = gid - series * P.Mq;
  const int64_t kp = P.kp[q];
  const double ampv = P.amp ? P.amp[series] : 1.0;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);
  const int i = g.gl;
  double* ri = Mx + (i < n ? i : 0) * LDM;
  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.discq + q * (int64_t)TSTRIDE, 0);
  rs.issue(g, P.discq + (P.Mq + q) * (int64_t)TSTRIDE, 1);
  zero_fill(g, Mx, NR * LDM + NR * ld);
  zero_fill(g, mv, 5 * LD);
  sq_tables(g, T, e1t, g1t);
  if (i == 0)
    for (int b = 0; b < TNB; ++b) hv[TBOFF(b)] = ((P.T.bmask[b] >> P.qinst) & 1u) ? P.T.bsig[b] : 0.0; // H of the queried (virtual) instrument
  rs.wait(0);
  rs.wait(1);
  g.sync();
  if (kp >= 0) {
    const double* fs = P.fstate + (series * P.K + kp) * (int64_t)ss;
    for (int c = i; c <= n; c += G)
      for (int r = 0; r < n; ++r) { if (c < n) Mx[r * LDM + c] = fs[n + r * n + c]; else mv[r] = fs[r]; }
    g.sync();
    const uint32_t mp = P.meta[kp]; // idle through (t_kp, t_kp+1): zeroed after kp, except an instrument that just started
    const unsigned idle = META_KIND(mp) ? (META_ZMASK(mp) & ~(1u << META_INST(mp))) : META_ZMASK(mp);
    const double* rec = recs;
    if (i < n) apply_F<G, LDM, LDM>(T, rec, idle, Mx + i, Mx + i, U);
    else if (i == n) apply_F<G, 1, 1>(T, rec, idle, mv, mv, U);
    g.sync(); // F S complete: the rows are written next (S from the state store is lower triangular)
    if (i < n) sq_fill_G_row(T, rec, idle, i, ri, g1t[i]);
    g.sync();
    tria_rows<G, LDM>(g, n, n + nq, Mx, e1t, g1t);
  } else { // before the first event: the stationary prior, idle z = 0 (retrodiction, reading R8)
    chol_psd_rows<G, LDM>(g, n, P.p0, n, Mx);
  }
  const bool have_next = kp + 1 < P.K;
  if (have_next) {
    const int64_t kn = kp + 1;
    const double* bs = P.binfo + (series * P.K + kn) * (int64_t)ss;
    for (int c = i; c <= n; c += G)
      for (int r = 0; r < n; ++r) { if (c < n) Wx[r * ld + c] = bs[n + r * n + c]; else lam[r] = bs[r]; }
    g.sync();
    const uint32_t meta = P.meta[kn];
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = META_KIND(meta) ? zm : (zm & ~(1u << META_INST(meta)));
    if (i < n) apply_Ft<G, LD, LD>(T, recs + TSTRIDE, tz, Wx + i, Wx + i);
    else if (i == n) apply_Ft<G, 1, 1>(T, recs + TSTRIDE, tz, lam, lam);
    g.sync();
  }
  if (i < n) { double a = 0.0; for (int r = 0; r < n; ++r) a = fma(Mx[r * LDM + i], hv[r], a); t1[i] = a; } // S*^T h
  g.sync();
  double sv = 0.0, sm = 0.0;
  if (i < n) {
    double a = 0.0;
    for (int c = 0; c < n; ++c) a = fma(ri[c], t1[c], a);
    ph[i] = a;                                                                                             // P* h
    sv = t1[i] * t1[i];
    sm = hv[i] * mv[i];
  }
  g.sync();
  if (have_next && i < n) {
    double a = 0.0;
    for (int r = 0; r < n; ++r) a = fma(Wx[r * ld + i], ph[r], a);                                          // (W*^T p)_i
    sv -= a * a;
    sm -= lam[i] * ph[i];
  }
  sv = group_sum(g, sv);
  sm = group_sum(g, sm);
  if (i == 0) {
    if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
    P.mean[series * P.Mtot + P.q0 + q] = ampv * sm;
    P.var[series * P.Mtot + P.q0 + q] = ampv * ampv * sv;
  }
}

template <int G, int LD>
__global__ void __launch_bounds__(128) k_query_sqrt(const __grid_constant__ QueryDev P) { query_sqrt_body<G, LD>(P); }
