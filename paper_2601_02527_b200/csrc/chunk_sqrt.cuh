// chunk_sqrt.cuh -- the per-chunk recursions of k_down0 in SQUARE-ROOT (Cholesky-factor) form: SURVEY 8(f) item 1,
// the paper's own remedy for the conditioning of the covariance recursions (Yaghoobi et al. 2025).
//
// Same two passes as down0_body (chunk_kernels.cuh), same inputs, outputs and kbuf records, but no covariance and no
// adjoint matrix is ever formed: the filter carries S with P = S S^T, the adjoint (modified Bryson-Frazier) recursion
// carries W with Lambda = W W^T, and every step is "put the factors side by side, re-triangularise":
//   predict   S <- tria([F S | G]),  G G^T = Q~: G is assembled from the blocks' own Cholesky factors, which k_disc
//             writes in place of (Qxx, q12, q22) when the model asks for them (Q~ itself is singular);
//   reset     zero row z_q of S;
//   update    scalar observation h = hs e_z: Potter's form  S <- S - gamma (S phi) phi^T,  phi = S^T h,
//             s = phi^T phi + r,  gamma = 1 / (s + sqrt(r s)):  no subtraction of covariances;
//   adjoint   end event:  W <- tria([W - h (W^T K)^T | h / sqrt s]),   step:  W <- F^T W;
//   smoothed  H~ P^ H~^T = hs^2 (p_z - |W^T p|^2),  p = P_f e_z (kept in kbuf by the forward pass, as in down0_body).
// tria(M) = lower-triangular L with L L^T = M M^T: Householder reflections from the right, LANE i OWNS ROW i of M
// (odd row stride: conflict-free), the reflector's row is read as a broadcast, so a reflection needs no cross-lane
// reduction; reflectors are applied in the scale-free form v / |u| (information factors span hundreds of orders).
// Generic (statically compiled) kernel, matrices in shared memory; one group of lanes per chunk.
// Plan: one chunk per series (the sequential filter, row a8) -- the dense levels have no factor form yet.
#pragma once
#include "chunk_kernels.cuh"

// row stride of the stacked matrix [S | G] (n + d + nblk <= 2.5 n columns) and [W | extra] (n + 1 columns): odd
__host__ __device__ constexpr int sqrt_ldm(int ld) { return ((5 * ld) / 2) | 1; }
__host__ __device__ inline int sqrt_group_doubles(int n, int ld, int stride, int nblk, int G) {
  return ((ld - 1) * sqrt_ldm(ld) + 2 * stride + 2 + nblk * G + 6 * ld + 1) & ~1;
}

// L L^T = M M^T in place: M = n rows x m columns at row stride LDM; on return the lower triangle of the first n
// columns holds L and the rest of those columns is zero.  All lanes of the group call it.
template <int G, int LDM>
__device__ __forceinline__ void tria_rows(const Grp<G>& g, int n, int m, double* Mx) {
  const int i = g.gl;
  double* ri = Mx + (i < n ? i : 0) * LDM;
  for (int j = 0; j < n; ++j) {
    const double* rj = Mx + j * LDM;
    const bool act = (i > j) && (i < n);
    const double u0 = rj[j];
    double ss = u0 * u0, dd = 0.0;
    for (int c = j + 1; c < m; ++c) {
      const double uj = rj[c];
      ss = fma(uj, uj, ss);
      if (act) dd = fma(ri[c], uj, dd);
    }
    const double sig = sqrt(ss);
    double alpha = 0.0;
    if (sig > 0.0) { // the same for every lane
      alpha = u0 > 0.0 ? -sig : sig;
      const double v0 = (u0 - alpha) / sig;            // reflector v = (u - alpha e_j) / |u|
      const double beta = 1.0 / (1.0 + fabs(u0) / sig); // H = I - beta v v^T
      if (act) {
        const double w = beta * fma(ri[j], v0, dd / sig);
        ri[j] = fma(-w, v0, ri[j]);
        const double ws = w / sig;
        for (int c = j + 1; c < m; ++c) ri[c] = fma(-ws, rj[c], ri[c]);
      }
    }
    g.sync();
    if (i == j && sig > 0.0) ri[j] = alpha; // row j is final; its tail (the reflector) is cleared below
  }
  if (i < n)
    for (int c = i + 1; c < n; ++c) ri[c] = 0.0;
  g.sync();
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
  double* recs = Mx + NR * LDM;            // 2 x stride + 2 mbarriers
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* mv = recs + 2 * TSTRIDE + 2 + TNB * G; // filtered mean, later lambda
  double* pv = mv + LD;
  double* kv = pv + LD;
  double* bv = kv + LD;
  double* av = bv + LD;
  const int ks = kbuf_stride(n);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ampv = P.amp ? P.amp[series] : 1.0;
  const double ramp = 1.0 / ampv;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);
  const int i = g.gl;                      // the lane's row (tria, Potter update) and column (products with F)
  double* ri = Mx + (i < n ? i : 0) * LDM;

  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)TSTRIDE, 0);
  zero_fill(g, Mx, NR * LDM);
  zero_fill(g, mv, 5 * LD);
  g.sync();
  chol_psd_rows<G, LDM>(g, n, P.p0, n, Mx); // S0 S0^T = blkdiag(Pinf, 0)  (Eq. 3.19, reading R6)
  double ll = 0.0;
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
    if (i < n) apply_F<G, LDM, LDM>(T, rec, tz, Mx + i, Mx + i, U);
    else if (i == n) apply_F<G, 1, 1>(T, rec, tz, mv, mv, U);
    for (int cg = i; cg < nq; cg += G) {
      double* col = Mx + n + cg;
      for (int r = 0; r < n; ++r) col[r * LDM] = 0.0;
      for (int b = 0; b < nblk; ++b) {
        const int db = TBDIM(b), off = TBOFF(b), l = cg - off - b; // block b owns columns off + b .. off + b + db
        if (l < 0 || l > db) continue;
        const double* r = rec + TROFF(b);
        if (l < db)
          for (int r2 = l; r2 < db; ++r2) col[(off + r2) * LDM] = r[db * db + db + r2 * db + l]; // L_xx
        const double lz = r[2 * db * db + db + l];                                               // L_zx[l], or L_zz at l = db
        for (int p = 0; p < TNI; ++p)
          if (!((tz >> p) & 1u)) col[(d + p) * LDM] = TCZ(p * nblk + b) * lz;
      }
    }
    g.sync();
    tria_rows<G, LDM>(g, n, n + nq, Mx);
    if (!kind) {
      const int zi = d + q;
      const double hs = TTAU(q) / dl_r;
      const double sg = sg_r * ramp;
      const double yy = y_r * ramp;
      if (i < n) pv[i] = hs * Mx[zi * LDM + i]; // phi = S^T h
      g.sync();
      double ss = 0.0, a = 0.0;
      for (int c = 0; c < n; ++c) { const double f = pv[c]; ss = fma(f, f, ss); if (i < n) a = fma(ri[c], f, a); } // a = (S phi)_i = (P h)_i
      const double S = ss + sg * sg;
      const double v = yy - hs * mv[zi];
      if (!(sg_r > 0.0) || !isfinite(sg_r)) atomicOr(P.flags, NUMF_SIGMA);
      if (!(S > 0.0) || !isfinite(S) || !isfinite(v)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      ll -= 0.5 * (log(6.283185307179586476925286766559 * S) + v * v * rS);
      const double gam = 1.0 / (S + sqrt(sg * sg * S));
      g.sync(); // every lane has read m_z
      if (i < n) {
        const double ga = gam * a;
        for (int c = 0; c < n; ++c) ri[c] = fma(-ga, pv[c], ri[c]);
        mv[i] = fma(a * rS, v, mv[i]);
        kv[i] = a * rS;
      }
      g.sync();
      if (P.want_smooth) {
        if (i < n) bv[i] = Mx[zi * LDM + i]; // row z of the updated factor
        g.sync();
        double* kb = P.kbuf + (series * P.N + ob) * (int64_t)ks;
        if (i < n) {
          double p = 0.0;
          for (int c = 0; c < n; ++c) p = fma(ri[c], bv[c], p); // P_f e_z
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
  }
  if (g.gl == 0) P.llpart[gid] = ll;
  if (!P.want_smooth) return;

  // ---- backward: adjoint recursion with Lambda = W W^T (zero after the last event of the series) ----
  rs.issue(g, P.disc + (k1 - 1) * (int64_t)TSTRIDE, 0);
  zero_fill(g, Mx, NR * LDM);
  zero_fill(g, mv, LD);
  g.sync();
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
        for (int r = 0; r < n; ++r) { const double x = Mx[r * LDM + i]; a = fma(x, pv[r], a); b = fma(x, kv[r], b); } // (W^T p)_i, (W^T K)_i
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
    if (k == k0) break;
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    if (i < n) apply_Ft<G, LDM, LDM>(T, rec, tz, Mx + i, Mx + i);
    else if (i == n) apply_Ft<G, 1, 1>(T, rec, tz, mv, mv);
    g.sync();
  }
}

template <int G, int LD>
__global__ void __launch_bounds__(128) k_down0_sqrt(const __grid_constant__ ScanDev P) { down0_sqrt_body<G, LD>(P); }
