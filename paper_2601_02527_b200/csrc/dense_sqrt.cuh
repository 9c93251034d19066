// dense_sqrt.cuh -- the dense levels of the scan in SQUARE-ROOT (Cholesky-factor) form (
// the parallel square-root filter / smoother of Yaghoobi et al. 2025, restated for the filter elements of reading R1).
//
// An element is (A, b, U, eta, Z) with C = U U^T and J = Z Z^T, stored in the layout of the covariance form ([A | b], then U
// in C's place, then [Z | eta] in [J | eta]'s); a state is [m | S] with P = S S^T, a backward information [eta | Z].
// With V = U_i^T Z_j and the two triangularisations  T T^T = I + V V^T,  T' T'^T = I + V^T V  (tria = Householder
// reflections from the right, one warp, lane = row):
//   X  = U_i T^-T :   X X^T   = (I + C_i J_j)^-1 C_i = M C_i,      M   = I - X X^T J_j
//   X' = Z_j T'^-T :  X' X'^T = (I + J_j C_i)^-1 J_j = M^T J_j,    M^T = I - X' X'^T C_i
// and the combine of SURVEY App. A becomes
//   A = A_j M A_i,   b = A_j (b_i + X X^T u) + b_j,  u = eta_j - J_j b_i,      U = tria([A_j X | U_j]),
//   eta = A_i^T M^T u + eta_i,                                                 Z = tria([A_i^T X' | Z_i])
// (b in its "mean + gain x innovation" form: M (b_i + C_i eta_j) = b_i + M C_i (eta_j - J_j b_i), which does not
// form the large C_i eta_j only to cancel it).
// Nothing is subtracted from a covariance, no I + C J is ever formed or inverted (the only solves are with T, T':
// triangular, diagonal >= 1), and no product is compensated.  The prefix walk ((m, S) then an element) and the suffix
// walk (an element then (eta, Z)) are the same formulas with one side empty.  One CTA of SG_DENSE_NT threads per group.
#pragma once
#include "chunk_sqrt.cuh"
#include "dense_kernels.cuh"

// L L^T = M M^T in place (n rows, m columns, row stride ld), by ONE WARP: lane i owns row i; on return the lower
// triangle of the first n columns holds L, the rest of those columns is zero.  Reflectors in the scale-free form of
// chunk_sqrt.cuh.  n <= 32.
__device__ __forceinline__ void tria_warp(int n, int m, int ld, double* Mx) {
  const int i = threadIdx.x & 31;
  double* ri = Mx + (i < n ? i : 0) * ld;
  for (int j = 0; j < n; ++j) {
    const double* rj = Mx + j * ld;
    const bool act = (i > j) && (i < n);
    const double u0 = rj[j];
    double ss = u0 * u0, dd = 0.0;
    hh_dots(rj, ri, j + 1, m, act, ss, dd);
    const double sig = sqrt(ss);
    double alpha = 0.0;
    if (sig > 0.0) {
      alpha = u0 > 0.0 ? -sig : sig;
      const double rsig = 1.0 / sig;
      const double v0 = (u0 - alpha) * rsig;
      const double beta = 1.0 / (1.0 + fabs(u0) * rsig);
      if (act) {
        const double w = beta * fma(ri[j], v0, dd * rsig);
        ri[j] = fma(-w, v0, ri[j]);
        hh_axpy(rj, ri, j + 1, m, w * rsig);
      }
    }
    __syncwarp();
    if (i == j && sig > 0.0) ri[j] = alpha;
  }
  if (i < n)
    for (int c = i + 1; c < n; ++c) ri[c] = 0.0;
  __syncwarp();
}

// rows of X = F T^-T (n x n): lane i of ONE WARP solves T x = (row i of F)^T by forward substitution (T lower
// triangular with a non-zero diagonal, row stride lt; F row stride lf) and writes row i of X (row stride lx)
__device__ __forceinline__ void solve_rows_warp(int n, const double* T, int lt, const double* F, int lf, double* X, int lx) {
  const int i = threadIdx.x & 31;
  if (i < n) {
    for (int c = 0; c < n; ++c) {
      double a = F[i * lf + c];
      for (int k = 0; k < c; ++k) a = fma(-T[c * lt + k], X[i * lx + k], a);
      X[i * lx + c] = a / T[c * lt + c];
    }
  }
  __syncwarp();
}

// D[i,j] = (C ? C[i,j] : 0) + alpha sum_l A[i,l] B[l,j] with strided operands, dealt to `nl` lanes (`lane` of them)
__device__ __forceinline__ void mmx(int lane, int nl, int nr, int nc, int nk, const double* A, int ar, int ac, const double* B, int br,
                                    int bc, const double* C, int cr, int cc, double alpha, double* D, int dr, int dc) {
  if (lane < 0) return;
  const float rnc = 1.0f / (float)nc;
  for (int e = lane; e < nr * nc; e += nl) {
    int i, j;
    divmod_small(e, nc, rnc, i, j);
    double acc = 0.0;
    for (int l = 0; l < nk; ++l) acc = fma(A[i * ar + l * ac], B[l * br + j * bc], acc);
    D[i * dr + j * dc] = (C ? C[i * cr + j * cc] : 0.0) + alpha * acc;
  }
}
// y = (c ? c : 0) + alpha A x  (A: n x n strided), one output per lane
__device__ __forceinline__ void mvx(int lane, int nl, int n, const double* A, int ar, int ac, const double* x, const double* c, double alpha,
                                    double* y, int ys = 1) {
  if (lane < 0) return;
  for (int i = lane; i < n; i += nl) {
    double acc = 0.0;
    for (int l = 0; l < n; ++l) acc = fma(A[i * ar + l * ac], x[l], acc);
    y[i * ys] = (c ? c[i] : 0.0) + alpha * acc;
  }
}

// lower Cholesky factor of the positive semi-definite prior covariance (zero rows for the integral states), by thread 0
__device__ __forceinline__ void chol_psd_serial(int n, const double* A, double* L) {
  for (int j = 0; j < n; ++j) {
    for (int i = 0; i < j; ++i) L[i * n + j] = 0.0;
    double p = A[j * n + j];
    for (int k = 0; k < j; ++k) p = fma(-L[j * n + k], L[j * n + k], p);
    const bool ok = p > A[j * n + j] * 5.7e-14;
    const double r = ok ? sqrt(p) : 0.0, rr = ok ? 1.0 / r : 0.0;
    L[j * n + j] = r;
    for (int i = j + 1; i < n; ++i) {
      double a = A[i * n + j];
      for (int k = 0; k < j; ++k) a = fma(-L[i * n + k], L[j * n + k], a);
      L[i * n + j] = a * rr;
    }
  }
}

__host__ __device__ inline int sq_ldw(int n) { return (2 * n + 1) | 1; } // row stride of a stacked n x 2n matrix (odd)
// workspace of one combine / walk step: two stacked matrices, X, X', three n x (n+1) temporaries, eight vectors
__host__ __device__ inline int sq_work_doubles(int n) { return 2 * n * sq_ldw(n) + 2 * n * n + 3 * n * (n + 1) + 8 * n; }
struct SqWork {
  double *WA, *WB, *X, *Xp, *T1, *T2, *T3, *v;
  int ldw;
  __device__ __forceinline__ void carve(double* p, int n) {
    ldw = sq_ldw(n);
    WA = p; WB = WA + n * ldw; X = WB + n * ldw; Xp = X + n * n; T1 = Xp + n * n; T2 = T1 + n * (n + 1); T3 = T2 + n * (n + 1); v = T3 + n * (n + 1);
  }
};

// eo = ei (x) ej (ei earlier).  All in shared memory; eo distinct from ei, ej.
template <int NT>
__device__ void dense_combine_sqrt(const Grp<NT>& g, int n, const double* ei, const double* ej, double* eo, const SqWork& w) {
  const int n1 = n + 1, ldw = w.ldw, tid = threadIdx.x, wp = tid >> 5;
  const double *Ai = ei, *Ui = ei + n * n1, *Zi = Ui + n * n;   // Zi: row stride n1, eta_i in column n
  const double *Aj = ej, *Uj = ej + n * n1, *Zj = Uj + n * n;
  double *Ao = eo, *Uo = eo + n * n1, *Zo = Uo + n * n;
  double *t = w.v, *s1 = w.v + n, *wv = w.v + 2 * n, *u = w.v + 3 * n, *t2 = w.v + 4 * n, *t3 = w.v + 5 * n, *t4 = w.v + 6 * n, *t5 = w.v + 7 * n;
  const int rest = tid - 64, nrest = NT - 64; // the lanes of warps 2.. (negative: not one of them)
  // 1: V = U_i^T Z_j -> WA = [I | V];  s1 = Z_j^T b_i
  mmx(tid, NT, n, n, n, Ui, 1, n, Zj, n1, 1, nullptr, 0, 0, 1.0, w.WA + n, ldw, 1);
  for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WA[i * ldw + j] = (i == j) ? 1.0 : 0.0; }
  if (tid < n) {
    double b = 0.0;
    for (int l = 0; l < n; ++l) b = fma(Zj[l * n1 + tid], Ai[l * n1 + n], b);
    s1[tid] = b;
  }
  g.sync();
  // 2: WB = [I | V^T];  T1 = [A_i | b_i];  u = eta_j - Z_j s1
  for (int e = tid; e < n * n; e += NT) {
    const int i = e / n, j = e - i * n;
    w.WB[i * ldw + j] = (i == j) ? 1.0 : 0.0;
    w.WB[i * ldw + n + j] = w.WA[j * ldw + n + i];
    w.T1[i * n1 + j] = Ai[i * n1 + j];
  }
  if (tid < n) {
    double a = Ai[tid * n1 + n], b = Zj[tid * n1 + n];
    for (int l = 0; l < n; ++l) b = fma(-Zj[tid * n1 + l], s1[l], b);
    wv[tid] = a; w.T1[tid * n1 + n] = a; u[tid] = b;
  }
  g.sync();
  // 3: the two triangularisations (warps 0, 1);  the others: T2 = Z_j^T T1;  t2 = U_i^T u
  if (wp == 0) tria_warp(n, 2 * n, ldw, w.WA);
  else if (wp == 1) tria_warp(n, 2 * n, ldw, w.WB);
  else {
    mmx(rest, nrest, n, n1, n, Zj, 1, n1, w.T1, n1, 1, nullptr, 0, 0, 1.0, w.T2, n1, 1);
    mvx(rest, nrest, n, Ui, 1, n, u, nullptr, 1.0, t2);
  }
  g.sync();
  // 4: X = U_i T^-T (warp 0), X' = Z_j T'^-T (warp 1);  the others: T3 = Z_j T2;  t3 = U_i t2
  if (wp == 0) solve_rows_warp(n, w.WA, ldw, Ui, n, w.X, n);
  else if (wp == 1) solve_rows_warp(n, w.WB, ldw, Zj, n1, w.Xp, n);
  else {
    mmx(rest, nrest, n, n1, n, Zj, n1, 1, w.T2, n1, 1, nullptr, 0, 0, 1.0, w.T3, n1, 1);
    mvx(rest, nrest, n, Ui, n, 1, t2, nullptr, 1.0, t3);
  }
  g.sync();
  // 5: T2 = X^T T3;  t4 = X'^T t3;  t = X^T u;  WA = [A_j X | U_j];  WB = [A_i^T X' | Z_i]
  mmx(tid, NT, n, n1, n, w.X, 1, n, w.T3, n1, 1, nullptr, 0, 0, 1.0, w.T2, n1, 1);
  mvx(tid - 32, NT - 32, n, w.Xp, 1, n, t3, nullptr, 1.0, t4);
  mvx(tid - 64, NT - 64, n, w.X, 1, n, u, nullptr, 1.0, t);
  mmx(tid, NT, n, n, n, Aj, n1, 1, w.X, n, 1, nullptr, 0, 0, 1.0, w.WA, ldw, 1);
  mmx(tid, NT, n, n, n, Ai, 1, n1, w.Xp, n, 1, nullptr, 0, 0, 1.0, w.WB, ldw, 1);
  for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WA[i * ldw + n + j] = Uj[e]; w.WB[i * ldw + n + j] = Zi[i * n1 + j]; }
  g.sync();
  // 6: U = tria(WA) (warp 0), Z = tria(WB) (warp 1);  the others: T3 = [A_i - X T2 | b_i + X t] = [M A_i | b_i + X X^T u];  t5 = u - X' t4 = M^T u
  if (wp == 0) tria_warp(n, 2 * n, ldw, w.WA);
  else if (wp == 1) tria_warp(n, 2 * n, ldw, w.WB);
  else {
    mmx(rest, nrest, n, n, n, w.X, n, 1, w.T2, n1, 1, w.T1, n1, 1, -1.0, w.T3, n1, 1);
    mvx(rest, nrest, n, w.X, n, 1, t, wv, 1.0, w.T3 + n, n1);
    mvx(rest, nrest, n, w.Xp, n, 1, t4, u, -1.0, t5);
  }
  g.sync();
  // 7: [A | b] = A_j T3 (+ b_j);  eta = A_i^T t5 + eta_i;  U, Z from the stacked buffers
  mmx(tid, NT, n, n1, n, Aj, n1, 1, w.T3, n1, 1, nullptr, 0, 0, 1.0, Ao, n1, 1);
  for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; Uo[e] = w.WA[i * ldw + j]; Zo[i * n1 + j] = w.WB[i * ldw + j]; }
  if (tid < n) {
    double a = Zi[tid * n1 + n];
    for (int l = 0; l < n; ++l) a = fma(Ai[l * n1 + tid], t5[l], a);
    Zo[tid * n1 + n] = a;
  }
  g.sync();
  if (tid < n) Ao[tid * n1 + n] += Aj[tid * n1 + n];
  g.sync();
}

__host__ __device__ inline int foldDs_group_doubles(int n) { return 3 * elem_size(n) + sq_work_doubles(n); }

template <int NT>
__global__ void __launch_bounds__(NT) k_foldD_sqrt(const __grid_constant__ DenseArgs P) {
  extern __shared__ __align__(16) char smem[];
  const int n = P.n, es = elem_size(n);
  const Grp<NT> g;
  const int64_t gid = blockIdx.x;
  if (gid >= P.batch * P.cout) return;
  double* e0 = (double*)smem; double* e1 = e0 + es; double* e2 = e1 + es;
  SqWork w;
  w.carve(e2 + es, n);
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double* src = P.Ein + (series * P.cin + m0) * (int64_t)es;
  const int first = (m0 + 1 < m1) ? 2 * es : es;
  for (int e = g.gl; e < first; e += NT) e0[e] = src[e];
  g.sync();
  double* acc = e0; double* nxt = e1; double* out = e2;
  for (int64_t m = m0 + 1; m < m1; ++m) {
    src += es;
    if (m > m0 + 1) {
      for (int e = g.gl; e < es; e += NT) nxt[e] = src[e];
      g.sync();
    }
    dense_combine_sqrt<NT>(g, n, acc, nxt, out, w);
    double* tq = acc; acc = out; out = tq; // the result becomes the accumulator
  }
  double* dst = P.Eout + gid * (int64_t)es;
  for (int e = g.gl; e < es; e += NT) dst[e] = acc[e];
}

// down-sweep in factor form.  blockIdx.y = 0: prefix states [m | S]; 1: suffix information [eta | Z].
__host__ __device__ inline int downDs_group_doubles(int n) { return elem_size(n) + 2 * state_size(n) + sq_work_doubles(n); }

template <int NT>
__global__ void __launch_bounds__(NT) k_downD_sqrt(const __grid_constant__ DenseArgs P) {
  extern __shared__ __align__(16) char smem[];
  const int n = P.n, n1 = n + 1, es = elem_size(n), ss = state_size(n);
  const Grp<NT> g;
  const int64_t gid = blockIdx.x;
  if (gid >= P.batch * P.cout) return;
  const int backward = blockIdx.y, tid = threadIdx.x, wp = tid >> 5;
  double* el = (double*)smem; double* st = el + es; double* st2 = st + ss;
  SqWork w;
  w.carve(st2 + ss, n);
  const int ldw = w.ldw;
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double *A = el, *U = el + n * n1, *Z = U + n * n; // [A | b], U, [Z | eta]
  double *t = w.v, *s1 = w.v + n, *wv = w.v + 2 * n, *s2 = w.v + 3 * n, *s3 = w.v + 4 * n, *s4 = w.v + 5 * n;
  if (!backward) {
    if (P.PREup) { const double* s = P.PREup + gid * (int64_t)ss; for (int e = tid; e < ss; e += NT) st[e] = s[e]; }
    else {
      for (int e = tid; e < n; e += NT) st[e] = 0.0;
      if (tid == 0) chol_psd_serial(n, P.p0, st + n); // S0 S0^T = blkdiag(Pinf, 0)
    }
    g.sync();
    for (int64_t m = m0; m < m1; ++m) {
      double* dst = P.PRE + (series * P.cin + m) * (int64_t)ss;
      for (int e = tid; e < ss; e += NT) dst[e] = st[e];
      if (m + 1 == m1) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = tid; e < es; e += NT) el[e] = src[e];
      g.sync();
      const double *mv = st, *S = st + n;
      // V = S^T Z -> WA = [I | V];  t = Z^T m.   The mean in its "mean + gain x innovation" form:
      // m' = A (m + X X^T (eta - J m)) + b
      mmx(tid, NT, n, n, n, S, 1, n, Z, n1, 1, nullptr, 0, 0, 1.0, w.WA + n, ldw, 1);
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WA[i * ldw + j] = (i == j) ? 1.0 : 0.0; }
      if (tid < n) { double a = 0.0; for (int l = 0; l < n; ++l) a = fma(Z[l * n1 + tid], mv[l], a); t[tid] = a; }
      g.sync();
      if (wp == 0) tria_warp(n, 2 * n, ldw, w.WA);
      else if (tid - 32 < n) { const int i = tid - 32; double a = Z[i * n1 + n]; for (int l = 0; l < n; ++l) a = fma(-Z[i * n1 + l], t[l], a); wv[i] = a; } // u = eta - Z t
      g.sync();
      if (wp == 0) solve_rows_warp(n, w.WA, ldw, S, n, w.X, n);                                                                              // X = S T^-T
      g.sync();
      mmx(tid, NT, n, n, n, A, n1, 1, w.X, n, 1, nullptr, 0, 0, 1.0, w.WA, ldw, 1);                                                         // WA = [A X | U]
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WA[i * ldw + n + j] = U[e]; }
      mvx(tid, NT, n, w.X, 1, n, wv, nullptr, 1.0, s3);                                                                                       // s3 = X^T u
      g.sync();
      if (wp == 0) tria_warp(n, 2 * n, ldw, w.WA);
      else mvx(tid - 32, NT - 32, n, w.X, n, 1, s3, mv, 1.0, s4);                                                                             // s4 = m + X s3
      g.sync();
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; st2[n + e] = w.WA[i * ldw + j]; }
      if (tid < n) { double a = A[tid * n1 + n]; for (int l = 0; l < n; ++l) a = fma(A[tid * n1 + l], s4[l], a); st2[tid] = a; }
      g.sync();
      double* tq = st; st = st2; st2 = tq;
    }
  } else {
    if (!P.want_suffix) return;
    if (P.SUFup) { const double* s = P.SUFup + gid * (int64_t)ss; for (int e = tid; e < ss; e += NT) st[e] = s[e]; }
    else { for (int e = tid; e < ss; e += NT) st[e] = 0.0; }
    g.sync();
    for (int64_t m = m1 - 1; m >= m0; --m) {
      double* dst = P.SUF + (series * P.cin + m) * (int64_t)ss;
      for (int e = tid; e < ss; e += NT) dst[e] = st[e];
      if (m == m0) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = tid; e < es; e += NT) el[e] = src[e];
      g.sync();
      const double *ev = st, *Zs = st + n; // suffix information [eta_s | Z_s], Z_s row stride n
      // V^T = Z_s^T U -> WB = [I | V^T];  s1 = Z_s^T b
      mmx(tid, NT, n, n, n, Zs, 1, n, U, n, 1, nullptr, 0, 0, 1.0, w.WB + n, ldw, 1);
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WB[i * ldw + j] = (i == j) ? 1.0 : 0.0; }
      if (tid < n) { double a = 0.0; for (int l = 0; l < n; ++l) a = fma(Zs[l * n + tid], A[l * n1 + n], a); s1[tid] = a; }
      g.sync();
      if (wp == 0) tria_warp(n, 2 * n, ldw, w.WB);
      else if (tid - 32 < n) { const int i = tid - 32; double a = ev[i]; for (int l = 0; l < n; ++l) a = fma(-Zs[i * n + l], s1[l], a); wv[i] = a; } // u = eta_s - Z_s s1
      g.sync();
      if (wp == 0) solve_rows_warp(n, w.WB, ldw, Zs, n, w.Xp, n);                                                                             // X' = Z_s T'^-T
      else if (tid - 32 < n) { const int i = tid - 32; double a = 0.0; for (int l = 0; l < n; ++l) a = fma(U[l * n + i], wv[l], a); t[i] = a; }   // t = U^T u
      g.sync();
      mmx(tid, NT, n, n, n, A, 1, n1, w.Xp, n, 1, nullptr, 0, 0, 1.0, w.WB, ldw, 1);                                                         // WB = [A^T X' | Z]
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; w.WB[i * ldw + n + j] = Z[i * n1 + j]; }
      mvx(tid, NT, n, U, n, 1, t, nullptr, 1.0, s2);                                                                                          // s2 = U t
      g.sync();
      if (wp == 0) tria_warp(n, 2 * n, ldw, w.WB);
      else mvx(tid - 32, NT - 32, n, w.Xp, 1, n, s2, nullptr, 1.0, s3);                                                                       // s3 = X'^T s2
      g.sync();
      mvx(tid, NT, n, w.Xp, n, 1, s3, wv, -1.0, s4);                                                                                          // s4 = M^T u
      g.sync();
      for (int e = tid; e < n * n; e += NT) { const int i = e / n, j = e - i * n; st2[n + e] = w.WB[i * ldw + j]; }
      if (tid < n) { double a = Z[tid * n1 + n]; for (int l = 0; l < n; ++l) a = fma(A[l * n1 + tid], s4[l], a); st2[tid] = a; }
      g.sync();
      double* tq = st; st = st2; st2 = tq;
    }
  }
}
