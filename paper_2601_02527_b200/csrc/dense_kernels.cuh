// dense_kernels.cuh -- the dense levels of the scan: combine of chunk aggregates (k_foldD) and the
// down-sweep of prefix states / suffix information (k_downD).  One CTA of NT threads per group of
// elements; all matrices n x n in shared memory.  Device-safe text on top of dev_consts.h and
// grp_dev.cuh: compiled statically with a run-time n and, specialised, with n as a constant (jit.cu).
#pragma once
#include "chunk_kernels.cuh"

#ifdef SG_JIT
#define DN JT_N
#else
#define DN (P.n)
#endif

// Which dot products are accumulated with the compensated Dot2 scheme (grp_dev.cuh): class A = the products
// that form the matrix of a solve, I + (covariance)(information), and its right-hand sides -- their terms cancel
// by orders of magnitude; class B = every other product of a combine (sums of like-signed or
// well-scaled terms).  Measured on config 3 at full size (profiles/r02_sweeps.md): compensating class A alone gives
// the same accuracy as compensating everything (variance 7.6e-10 either way; 2.8e-8 with class B alone, 5.7e-8
// with none), so class B is plain FMA.  Option "dot2" (bit 0 = A, bit 1 = B) overrides it in the specialised build.
#if defined(SG_JIT) && defined(JT_DOT2)
#define SG_DOT2_A ((JT_DOT2 & 1) != 0)
#define SG_DOT2_B ((JT_DOT2 & 2) != 0)
#else
#define SG_DOT2_A true
#define SG_DOT2_B false
#endif
template <bool COMP>
__device__ __forceinline__ void dot_step(double a, double b, double& s, double& c) {
  if constexpr (COMP) dot2_step(a, b, s, c);
  else s = fma(a, b, s);
}

// general dense product  D[i,j] = (C ? C[i,j] : 0) + sum_l A[i,l] B[l,j],  strided operands.  A thread works on
// two outputs at a time: the two compensated chains are independent, so their fixed-latency FP64 dependencies
// overlap (the dense levels are latency-bound, profiles/r01_dense_level_ncu.md).  skew: number of work items the
// group has already been dealt in this phase (the next item goes to lane skew % G), so that several products
// between two barriers load the lanes evenly.
template <bool COMP, int G>
__device__ __forceinline__ void mm(const Grp<G>& g, int nr, int nc, int nk, const double* A, int ar, int ac,
                                   const double* B, int br, int bc, const double* C, int cr, int cc, double* D, int dr, int dc,
                                   int skew = 0) {
  const float rnc = 1.0f / (float)nc;
  const int tot = nr * nc;
  int e0 = g.gl - skew % G;
  if (e0 < 0) e0 += G;
  for (int e = e0; e < tot; e += 2 * G) {
    const int eb = (e + G < tot) ? e + G : e; // no second output left: the first one is computed twice
    int i, j, ib, jb;
    divmod_small(e, nc, rnc, i, j);
    divmod_small(eb, nc, rnc, ib, jb);
    double acc = C ? C[i * cr + j * cc] : 0.0, accb = C ? C[ib * cr + jb * cc] : 0.0;
    double cmp = 0.0, cmpb = 0.0;
    for (int l = 0; l < nk; ++l) {
      dot_step<COMP>(A[i * ar + l * ac], B[l * br + j * bc], acc, cmp);
      dot_step<COMP>(A[ib * ar + l * ac], B[l * br + jb * bc], accb, cmpb);
    }
    D[i * dr + j * dc] = acc + cmp;
    if (eb != e) D[ib * dr + jb * dc] = accb + cmpb;
  }
}
// e -> (i, j), j <= i, of the e-th entry of the lower triangle in row order (e < 2^20)
__device__ __forceinline__ void tri_index(int e, int& i, int& j) {
  i = (int)((sqrtf((float)(8 * e + 1)) - 1.0f) * 0.5f);
  if (i * (i + 1) / 2 > e) --i;
  if ((i + 1) * (i + 2) / 2 <= e) ++i;
  j = e - i * (i + 1) / 2;
}
// symmetric result: D[i,j] = D[j,i] = C[i,j] + sum_l A[i,l] B[l,j] for i >= j (n x n; row strides cr, dr);
// the n (n + 1) / 2 entries of the lower triangle are the work items, two at a time as in mm
template <bool COMP, int G>
__device__ __forceinline__ void mm_sym(const Grp<G>& g, int n, int nk, const double* A, int ar, int ac,
                                       const double* B, int br, int bc, const double* C, int cr, double* D, int dr, int skew = 0) {
  const int tot = n * (n + 1) / 2;
  int e0 = g.gl - skew % G;
  if (e0 < 0) e0 += G;
  for (int e = e0; e < tot; e += 2 * G) {
    const int eb = (e + G < tot) ? e + G : e;
    int i, j, ib, jb;
    tri_index(e, i, j);
    tri_index(eb, ib, jb);
    double acc = C[i * cr + j], accb = C[ib * cr + jb];
    double cmp = 0.0, cmpb = 0.0;
    for (int l = 0; l < nk; ++l) {
      dot_step<COMP>(A[i * ar + l * ac], B[l * br + j * bc], acc, cmp);
      dot_step<COMP>(A[ib * ar + l * ac], B[l * br + jb * bc], accb, cmpb);
    }
    acc += cmp;
    D[i * dr + j] = acc;
    D[j * dr + i] = acc;
    if (eb != e) { accb += cmpb; D[ib * dr + jb] = accb; D[jb * dr + ib] = accb; }
  }
}

// ---------------------------------------------------------------------------------------------------
// dense combine (SG21 Eq. 11 as cited P:502; the paper prints neither): with
// M = (I + C_i J_j)^-1,
//   A = A_j M A_i,  b = A_j M (b_i + C_i eta_j) + b_j,  C = A_j M C_i A_j^T + C_j,
//   eta = A_i^T M^T (eta_j - J_j b_i) + eta_i,           J = A_i^T M^T J_j A_i + J_i.
// One CTA per group.  ei, ej, eo: elements in shared memory (layout above); Ws: n x (3n+1); Tm: n x (n+1);
// Xs: n x (2n+1), receives M^-1 [A_i | b_i + C_i eta_j | C_i].
// ---------------------------------------------------------------------------------------------------
template <int G>
__device__ void dense_combine(const Grp<G>& g, int n, const double* ei, const double* ej, double* eo,
                              double* Ws, double* Tm, double* uv, double* Xs, double* T2) {
  const int n1 = n + 1, ld = (3 * n + 1) | 1, lx = 2 * n + 1, ntri = n * (n + 1) / 2; // ld: odd row stride of Ws
  const double *Ai = ei, *Ci = ei + n * n1, *Ji = Ci + n * n;
  const double *Aj = ej, *Cj = ej + n * n1, *Jj = Cj + n * n;
  double *Ao = eo, *Co = eo + n * n1, *Jo = Co + n * n;
#ifdef SG_DENSE_CLK
  long long ck[8]; int ci = 0;
#define SG_CK() do { ck[ci++] = clock64(); } while (0)
#else
#define SG_CK() do {} while (0)
#endif
  SG_CK();
  // phase 1 (everything that needs no solve): Tm = C_i [J_j | eta_j] (n x (n+1)); T2 = J_j A_i; u = eta_j - J_j b_i
  mm<SG_DOT2_A>(g, n, n1, n, Ci, n, 1, Jj, n1, 1, (const double*)nullptr, 0, 0, Tm, n1, 1);
  mm<SG_DOT2_B>(g, n, n, n, Jj, n1, 1, Ai, n1, 1, (const double*)nullptr, 0, 0, T2, n, 1, n * n1);
  for (int i = G - 1 - g.gl; i < n; i += G) { // dealt from the last lane down: those have the fewest items above
    double acc = Jj[i * n1 + n];
    { double cmp = 0.0; for (int l = 0; l < n; ++l) dot_step<SG_DOT2_B>(-Jj[i * n1 + l], Ai[l * n1 + n], acc, cmp); acc += cmp; }
    uv[i] = acc;
  }
  g.sync();
  SG_CK();
  // Ws = [I + C_i J_j | A_i | b_i + C_i eta_j | C_i]
  for (int e = g.gl; e < n * n; e += G) {
    const int i = e / n, j = e - i * n;
    Ws[i * ld + j] = Tm[i * n1 + j] + (i == j ? 1.0 : 0.0);
    Ws[i * ld + n + j] = Ai[i * n1 + j];
    Ws[i * ld + 2 * n + 1 + j] = Ci[i * n + j];
  }
  for (int i = g.gl; i < n; i += G) Ws[i * ld + 2 * n] = Ai[i * n1 + n] + Tm[i * n1 + n];
  g.sync();
  SG_CK();
  gj_solve_wcol<G, SG_GJ_WCPT>(g, n, 3 * n + 1, ld, Ws, Xs);
  SG_CK();
  const double* X1 = Xs;             // M A_i           (row stride lx)
  const double* X2 = Xs + n;         // M (b_i + C_i eta_j), then X3 = M C_i follows
  // phase 2: [A | b] = A_j [X1 | x2] (b_j is added in phase 3); Tm = A_j X3
  mm<SG_DOT2_B>(g, n, n1, n, Aj, n1, 1, X1, lx, 1, (const double*)nullptr, 0, 0, Ao, n1, 1);
  mm<SG_DOT2_B>(g, n, n, n, Aj, n1, 1, X2 + 1, lx, 1, (const double*)nullptr, 0, 0, Tm, n, 1, n * n1);
  g.sync();
  SG_CK();
  // phase 3: C = Tm A_j^T + C_j;  J = X1^T T2 + J_i;  eta = X1^T u + eta_i;  b += b_j
  mm_sym<SG_DOT2_B>(g, n, n, Tm, n, 1, Aj, 1, n1, Cj, n, Co, n);
  mm_sym<SG_DOT2_B>(g, n, n, X1, 1, lx, T2, n, 1, Ji, n1, Jo, n1, ntri);
  for (int i = G - 1 - g.gl; i < n; i += G) {
    double acc = Ji[i * n1 + n];
    { double cmp = 0.0; for (int l = 0; l < n; ++l) dot_step<SG_DOT2_B>(X1[l * lx + i], uv[l], acc, cmp); acc += cmp; }
    Jo[i * n1 + n] = acc;
    Ao[i * n1 + n] += Aj[i * n1 + n];
  }
  g.sync();
  SG_CK();
#ifdef SG_DENSE_CLK
  if (threadIdx.x == 0 && blockIdx.x == 0) printf("combine cycles: phase1 %lld assemble %lld gj %lld phase2 %lld phase3 %lld\n", ck[1] - ck[0], ck[2] - ck[1], ck[3] - ck[2], ck[4] - ck[3], ck[5] - ck[4]);
#endif
}

__host__ __device__ inline int foldD_group_doubles(int n) { return 3 * elem_size(n) + n * (3 * n + 2) + n * (n + 1) + n + n * (2 * n + 1) + n * n; }

struct DenseArgs {
  int n;              // augmented state dimension
  const double* p0;   // [n][n] prior covariance
  const double* Ein;  // [batch*cin][elem]
  double* Eout;       // [batch*cout][elem]
  int64_t cin, cout, batch;
  int g;              // fan-in
  // down-sweep
  const double* PREup; // [batch*cout][state] or NULL -> prior
  const double* SUFup; // [batch*cout][state] or NULL -> zero
  double* PRE;         // [batch*cin][state]
  double* SUF;         // [batch*cin][state]
  int want_suffix;
};

template <int NT>
__device__ __forceinline__ void foldD_body(const DenseArgs& P) {
  extern __shared__ __align__(16) char smem[];
  const int n = DN, es = elem_size(n);
  const size_t tb = 0;
  const Grp<NT> g;
  const int64_t gid = blockIdx.x;
  if (gid >= P.batch * P.cout) return;
  double* base = (double*)(smem + tb);
  double* e0 = base; double* e1 = e0 + es; double* e2 = e1 + es;
  double* Ws = e2 + es; double* Tm = Ws + n * (3 * n + 2); double* uv = Tm + n * (n + 1); double* Xs = uv + n; double* T2 = Xs + n * (2 * n + 1);
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double* src = P.Ein + (series * P.cin + m0) * (int64_t)es;
  // the first two elements of the group are consecutive in memory (e0, e1 too): one pass of loads for both
  const int first = (m0 + 1 < m1) ? 2 * es : es;
#ifdef SG_DENSE_CLK
  const long long c_ld0 = clock64();
#endif
  for (int e = g.gl; e < first; e += NT) e0[e] = src[e];
  g.sync();
#ifdef SG_DENSE_CLK
  if (threadIdx.x == 0 && blockIdx.x == 0) printf("foldD load cycles %lld (grid %d)\n", clock64() - c_ld0, gridDim.x);
#endif
  double* acc = e0; double* nxt = e1; double* out = e2;
  for (int64_t m = m0 + 1; m < m1; ++m) {
    src += es;
    if (m > m0 + 1) {
      for (int e = g.gl; e < es; e += NT) nxt[e] = src[e];
      g.sync();
    }
    dense_combine(g, n, acc, nxt, out, Ws, Tm, uv, Xs, T2);
    double* t = acc; acc = out; out = t;
  }
  double* dst = P.Eout + gid * (int64_t)es;
  for (int e = g.gl; e < es; e += NT) dst[e] = acc[e];
}

// ---------------------------------------------------------------------------------------------------
// down-sweep over dense elements.  blockIdx.y = 0: prefix states; 1: suffix information.
//   forward : (m,P) (x) element:  M = (I + P J)^-1;  m' = A M (m + P eta) + b;  P' = A M P A^T + C
//   backward: element (x) (eta_e, J_e):  M = (I + C J_e)^-1;  eta' = A^T M^T (eta_e - J_e b) + eta;
//             J' = A^T M^T J_e A + J
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int downD_group_doubles(int n) { return elem_size(n) + 2 * state_size(n) + n * (2 * n + 1) + n * n + n + n * (n + 1); }

template <int NT>
__device__ __forceinline__ void downD_body(const DenseArgs& P) {
  extern __shared__ __align__(16) char smem[];
  const int n = DN, n1 = n + 1, es = elem_size(n), ss = state_size(n), ld = 2 * n + 1;
  const size_t tb = 0;
  const Grp<NT> g;
  const int64_t gid = blockIdx.x;
  if (gid >= P.batch * P.cout) return;
  const int backward = blockIdx.y;
  double* base = (double*)(smem + tb);
  double* el = base; double* st = el + es; double* st2 = st + ss; double* Ws = st2 + ss; double* Tm = Ws + n * ld; double* uv = Tm + n * n; double* Xs = uv + n;
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double *A = el, *C = el + n * n1, *J = C + n * n; // [A|b], C, [J|eta]
  if (!backward) {
    // st = [m | P]
    if (P.PREup) { const double* s = P.PREup + gid * (int64_t)ss; for (int e = g.gl; e < ss; e += NT) st[e] = s[e]; }
    else { for (int e = g.gl; e < n; e += NT) st[e] = 0.0; for (int e = g.gl; e < n * n; e += NT) st[n + e] = P.p0[e]; }
    g.sync();
    for (int64_t m = m0; m < m1; ++m) {
      double* dst = P.PRE + (series * P.cin + m) * (int64_t)ss;
      for (int e = g.gl; e < ss; e += NT) dst[e] = st[e];
      if (m + 1 == m1) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = g.gl; e < es; e += NT) el[e] = src[e];
      g.sync();
      const double *mv = st, *Pm = st + n;
      // Ws = [I + P J | m + P eta | P]
      mm<SG_DOT2_A>(g, n, n1, n, Pm, n, 1, J, n1, 1, (const double*)nullptr, 0, 0, Ws, ld, 1); // cols 0..n: P [J | eta]
      g.sync();
      for (int e = g.gl; e < n * n; e += NT) { const int i = e / n, j = e - i * n; Ws[i * ld + n1 + j] = Pm[e]; }
      for (int i = g.gl; i < n; i += NT) { Ws[i * ld + i] += 1.0; Ws[i * ld + n] += mv[i]; }
      g.sync();
      gj_solve_wcol<NT, SG_GJ_WCPT>(g, n, ld, ld, Ws, Xs); // Xs = M^-1 [m + P eta | P], row stride n + 1
      // m' = A x + b ; Tm = A X ; P' = Tm A^T + C
      for (int i = g.gl; i < n; i += NT) {
        double acc = A[i * n1 + n];
        { double cmp = 0.0; for (int l = 0; l < n; ++l) dot_step<SG_DOT2_B>(A[i * n1 + l], Xs[l * n1], acc, cmp); acc += cmp; }
        st2[i] = acc;
      }
      mm<SG_DOT2_B>(g, n, n, n, A, n1, 1, Xs + 1, n1, 1, (const double*)nullptr, 0, 0, Tm, n, 1);
      g.sync();
      mm_sym<SG_DOT2_B>(g, n, n, Tm, n, 1, A, 1, n1, C, n, st2 + n, n);
      g.sync();
      double* t = st; st = st2; st2 = t;
    }
  } else {
    if (!P.want_suffix) return;
    // st = [eta | J]
    if (P.SUFup) { const double* s = P.SUFup + gid * (int64_t)ss; for (int e = g.gl; e < ss; e += NT) st[e] = s[e]; }
    else { for (int e = g.gl; e < ss; e += NT) st[e] = 0.0; }
    g.sync();
    for (int64_t m = m1 - 1; m >= m0; --m) {
      double* dst = P.SUF + (series * P.cin + m) * (int64_t)ss;
      for (int e = g.gl; e < ss; e += NT) dst[e] = st[e];
      if (m == m0) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = g.gl; e < es; e += NT) el[e] = src[e];
      g.sync();
      const double *ev = st, *Je = st + n;
      const int ld2 = 2 * n + 1; // odd row stride, 2n columns in use
      // Ws = [I + C J_e | A]
      mm<SG_DOT2_A>(g, n, n, n, C, n, 1, Je, n, 1, (const double*)nullptr, 0, 0, Ws, ld2, 1);
      g.sync();
      for (int e = g.gl; e < n * n; e += NT) { const int i = e / n, j = e - i * n; Ws[i * ld2 + n + j] = A[i * n1 + j]; }
      for (int i = g.gl; i < n; i += NT) Ws[i * ld2 + i] += 1.0;
      // u = eta_e - J_e b
      for (int i = g.gl; i < n; i += NT) {
        double acc = ev[i];
        { double cmp = 0.0; for (int l = 0; l < n; ++l) dot_step<SG_DOT2_B>(-Je[i * n + l], A[l * n1 + n], acc, cmp); acc += cmp; }
        uv[i] = acc;
      }
      g.sync();
      gj_solve_wcol<NT, SG_GJ_WCPT>(g, n, 2 * n, ld2, Ws, Xs);
      const double* X = Xs; // M A, row stride n
      for (int i = g.gl; i < n; i += NT) {
        double acc = J[i * n1 + n];
        { double cmp = 0.0; for (int l = 0; l < n; ++l) dot_step<SG_DOT2_B>(X[l * n + i], uv[l], acc, cmp); acc += cmp; }
        st2[i] = acc;
      }
      mm<SG_DOT2_B>(g, n, n, n, Je, n, 1, A, n1, 1, (const double*)nullptr, 0, 0, Tm, n, 1); // Tm = J_e A
      g.sync();
      mm_sym<SG_DOT2_B>(g, n, n, X, 1, n, Tm, n, 1, J, n1, st2 + n, n); // J' = X^T (J_e A) + J
      g.sync();
      double* t = st; st = st2; st2 = t;
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// k_adjD: the adjoint of the forward filter at each chunk's last event from the reverse scan's suffix
// information (eta, J) about the state after the chunk and the state (m, P) there (= the prefix state of the
// next chunk):  Lambda^ = (I + J P)^-1 J,  lambda^ = (I + J P)^-1 (J m - eta)   (I + J P has eigenvalues >= 1).
// It starts the adjoint recursion of the register-resident k_down0, which therefore carries no solve workspace.
// One CTA per chunk; the last chunk of a series has no later data: zero.  J P cancels like the products of the
// dense combine: compensated (Dot2).
// ---------------------------------------------------------------------------------------------------
struct AdjArgs {
  int n;
  const double* PRE; // [batch*c1][state] prefix states [m | P]
  const double* SUF; // [batch*c1][state] suffix information [eta | J]
  double* ADJ;       // [batch*c1][state] out: [lambda^ | Lambda^]
  int64_t c1, batch;
};
__host__ __device__ inline int adjD_group_doubles(int n) { return 2 * state_size(n) + n * (2 * n + 2) + n * (n + 1) + n; }

template <int NT>
__device__ __forceinline__ void adjD_body(const AdjArgs& P) {
  extern __shared__ __align__(16) char smem[];
#ifdef SG_JIT
  const int n = JT_N;
#else
  const int n = P.n;
#endif
  const int n1 = n + 1, ss = state_size(n), ld = 2 * n + 1;
  const Grp<NT> g;
  const int64_t gid = blockIdx.x;
  if (gid >= P.batch * P.c1) return;
  const int64_t m = gid % P.c1;
  double* out = P.ADJ + gid * (int64_t)ss;
  if (m == P.c1 - 1) {
    for (int e = g.gl; e < ss; e += NT) out[e] = 0.0;
    return;
  }
  double* sJ = (double*)smem; double* sP = sJ + ss; double* Ws = sP + ss; double* Xs = Ws + n * (2 * n + 2); double* uv = Xs + n * n1;
  const double* pj = P.SUF + gid * (int64_t)ss;
  const double* pp = P.PRE + (gid + 1) * (int64_t)ss;
  for (int e = g.gl; e < ss; e += NT) { sJ[e] = pj[e]; sP[e] = pp[e]; }
  g.sync();
  const double *eta = sJ, *J = sJ + n, *mv = sP, *Pm = sP + n;
  mm<SG_DOT2_A>(g, n, n, n, J, n, 1, Pm, n, 1, (const double*)nullptr, 0, 0, Ws, ld, 1); // J P
  for (int i = NT - 1 - g.gl; i < n; i += NT) {
    double acc = -eta[i], cmp = 0.0;
    for (int l = 0; l < n; ++l) dot_step<SG_DOT2_A>(J[i * n + l], mv[l], acc, cmp);
    uv[i] = acc + cmp;
  }
  g.sync();
  for (int e = g.gl; e < n * n; e += NT) { const int i = e / n, j = e - i * n; Ws[i * ld + n + j] = J[e]; }
  for (int i = g.gl; i < n; i += NT) { Ws[i * ld + i] += 1.0; Ws[i * ld + 2 * n] = uv[i]; }
  g.sync();
  gj_solve_wcol<NT, SG_GJ_WCPT>(g, n, 2 * n + 1, ld, Ws, Xs); // Xs = [Lambda^ | lambda^], row stride n + 1
  for (int e = g.gl; e < n * n; e += NT) { const int i = e / n, j = e - i * n; out[n + e] = 0.5 * (Xs[i * n1 + j] + Xs[j * n1 + i]); }
  for (int i = g.gl; i < n; i += NT) out[i] = Xs[i * n1 + n];
}


#ifdef SG_JIT
extern "C" __global__ void __launch_bounds__(SG_DENSE_NT) jit_adjD(const __grid_constant__ AdjArgs P) { adjD_body<SG_DENSE_NT>(P); }
extern "C" __global__ void __launch_bounds__(SG_DENSE_NT) jit_foldD(const __grid_constant__ DenseArgs P) { foldD_body<SG_DENSE_NT>(P); }
extern "C" __global__ void __launch_bounds__(SG_DENSE_NT) jit_downD(const __grid_constant__ DenseArgs P) { downD_body<SG_DENSE_NT>(P); }
#else
template <int NT>
__global__ void __launch_bounds__(NT) k_foldD(const __grid_constant__ DenseArgs P) { foldD_body<NT>(P); }
template <int NT>
__global__ void __launch_bounds__(NT) k_downD(const __grid_constant__ DenseArgs P) { downD_body<NT>(P); }
#endif
