// scan.cu -- steps a3-a6: filter scan elements and their associative combine, the two-filter
// smoother, the log-likelihood reduction and the projection onto the observations.
//
// Scan layout: the K events of a series are cut into chunks of Lc events.
//   up-sweep   k_fold0 : one group of lanes per chunk folds the chunk's primitive elements
//                        (Eq. 3.20/3.21; SG21 Eq. 10) into ONE element (A,b,C,eta,J).
//                        Folding a primitive element onto an aggregate is the associative combine
//                        with a rank-one J_j and a block-structured A_j: O(n^2 bs), not O(n^3).
//              k_foldD : dense combine of g consecutive elements, level by level.
//   down-sweep k_downD : from the top, the state (m,P) before every element (prefix) and the
//                        backward information (eta,J) after it (suffix of the SAME elements).
//              k_down0 : per chunk, the plain integrated Kalman filter (Eq. 3.14-3.15, 2.22) from
//                        the chunk's prefix state -> innovations -> log-likelihood terms (Eq. 2.26);
//                        then the backward information recursion from the chunk's suffix and the
//                        smoothed exposure average at each end event (two-filter form; reading R7).
// With one chunk per series (Lc >= K) only k_down0 runs: the sequential per-series filter (row a8).
#include <math.h>

#include "scan_dev.cuh"

#define NUMF_BAD 1

// element layout in global memory: AB [n x (n+1)] = [A | b],  C [n x n],  JE [n x (n+1)] = [J | eta]
__host__ __device__ inline int elem_size(int n) { return 3 * n * n + 2 * n; }
__host__ __device__ inline int state_size(int n) { return n * n + n; } // [vector | matrix]

struct ScanDev {
  const ModelDev* M;
  const double* disc;
  const double* dt;
  const double* delta;
  const uint32_t* meta;
  const int32_t* obs;
  const double* y;
  const double* sigma;
  const double* amp;
  int64_t K, N, batch;
  int Lc;          // events per chunk
  int64_t c1;      // chunks per series
  double* E1;      // [batch*c1][elem]
  const double* PRE1; // [batch*c1][state] or NULL (prior)
  const double* SUF1; // [batch*c1][state] or NULL (zero)
  double* xbuf;    // [batch*N][state] filtered state at each end event
  double* fstate;  // [batch*K][state] post-event filtered state of every event, or NULL (a7)
  double* binfo;   // [batch*K][state] information [eta | J] about the pre-update state of every event, or NULL (a7)
  double* llpart;  // [batch*c1]
  double* mean;
  double* var;
  int* flags;
  int want_smooth;
};

template <int G>
__device__ __forceinline__ void zero_fill(const Grp<G>& g, double* p, int cnt) {
  for (int e = g.gl; e < cnt; e += G) p[e] = 0.0;
}

// ---------------------------------------------------------------------------------------------------
// k_fold0: chunk -> element
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int fold0_group_doubles(int n) { return 7 * n * n + 5 * n + 2; }

template <int G>
__global__ void __launch_bounds__(128) k_fold0(ScanDev P) {
  extern __shared__ __align__(16) char smem[];
  Tables T;
  tables_build(P.M, smem, T);
  __syncthreads();
  const int n = T.n, d = T.d, n1 = n + 1;
  const size_t tb = tables_bytes(n, d, T.ninst, T.nblk, T.nent);
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * fold0_group_doubles(n);
  double* Fs = base;            // n*n
  double* Qs = Fs + n * n;      // n*n
  double* AB0 = Qs + n * n;     // n*(n+1)
  double* AB1 = AB0 + n * n1;   // n*(n+1)
  double* C = AB1 + n * n1;     // n*n
  double* Tm = C + n * n;       // n*n
  double* JE = Tm + n * n;      // n*(n+1)
  double* av = JE + n * n1;     // n+1
  double* cv = av + n1;         // n
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ramp = P.amp ? 1.0 / P.amp[series] : 1.0;

  zero_fill(g, Fs, 2 * n * n);
  zero_fill(g, AB0, n * n1);
  zero_fill(g, C, n * n);
  zero_fill(g, JE, n * n1);
  g.sync();
  for (int i = g.gl; i < n; i += G) AB0[i * n1 + i] = 1.0;
  g.sync();

  for (int64_t k = k0; k < k1; ++k) {
    const uint32_t meta = P.meta[k];
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    assemble_step(g, T, P.disc + k * (int64_t)T.stride, tz, Fs, Qs);
    g.sync();
    lmul_F(g, T, Fs, AB0, n1, 1, AB1, n1, 1, n1); // [A | b] <- F [A | b]
    lmul_F(g, T, Fs, C, n, 1, Tm, n, 1, n);       // T = F C
    g.sync();
    rmul_Ft_sym(g, T, Fs, Tm, Qs, C);             // C <- F C F^T + Q
    g.sync();
    { double* t = AB0; AB0 = AB1; AB1 = t; }
    if (!kind) {
      // observe z_q / delta: h = hs e_z in equilibrated units (Eq. 3.12); SG21 Eq. 10 with
      // the aggregate as the earlier element (rank-one J_j): Sherman-Morrison form of the combine
      const int zi = d + q;
      const int32_t ob = P.obs[k];
      const double hs = T.tau[q] / P.delta[k];
      const double sg = P.sigma[ob] * ramp;
      const double yy = P.y[series * P.N + ob] * ramp;
      const double S = hs * hs * C[zi * n + zi] + sg * sg;
      if (!(S > 0.0) || !isfinite(S)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      for (int j = g.gl; j <= n; j += G) av[j] = hs * AB0[zi * n1 + j];
      for (int i = g.gl; i < n; i += G) cv[i] = hs * C[i * n + zi];
      g.sync();
      const double resid = yy - av[n];
      const float rn1 = 1.0f / (float)n1;
      for (int e = g.gl; e < n * n1; e += G) {
        int i, j;
        divmod_small(e, n1, rn1, i, j);
        const double aj = (j < n) ? av[j] : -resid; // last column: eta += a resid / S;  b += K resid
        JE[e] = fma(av[i] * rS, (j < n) ? aj : resid, JE[e]);
        AB0[e] = fma(-cv[i] * rS, aj, AB0[e]);
      }
      for (int e = g.gl; e < T.ntri; e += G) {
        const int i = T.tri_i[e], j = T.tri_j[e];
        const double v = fma(-cv[i] * rS, cv[j], C[i * n + j]);
        C[i * n + j] = v;
        C[j * n + i] = v;
      }
      g.sync();
      // the instrument is idle after its end: zero z_q (reading R6)
      for (int j = g.gl; j <= n; j += G) AB0[zi * n1 + j] = 0.0;
      for (int j = g.gl; j < n; j += G) { C[zi * n + j] = 0.0; C[j * n + zi] = 0.0; }
      g.sync();
    }
  }
  double* out = P.E1 + gid * (int64_t)elem_size(n);
  for (int e = g.gl; e < n * n1; e += G) { out[e] = AB0[e]; out[n * n1 + n * n + e] = JE[e]; }
  for (int e = g.gl; e < n * n; e += G) out[n * n1 + e] = C[e];
}

// ---------------------------------------------------------------------------------------------------
// dense combine (SG21 Eq. 11 as cited P:502; the paper prints neither): with
// M = (I + C_i J_j)^-1,
//   A = A_j M A_i,  b = A_j M (b_i + C_i eta_j) + b_j,  C = A_j M C_i A_j^T + C_j,
//   eta = A_i^T M^T (eta_j - J_j b_i) + eta_i,           J = A_i^T M^T J_j A_i + J_i.
// One warp per group.  ei, ej, eo: elements in shared memory (layout above); Ws: n x (3n+1); Tm: n x n.
// ---------------------------------------------------------------------------------------------------
typedef Grp<32> G32;

__device__ void dense_combine(const G32& g, const Tables& T, const double* ei, const double* ej, double* eo,
                              double* Ws, double* Tm, double* uv) {
  const int n = T.n, n1 = n + 1, ld = 3 * n + 1;
  const double *Ai = ei, *Ci = ei + n * n1, *Ji = Ci + n * n;
  const double *Aj = ej, *Cj = ej + n * n1, *Jj = Cj + n * n;
  double *Ao = eo, *Co = eo + n * n1, *Jo = Co + n * n;
  // Ws = [I + C_i J_j | A_i | b_i + C_i eta_j | C_i]
  mm(g, n, n1, n, Ci, n, 1, Jj, n1, 1, (const double*)nullptr, 0, 0, Tm, n1, 1); // n x (n+1): C_i [J_j | eta_j]  (Tm has room: see caller)
  g.sync();
  for (int e = g.gl; e < n * n; e += 32) {
    const int i = e / n, j = e - i * n;
    Ws[i * ld + j] = Tm[i * n1 + j] + (i == j ? 1.0 : 0.0);
    Ws[i * ld + n + j] = Ai[i * n1 + j];
    Ws[i * ld + 2 * n + 1 + j] = Ci[i * n + j];
  }
  for (int i = g.gl; i < n; i += 32) Ws[i * ld + 2 * n] = Ai[i * n1 + n] + Tm[i * n1 + n];
  // u = eta_j - J_j b_i
  for (int i = g.gl; i < n; i += 32) {
    double acc = Jj[i * n1 + n];
    for (int l = 0; l < n; ++l) acc = fma(-Jj[i * n1 + l], Ai[l * n1 + n], acc);
    uv[i] = acc;
  }
  g.sync();
  gj_solve(g, n, ld, Ws);
  const double* X1 = Ws + n;         // M A_i           (row stride ld)
  const double* X2 = Ws + 2 * n;     // M (b_i + C_i eta_j), then X3 = M C_i follows
  // [A | b] = A_j [X1 | x2] (+ b_j in the last column)
  mm(g, n, n1, n, Aj, n1, 1, X1, ld, 1, (const double*)nullptr, 0, 0, Ao, n1, 1);
  // Tm = A_j X3
  mm(g, n, n, n, Aj, n1, 1, X2 + 1, ld, 1, (const double*)nullptr, 0, 0, Tm, n, 1);
  g.sync();
  for (int i = g.gl; i < n; i += 32) Ao[i * n1 + n] += Aj[i * n1 + n];
  // C = Tm A_j^T + C_j
  mm_sym(g, T, n, Tm, n, 1, Aj, 1, n1, Cj, Co);
  // eta = X1^T u + eta_i
  for (int i = g.gl; i < n; i += 32) {
    double acc = Ji[i * n1 + n];
    for (int l = 0; l < n; ++l) acc = fma(X1[l * ld + i], uv[l], acc);
    Jo[i * n1 + n] = acc;
  }
  g.sync();
  // Tm = J_j A_i ; J = X1^T Tm + J_i
  mm(g, n, n, n, Jj, n1, 1, Ai, n1, 1, (const double*)nullptr, 0, 0, Tm, n, 1);
  g.sync();
  for (int e = g.gl; e < T.ntri; e += 32) {
    const int i = T.tri_i[e], j = T.tri_j[e];
    double acc = Ji[i * n1 + j];
    for (int l = 0; l < n; ++l) acc = fma(X1[l * ld + i], Tm[l * n + j], acc);
    Jo[i * n1 + j] = acc;
    Jo[j * n1 + i] = acc;
  }
  g.sync();
}

__host__ __device__ inline int foldD_group_doubles(int n) { return 3 * elem_size(n) + n * (3 * n + 1) + n * (n + 1) + n; }

struct DenseArgs {
  const ModelDev* M;
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

__global__ void __launch_bounds__(64) k_foldD(DenseArgs P) {
  extern __shared__ __align__(16) char smem[];
  Tables T;
  tables_build(P.M, smem, T);
  __syncthreads();
  const int n = T.n, es = elem_size(n);
  const size_t tb = tables_bytes(n, T.d, T.ninst, T.nblk, T.nent);
  const G32 g;
  const int gpc = blockDim.x / 32;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / 32;
  if (gid >= P.batch * P.cout) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / 32) * foldD_group_doubles(n);
  double* e0 = base; double* e1 = e0 + es; double* e2 = e1 + es;
  double* Ws = e2 + es; double* Tm = Ws + n * (3 * n + 1); double* uv = Tm + n * (n + 1);
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double* src = P.Ein + (series * P.cin + m0) * (int64_t)es;
  for (int e = g.gl; e < es; e += 32) e0[e] = src[e];
  g.sync();
  double* acc = e0; double* nxt = e1; double* out = e2;
  for (int64_t m = m0 + 1; m < m1; ++m) {
    src += es;
    for (int e = g.gl; e < es; e += 32) nxt[e] = src[e];
    g.sync();
    dense_combine(g, T, acc, nxt, out, Ws, Tm, uv);
    double* t = acc; acc = out; out = t;
  }
  double* dst = P.Eout + gid * (int64_t)es;
  for (int e = g.gl; e < es; e += 32) dst[e] = acc[e];
}

// ---------------------------------------------------------------------------------------------------
// down-sweep over dense elements.  blockIdx.y = 0: prefix states; 1: suffix information.
//   forward : (m,P) (x) element:  M = (I + P J)^-1;  m' = A M (m + P eta) + b;  P' = A M P A^T + C
//   backward: element (x) (eta_e, J_e):  M = (I + C J_e)^-1;  eta' = A^T M^T (eta_e - J_e b) + eta;
//             J' = A^T M^T J_e A + J
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int downD_group_doubles(int n) { return elem_size(n) + 2 * state_size(n) + n * (2 * n + 1) + n * n + n; }

__global__ void __launch_bounds__(64) k_downD(DenseArgs P) {
  extern __shared__ __align__(16) char smem[];
  Tables T;
  tables_build(P.M, smem, T);
  __syncthreads();
  const int n = T.n, n1 = n + 1, es = elem_size(n), ss = state_size(n), ld = 2 * n + 1;
  const size_t tb = tables_bytes(n, T.d, T.ninst, T.nblk, T.nent);
  const G32 g;
  const int gpc = blockDim.x / 32;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / 32;
  if (gid >= P.batch * P.cout) return;
  const int backward = blockIdx.y;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / 32) * downD_group_doubles(n);
  double* el = base; double* st = el + es; double* st2 = st + ss; double* Ws = st2 + ss; double* Tm = Ws + n * ld; double* uv = Tm + n * n;
  const int64_t series = gid / P.cout, grp = gid - series * P.cout;
  const int64_t m0 = grp * P.g, m1 = (m0 + P.g < P.cin) ? m0 + P.g : P.cin;
  const double *A = el, *C = el + n * n1, *J = C + n * n; // [A|b], C, [J|eta]
  if (!backward) {
    // st = [m | P]
    if (P.PREup) { const double* s = P.PREup + gid * (int64_t)ss; for (int e = g.gl; e < ss; e += 32) st[e] = s[e]; }
    else { for (int e = g.gl; e < n; e += 32) st[e] = 0.0; for (int e = g.gl; e < n * n; e += 32) st[n + e] = P.M->p0[e]; }
    g.sync();
    for (int64_t m = m0; m < m1; ++m) {
      double* dst = P.PRE + (series * P.cin + m) * (int64_t)ss;
      for (int e = g.gl; e < ss; e += 32) dst[e] = st[e];
      if (m + 1 == m1) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = g.gl; e < es; e += 32) el[e] = src[e];
      g.sync();
      const double *mv = st, *Pm = st + n;
      // Ws = [I + P J | m + P eta | P]
      mm(g, n, n1, n, Pm, n, 1, J, n1, 1, (const double*)nullptr, 0, 0, Ws, ld, 1); // cols 0..n: P [J | eta]
      g.sync();
      for (int e = g.gl; e < n * n; e += 32) { const int i = e / n, j = e - i * n; Ws[i * ld + n1 + j] = Pm[e]; }
      for (int i = g.gl; i < n; i += 32) { Ws[i * ld + i] += 1.0; Ws[i * ld + n] += mv[i]; }
      g.sync();
      gj_solve(g, n, ld, Ws);
      // m' = A x + b ; Tm = A X ; P' = Tm A^T + C
      for (int i = g.gl; i < n; i += 32) {
        double acc = A[i * n1 + n];
        for (int l = 0; l < n; ++l) acc = fma(A[i * n1 + l], Ws[l * ld + n], acc);
        st2[i] = acc;
      }
      mm(g, n, n, n, A, n1, 1, Ws + n1, ld, 1, (const double*)nullptr, 0, 0, Tm, n, 1);
      g.sync();
      mm_sym(g, T, n, Tm, n, 1, A, 1, n1, C, st2 + n);
      g.sync();
      double* t = st; st = st2; st2 = t;
    }
  } else {
    if (!P.want_suffix) return;
    // st = [eta | J]
    if (P.SUFup) { const double* s = P.SUFup + gid * (int64_t)ss; for (int e = g.gl; e < ss; e += 32) st[e] = s[e]; }
    else { for (int e = g.gl; e < ss; e += 32) st[e] = 0.0; }
    g.sync();
    for (int64_t m = m1 - 1; m >= m0; --m) {
      double* dst = P.SUF + (series * P.cin + m) * (int64_t)ss;
      for (int e = g.gl; e < ss; e += 32) dst[e] = st[e];
      if (m == m0) break;
      const double* src = P.Ein + (series * P.cin + m) * (int64_t)es;
      for (int e = g.gl; e < es; e += 32) el[e] = src[e];
      g.sync();
      const double *ev = st, *Je = st + n;
      const int ld2 = 2 * n;
      // Ws = [I + C J_e | A]
      mm(g, n, n, n, C, n, 1, Je, n, 1, (const double*)nullptr, 0, 0, Ws, ld2, 1);
      g.sync();
      for (int e = g.gl; e < n * n; e += 32) { const int i = e / n, j = e - i * n; Ws[i * ld2 + n + j] = A[i * n1 + j]; }
      for (int i = g.gl; i < n; i += 32) Ws[i * ld2 + i] += 1.0;
      // u = eta_e - J_e b
      for (int i = g.gl; i < n; i += 32) {
        double acc = ev[i];
        for (int l = 0; l < n; ++l) acc = fma(-Je[i * n + l], A[l * n1 + n], acc);
        uv[i] = acc;
      }
      g.sync();
      gj_solve(g, n, ld2, Ws);
      const double* X = Ws + n; // M A, row stride ld2
      for (int i = g.gl; i < n; i += 32) {
        double acc = J[i * n1 + n];
        for (int l = 0; l < n; ++l) acc = fma(X[l * ld2 + i], uv[l], acc);
        st2[i] = acc;
      }
      mm(g, n, n, n, Je, n, 1, A, n1, 1, (const double*)nullptr, 0, 0, Tm, n, 1); // Tm = J_e A
      g.sync();
      for (int e = g.gl; e < T.ntri; e += 32) {
        const int i = T.tri_i[e], j = T.tri_j[e];
        double acc = J[i * n1 + j];
        for (int l = 0; l < n; ++l) acc = fma(X[l * ld2 + i], Tm[l * n + j], acc);
        st2[n + i * n + j] = acc;
        st2[n + j * n + i] = acc;
      }
      g.sync();
      double* t = st; st = st2; st2 = t;
    }
  }
}

// Backward information step over one transition (F, Q):  J <- F^T (I + J Q)^-1 J F,
// eta <- F^T (I + J Q)^-1 eta  (the (eta, J) part of the SG21 combine with a primitive start-type
// element on the left, reading R1).  Ws: n x (2n+1), Tm: n x n scratch.  Ends synchronised.
template <int G>
__device__ void info_backstep(const Grp<G>& g, const Tables& T, const double* Fs, const double* Qs, double* Jm, double* ev,
                              double* Ws, double* Tm) {
  const int n = T.n, ld = 2 * n + 1;
  mm(g, n, n, n, Jm, n, 1, Qs, n, 1, (const double*)nullptr, 0, 0, Ws, ld, 1);
  g.sync();
  for (int e = g.gl; e < n * n; e += G) { const int i = e / n, j = e - i * n; Ws[i * ld + n + j] = Jm[e]; }
  for (int i = g.gl; i < n; i += G) { Ws[i * ld + i] += 1.0; Ws[i * ld + 2 * n] = ev[i]; }
  g.sync();
  gj_solve(g, n, ld, Ws);
  // Tm = F^T Y ; eta = F^T y ; J = F^T Tm^T  (Y symmetric)
  lmul_Ft(g, T, Fs, Ws + n, ld, 1, Tm, n, 1, n);
  lmul_Ft(g, T, Fs, Ws + 2 * n, ld, 0, ev, 1, 0, 1);
  g.sync();
  lmul_Ft(g, T, Fs, Tm, 1, n, Jm, n, 1, n); // src = Tm^T
  g.sync();
  // symmetrise (the two triangles were computed independently)
  for (int e = g.gl; e < T.ntri; e += G) {
    const int i = T.tri_i[e], j = T.tri_j[e];
    const double w = 0.5 * (Jm[i * n + j] + Jm[j * n + i]);
    Jm[i * n + j] = w;
    Jm[j * n + i] = w;
  }
  g.sync();
}

// ---------------------------------------------------------------------------------------------------
// k_down0: per chunk, forward Kalman filter from the prefix state, then backward information
// recursion from the suffix information with the smoothed output at every end event.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int down0_group_doubles(int n) { return 7 * n * n + 6 * n + 2; }

template <int G>
__global__ void __launch_bounds__(128) k_down0(ScanDev P) {
  extern __shared__ __align__(16) char smem[];
  Tables T;
  tables_build(P.M, smem, T);
  __syncthreads();
  const int n = T.n, d = T.d;
  const size_t tb = tables_bytes(n, d, T.ninst, T.nblk, T.nent);
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * down0_group_doubles(n);
  double* Fs = base;
  double* Qs = Fs + n * n;
  double* Pm = Qs + n * n;
  double* Tm = Pm + n * n;
  double* Jm = Tm + n * n;
  double* Ws = Jm + n * n;           // n x (2n+1)
  double* mv = Ws + n * (2 * n + 1); // n
  double* m2 = mv + n;               // n
  double* ev = m2 + n;               // n
  double* cv = ev + n;               // n
  const int ss = state_size(n);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ampv = P.amp ? P.amp[series] : 1.0;
  const double ramp = 1.0 / ampv;

  zero_fill(g, Fs, 2 * n * n);
  if (P.PRE1) {
    const double* s = P.PRE1 + gid * (int64_t)ss;
    for (int e = g.gl; e < n; e += G) mv[e] = s[e];
    for (int e = g.gl; e < n * n; e += G) Pm[e] = s[n + e];
  } else {
    for (int e = g.gl; e < n; e += G) mv[e] = 0.0;
    for (int e = g.gl; e < n * n; e += G) Pm[e] = P.M->p0[e];
  }
  g.sync();
  double ll = 0.0;
  // ---- forward: Eq. 3.14 (predict), 3.15 (reset, folded into the step), 2.22 (update), 2.26 ----
  for (int64_t k = k0; k < k1; ++k) {
    const uint32_t meta = P.meta[k];
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    assemble_step(g, T, P.disc + k * (int64_t)T.stride, tz, Fs, Qs);
    g.sync();
    lmul_F(g, T, Fs, mv, 1, 0, m2, 1, 0, 1);
    lmul_F(g, T, Fs, Pm, n, 1, Tm, n, 1, n);
    g.sync();
    rmul_Ft_sym(g, T, Fs, Tm, Qs, Pm);
    g.sync();
    { double* t = mv; mv = m2; m2 = t; }
    if (!kind) {
      const int zi = d + q;
      const int32_t ob = P.obs[k];
      const double hs = T.tau[q] / P.delta[k];
      const double sg = P.sigma[ob] * ramp;
      const double yy = P.y[series * P.N + ob] * ramp;
      const double S = hs * hs * Pm[zi * n + zi] + sg * sg;
      const double v = yy - hs * mv[zi];
      if (!(S > 0.0) || !isfinite(S) || !isfinite(v)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      ll -= 0.5 * (log(6.283185307179586476925286766559 * S) + v * v * rS);
      for (int i = g.gl; i < n; i += G) cv[i] = hs * Pm[i * n + zi];
      g.sync();
      for (int i = g.gl; i < n; i += G) mv[i] = fma(cv[i] * rS, v, mv[i]);
      for (int e = g.gl; e < T.ntri; e += G) {
        const int i = T.tri_i[e], j = T.tri_j[e];
        const double w = fma(-cv[i] * rS, cv[j], Pm[i * n + j]);
        Pm[i * n + j] = w;
        Pm[j * n + i] = w;
      }
      g.sync();
      if (P.want_smooth) { // X_k: filtered state at the end event (before z_q is dropped)
        double* x = P.xbuf + (series * P.N + ob) * (int64_t)ss;
        for (int e = g.gl; e < n; e += G) x[e] = mv[e];
        for (int e = g.gl; e < n * n; e += G) x[n + e] = Pm[e];
      }
      g.sync();
      if (g.gl == 0) mv[zi] = 0.0;
      for (int j = g.gl; j < n; j += G) { Pm[zi * n + j] = 0.0; Pm[j * n + zi] = 0.0; }
      g.sync();
    }
    if (P.fstate) { // row a7: all 2N filtered states are kept for prediction at arbitrary times
      double* x = P.fstate + (series * P.K + k) * (int64_t)ss;
      for (int e = g.gl; e < n; e += G) x[e] = mv[e];
      for (int e = g.gl; e < n * n; e += G) x[n + e] = Pm[e];
    }
  }
  if (g.gl == 0) P.llpart[gid] = ll;
  if (!P.want_smooth) return;

  // ---- backward: information (eta, J) about the state after event k held by all later data ----
  if (P.SUF1) {
    const double* s = P.SUF1 + gid * (int64_t)ss;
    for (int e = g.gl; e < n; e += G) ev[e] = s[e];
    for (int e = g.gl; e < n * n; e += G) Jm[e] = s[n + e];
  } else {
    for (int e = g.gl; e < n; e += G) ev[e] = 0.0;
    for (int e = g.gl; e < n * n; e += G) Jm[e] = 0.0;
  }
  g.sync();
  for (int64_t k = k1 - 1; k >= k0; --k) {
    const uint32_t meta = P.meta[k];
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    // components zeroed after event k carry no information backwards
    for (int r = 0; r < T.ninst; ++r)
      if ((zm >> r) & 1u) {
        const int zr = d + r;
        if (g.gl == 0) ev[zr] = 0.0;
        for (int j = g.gl; j < n; j += G) { Jm[zr * n + j] = 0.0; Jm[j * n + zr] = 0.0; }
      }
    g.sync();
    if (!kind) {
      const int zi = d + q;
      const int32_t ob = P.obs[k];
      const double hs = T.tau[q] / P.delta[k];
      const double sg = P.sigma[ob] * ramp;
      const double yy = P.y[series * P.N + ob] * ramp;
      const double* x = P.xbuf + (series * P.N + ob) * (int64_t)ss;
      for (int e = g.gl; e < n; e += G) m2[e] = x[e];
      for (int e = g.gl; e < n * n; e += G) Pm[e] = x[n + e];
      g.sync();
      // P^ = (I + P J)^-1 P,  m^ = (I + P J)^-1 (m + P eta): solve for the z_q column / the mean
      const int ld = n + 2;
      mm(g, n, n, n, Pm, n, 1, Jm, n, 1, (const double*)nullptr, 0, 0, Ws, ld, 1);
      g.sync();
      for (int i = g.gl; i < n; i += G) {
        Ws[i * ld + i] += 1.0;
        Ws[i * ld + n] = Pm[i * n + zi];
        double acc = m2[i];
        for (int l = 0; l < n; ++l) acc = fma(Pm[i * n + l], ev[l], acc);
        Ws[i * ld + n + 1] = acc;
      }
      g.sync();
      gj_solve(g, n, ld, Ws);
      if (g.gl == 0) {
        const double sv = Ws[zi * ld + n], sm = Ws[zi * ld + n + 1];
        if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
        P.mean[series * P.N + ob] = ampv * hs * sm;          // H~ m^
        P.var[series * P.N + ob] = ampv * ampv * hs * hs * sv; // H~ P^ H~^T
        // the observation's own information: h h^T / r, h y / r
        const double rr = 1.0 / (sg * sg);
        Jm[zi * n + zi] += hs * hs * rr;
        ev[zi] += hs * yy * rr;
      }
      g.sync();
    }
    if (P.binfo) {
      double* x = P.binfo + (series * P.K + k) * (int64_t)ss;
      for (int e = g.gl; e < n; e += G) x[e] = ev[e];
      for (int e = g.gl; e < n * n; e += G) x[n + e] = Jm[e];
    }
    if (k == k0) break;
    // back over the step into event k:  J <- F^T (I + J Q)^-1 J F,  eta <- F^T (I + J Q)^-1 eta
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    assemble_step(g, T, P.disc + k * (int64_t)T.stride, tz, Fs, Qs);
    g.sync();
    info_backstep(g, T, Fs, Qs, Jm, ev, Ws, Tm);
  }
}

__global__ void k_ll_reduce(const double* __restrict__ llpart, int64_t c1, int64_t batch, int64_t N,
                            const double* __restrict__ amp, double* __restrict__ loglik) {
  // one warp per series; fixed summation order (lane-strided partial sums, then a butterfly)
  const int64_t s = (int64_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  if (s >= batch) return;
  const int lane = threadIdx.x & 31;
  double acc = 0.0;
  for (int64_t c = lane; c < c1; c += 32) acc += llpart[s * c1 + c];
  for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) loglik[s] = acc - (amp ? (double)N * log(amp[s]) : 0.0);
}

// ---------------------------------------------------------------------------------------------------
// Row a7: prediction at arbitrary times (Algorithm 1) in two-filter form.
// k_query_locate: kp[q] = last event with t_k <= t*_q (-1 if none);  dtq[q] = t* - t_kp (0 if none),
// dtq[M + q] = t_{kp+1} - t* (0 if kp is the last event).  k_disc then discretises the 2M steps.
// k_query: one group per (series, query).
// ---------------------------------------------------------------------------------------------------
__global__ void k_query_locate(int64_t M, const double* __restrict__ tq, int64_t K, const double* __restrict__ t,
                               int64_t* __restrict__ kp, double* __restrict__ dtq) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= M) return;
  const double ts = tq[q];
  int64_t lo = -1, hi = K; // invariant: t[lo] <= ts < t[hi]
  while (hi - lo > 1) {
    const int64_t mid = (lo + hi) >> 1;
    if (t[mid] <= ts) lo = mid; else hi = mid;
  }
  kp[q] = lo;
  dtq[q] = (lo >= 0) ? ts - t[lo] : 0.0;
  dtq[M + q] = (lo + 1 < K) ? t[lo + 1] - ts : 0.0;
}

struct QueryDev {
  const ModelDev* M;
  const double* discq; // [2M][stride]
  const int64_t* kp;   // [M]
  const uint32_t* meta;
  const double* fstate;
  const double* binfo;
  const double* amp;
  int64_t K, Mq, batch;
  int qinst;
  double* mean; // [batch][M]
  double* var;
  int* flags;
};

template <int G>
__global__ void __launch_bounds__(128) k_query(QueryDev P) {
  extern __shared__ __align__(16) char smem[];
  Tables T;
  tables_build(P.M, smem, T);
  __syncthreads();
  const int n = T.n, d = T.d;
  const size_t tb = tables_bytes(n, d, T.ninst, T.nblk, T.nent);
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.Mq) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * down0_group_doubles(n);
  double* Fs = base;
  double* Qs = Fs + n * n;
  double* Pm = Qs + n * n;
  double* Tm = Pm + n * n;
  double* Jm = Tm + n * n;
  double* Ws = Jm + n * n;           // n x (2n+1)
  double* mv = Ws + n * (2 * n + 1); // n
  double* m2 = mv + n;               // n
  double* ev = m2 + n;               // n
  double* hv = ev + n;               // n: H_q in block units
  const int ss = state_size(n);
  const int64_t series = gid / P.Mq, q = gid - series * P.Mq;
  const int64_t kp = P.kp[q];
  const double ampv = P.amp ? P.amp[series] : 1.0;
  zero_fill(g, Fs, 2 * n * n);
  for (int i = g.gl; i < n; i += G) hv[i] = 0.0;
  g.sync();
  if (g.gl == 0)
    for (int b = 0; b < T.nblk; ++b) hv[P.M->blk[b].off] = P.M->hq[P.qinst][b];
  // ---- state just after the last event at or before t* (stationary prior with idle z = 0 if none) ----
  if (kp >= 0) {
    const double* s = P.fstate + (series * P.K + kp) * (int64_t)ss;
    for (int e = g.gl; e < n; e += G) mv[e] = s[e];
    for (int e = g.gl; e < n * n; e += G) Pm[e] = s[n + e];
    g.sync();
    // predict over Delta_1 (Eq. 3.14); instruments idle after event kp stay zeroed
    const uint32_t mp = P.meta[kp]; // idle through (t_kp, t_kp+1): zeroed after kp, except an instrument that just started
    const unsigned idle = META_KIND(mp) ? (META_ZMASK(mp) & ~(1u << META_INST(mp))) : META_ZMASK(mp);
    assemble_step(g, T, P.discq + q * (int64_t)T.stride, idle, Fs, Qs);
    g.sync();
    lmul_F(g, T, Fs, mv, 1, 0, m2, 1, 0, 1);
    lmul_F(g, T, Fs, Pm, n, 1, Tm, n, 1, n);
    g.sync();
    rmul_Ft_sym(g, T, Fs, Tm, Qs, Pm);
    g.sync();
    { double* t = mv; mv = m2; m2 = t; }
  } else {
    for (int e = g.gl; e < n; e += G) mv[e] = 0.0;
    for (int e = g.gl; e < n * n; e += G) Pm[e] = P.M->p0[e];
    g.sync();
  }
  // ---- information about the state at t* from every later event ----
  if (kp + 1 < P.K) {
    const int64_t kn = kp + 1;
    const double* s = P.binfo + (series * P.K + kn) * (int64_t)ss;
    for (int e = g.gl; e < n; e += G) ev[e] = s[e];
    for (int e = g.gl; e < n * n; e += G) Jm[e] = s[n + e];
    const uint32_t meta = P.meta[kn];
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = META_KIND(meta) ? zm : (zm & ~(1u << META_INST(meta)));
    g.sync();
    assemble_step(g, T, P.discq + (P.Mq + q) * (int64_t)T.stride, tz, Fs, Qs);
    g.sync();
    info_backstep(g, T, Fs, Qs, Jm, ev, Ws, Tm);
    // fuse: P^ = (I + P J)^-1 P, m^ = (I + P J)^-1 (m + P eta); right-hand sides P h and m + P eta
    const int ld = n + 2;
    mm(g, n, n, n, Pm, n, 1, Jm, n, 1, (const double*)nullptr, 0, 0, Ws, ld, 1);
    g.sync();
    for (int i = g.gl; i < n; i += G) {
      Ws[i * ld + i] += 1.0;
      double a = 0.0, acc = mv[i];
      for (int l = 0; l < n; ++l) { a = fma(Pm[i * n + l], hv[l], a); acc = fma(Pm[i * n + l], ev[l], acc); }
      Ws[i * ld + n] = a;
      Ws[i * ld + n + 1] = acc;
    }
    g.sync();
    gj_solve(g, n, ld, Ws);
    if (g.gl == 0) {
      double sv = 0.0, sm = 0.0;
      for (int i = 0; i < n; ++i) { sv = fma(hv[i], Ws[i * ld + n], sv); sm = fma(hv[i], Ws[i * ld + n + 1], sm); }
      if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
      P.mean[series * P.Mq + q] = ampv * sm;
      P.var[series * P.Mq + q] = ampv * ampv * sv;
    }
  } else if (g.gl == 0) { // extrapolation past the last event: the prediction itself
    double sv = 0.0, sm = 0.0;
    for (int i = 0; i < n; ++i) {
      sm = fma(hv[i], mv[i], sm);
      for (int j = 0; j < n; ++j) sv = fma(hv[i] * hv[j], Pm[i * n + j], sv);
    }
    P.mean[series * P.Mq + q] = ampv * sm;
    P.var[series * P.Mq + q] = ampv * ampv * sv;
  }
}

#include "scan_host.cu"
