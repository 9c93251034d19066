// chunk_kernels.cuh -- the per-chunk sequential kernels (k_fold0, k_down0, k_query) and their
// parameter blocks.  Self-contained device code on top of dev_consts.h, grp_dev.cuh and chunk_dev.cuh:
// the same text is compiled statically (generic tables in the kernel parameters) and, specialised for
// one model, at run time (jit.cu: tables become compile-time constants, every loop unrolls).
#pragma once
#include "chunk_dev.cuh"

// element layout in global memory: AB [n x (n+1)] = [A | b],  C [n x n],  JE [n x (n+1)] = [J | eta]
__host__ __device__ inline int elem_size(int n) { return 3 * n * n + 2 * n; }
__host__ __device__ inline int state_size(int n) { return n * n + n; } // [vector | matrix]

struct ScanDev {
  Tab T;           // model tables (constant bank)
  const double* p0;  // [n][n] prior covariance blkdiag(Pinf, 0) in block units (Eq. 3.19, reading R6)
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
  const double* ADJ1; // [batch*c1][state] adjoint [lambda^ | Lambda^] at each chunk's last event (k_adjD; register kernels only) or NULL (zero)
  double* kbuf;    // [batch*N][2n+4] per end event: gain K, filtered z-column p, S, v, filtered z mean
  double* fstate;  // [batch*K][state] post-event filtered state of every event, or NULL (a7)
  double* binfo;   // [batch*K][state] information [eta | J] about the pre-update state of every event, or NULL (a7)
  double* llpart;  // [batch*c1]
  double* mean;
  double* var;
  int* flags;
  int want_smooth;
};

// shared memory of one group of the register-resident kernels (chunk_reg.cuh): exchange buffer, two record
// buffers + 2 mbarriers, three vector buffers.  Sizes in doubles; = 8 (mod 16) so that neighbouring groups of a
// warp fall on complementary banks.
__host__ __device__ inline int reg_ldt(int n) { return (n + 2) | 1; }
__host__ __device__ inline int reg_tm(int n) { return ((n * reg_ldt(n) + 7) / 16) * 16 + 8; }
__host__ __device__ inline int reg_vb(int n) { return 2 * (n + 2); }
__host__ __device__ inline int reg_group_doubles(int n, int stride) { return ((reg_tm(n) + 2 * stride + 2 + 3 * reg_vb(n) + 7) / 16) * 16 + 8; }
__host__ __device__ inline int reg_czs(int ni, int nb) { return ((ni + 1) * nb + 1) & ~1; }

// ---------------------------------------------------------------------------------------------------
// k_fold0: chunk -> element.  Column-owned layout of chunk_dev.cuh.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int fold0_group_doubles(int n, int ld, int stride, int nblk, int G) {
  const int nr = ld - 1; // nr >= n rows: the padding rows stay zero, so row loops run to the compile-time nr
  return (4 * nr * ld + 2 * stride + 2 + nblk * G + 2 * ld + 2 + 1) & ~1; // even: record buffers stay 16-byte aligned; + 2 mbarriers
}

template <int G, int LD>
__device__ __forceinline__ void fold0_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int ld = LD;
  const int n = TN, d = TD;
  const size_t tb = 0;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * fold0_group_doubles(n, LD, TSTRIDE, TNB, G);
  constexpr int NR = LD - 1;
  double* AB0 = base;            // [A | b]
  double* C = AB0 + NR * ld;
  double* Tm = C + NR * ld;
  double* JE = Tm + NR * ld;     // [J | eta]
  double* recs = JE + NR * ld;   // 2 x stride
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* av = recs + 2 * TSTRIDE + 2 + TNB * G; // NR (zero padded) + 1: av[NR] = hs b_z
  double* cv = av + ld;                           // NR (zero padded)
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ramp = P.amp ? 1.0 / P.amp[series] : 1.0;

  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)TSTRIDE, 0);
  zero_fill(g, AB0, 4 * NR * ld);
  zero_fill(g, av, 2 * ld);
  g.sync();
  for (int i = g.gl; i < n; i += G) AB0[i * ld + i] = 1.0;
  g.sync();

  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const double* rec = rs.wait((int)((k - k0) & 1));
    g.sync();
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)TSTRIDE, (int)((k + 1 - k0) & 1));
    // event k's scalars were requested one iteration ago; the data of an end event are requested now
    // and consumed after the products, so no global latency sits on the per-event critical path
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    // [A | b] <- F [A | b], in place: a lane reads a block of its column into registers before it
    // writes that block, and the z rows read only z entries, which are written last
    if (g.gl <= n) apply_F<G, LD, LD>(T, rec, tz, AB0 + g.gl, AB0 + g.gl, U);
    // C <- F C F^T + Q
    sandwich_F<G, LD, true>(g, T, rec, tz, C, Tm, U);
    if (!kind) {
      // observe z_q / delta: h = hs e_z in equilibrated units (Eq. 3.12); SG21 Eq. 10 with the
      // aggregate as the earlier element (rank-one J_j): Sherman-Morrison form of the combine
      const int zi = d + q;
      const double hs = TTAU(q) / dl_r;
      const double sg = sg_r * ramp;
      const double yy = y_r * ramp;
      const double S = hs * hs * C[zi * ld + zi] + sg * sg;
      if (!(S > 0.0) || !isfinite(S)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      const int j = g.gl;
      if (j < n) { av[j] = hs * AB0[zi * ld + j]; cv[j] = hs * C[j * ld + zi]; }
      else if (j == n) av[NR] = hs * AB0[zi * ld + n];
      g.sync();
      const double resid = yy - av[NR];
      if (j <= n) {
        // column j of J += a a_j / S, of A -= c a_j / S; last column: eta += a resid / S, b += c resid / S
        const double aj = (j < n) ? av[j] * rS : resid * rS;
        const double sgn = (j < n) ? -1.0 : 1.0;
        const double cj = (j < n) ? cv[j] * rS : 0.0;
#pragma unroll
        for (int i = 0; i < NR; ++i) {
          JE[i * ld + j] = fma(av[i], aj, JE[i * ld + j]);
          AB0[i * ld + j] = fma(sgn * cv[i], aj, AB0[i * ld + j]);
          C[i * ld + j] = fma(-cv[i], cj, C[i * ld + j]); // column n of C is scratch (cj = 0 there)
        }
      }
      g.sync();
      // the instrument is idle after its end: zero z_q (reading R6)
      if (j <= n) { AB0[zi * ld + j] = 0.0; if (j < n) { C[zi * ld + j] = 0.0; C[j * ld + zi] = 0.0; } }
      g.sync();
    }
  }
  double* out = P.E1 + gid * (int64_t)elem_size(n);
  const int n1 = n + 1;
  for (int j = g.gl; j <= n; j += G)
    for (int i = 0; i < n; ++i) {
      out[i * n1 + j] = AB0[i * ld + j];
      out[n * n1 + n * n + i * n1 + j] = JE[i * ld + j];
      if (j < n) out[n * n1 + i * n + j] = 0.5 * (C[i * ld + j] + C[j * ld + i]);
    }
}

// ---------------------------------------------------------------------------------------------------
// k_down0: per chunk, (1) the plain integrated Kalman filter (Eq. 3.14 predict, 3.15 reset folded into
// the step, 2.22 update) from the chunk's prefix state: innovations -> log-likelihood terms (Eq. 2.26),
// and per end event the gain K, innovation (v, S) and the filtered z-column p kept in `kbuf`;
// (2) the smoother as the adjoint (modified Bryson-Frazier) recursion of that same filter, started
// from the chunk's suffix information (eta, J) of the reverse scan:
//     Lambda^ = (I + J P)^-1 J,  lambda^ = (I + J P)^-1 (J m - eta)        at the chunk's last event,
//     end event:  smoothed  m^ = m_f - P_f lambda^,  P^ = P_f - P_f Lambda^ P_f   (z entries only),
//                 Lambda~ = C^T Lambda^ C + h h^T / S,  lambda~ = C^T lambda^ - h v / S,  C = I - K h^T,
//     step:       Lambda^ <- F^T Lambda~ F,  lambda^ <- F^T lambda~.
// It is the two-filter posterior of reading R7 written without any per-event inverse (Lambda^ =
// (I + J P)^-1 J at every event): the only solves left are one per chunk here and those of the
// dense levels.  DESIGN.md 5.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int kbuf_stride(int n) { return 2 * n + 4; }
__host__ __device__ inline int down0_group_doubles(int n, int ld, int stride, int nblk, int G) {
  const int nr = ld - 1, ws = ((n * (2 * n + 1) > nr * ld ? n * (2 * n + 1) : nr * ld) + 1) & ~1;
  return (nr * ld + ws + 2 * stride + 2 + nblk * G + 5 * ld + 1 + 1) & ~1; // Tm is the head of Ws; even sizes keep the record buffers aligned
}

// [vector | matrix(n x n)] in global memory  <->  column-owned [matrix | vector] with row stride ld
template <int G, int LD>
__device__ __forceinline__ void load_state(const Grp<G>& g, const Tab& T, const double* s, double* X) {
  constexpr int ld = LD;
  const int n = TN;
  for (int j = g.gl; j <= n; j += G)
    for (int i = 0; i < n; ++i) X[i * ld + j] = (j < n) ? s[n + i * n + j] : s[i];
}
template <int G, int LD>
__device__ __forceinline__ void store_state(const Grp<G>& g, const Tab& T, const double* X, double* s) {
  constexpr int ld = LD;
  const int n = TN;
  for (int j = g.gl; j <= n; j += G)
    for (int i = 0; i < n; ++i) {
      if (j < n) s[n + i * n + j] = X[i * ld + j];
      else s[i] = X[i * ld + n];
    }
}

template <int G, int LD>
__device__ __forceinline__ void down0_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int ld = LD;
  const int n = TN, d = TD;
  const size_t tb = 0;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * down0_group_doubles(n, LD, TSTRIDE, TNB, G);
  constexpr int NR = LD - 1;        // rows allocated (>= n): padding rows and vector tails stay zero
  double* X = base;                 // [P | m], later [Lambda | lambda]
  double* Tm = X + NR * ld;
  double* Ws = Tm;                  // n x (2n+1), used only for the one solve per chunk (Tm is dead there)
  double* recs = Ws + (((n * (2 * n + 1) > NR * ld ? n * (2 * n + 1) : NR * ld) + 1) & ~1);
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* cv = recs + 2 * TSTRIDE + 2 + TNB * G; // NR, zero padded
  double* kv = cv + ld;
  double* pv = kv + ld;
  double* av = pv + ld;             // n + 1
  double* gv = av + ld;             // n + 1
  const int ss = state_size(n), ks = kbuf_stride(n);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ampv = P.amp ? P.amp[series] : 1.0;
  const double ramp = 1.0 / ampv;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);

  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)TSTRIDE, 0);
  zero_fill(g, X, 2 * NR * ld);
  zero_fill(g, cv, 5 * ld);
  g.sync();
  if (P.PRE1) load_state<G, LD>(g, T, P.PRE1 + gid * (int64_t)ss, X);
  else
    for (int j = g.gl; j <= n; j += G)
      for (int i = 0; i < n; ++i) X[i * ld + j] = (j < n) ? P.p0[i * n + j] : 0.0;
  g.sync();
  double ll = 0.0;
  int nend = 0; // end events seen by this chunk (forward, then backward)
  // ---- forward ----
  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const double* rec = rs.wait((int)((k - k0) & 1));
    g.sync();
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)TSTRIDE, (int)((k + 1 - k0) & 1));
    const uint32_t meta = meta_nx; // prefetched: see k_fold0
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    sandwich_F<G, LD, true>(g, T, rec, tz, X, Tm, U);
    if (!kind) {
      const int zi = d + q;
      const double hs = TTAU(q) / dl_r;
      const double sg = sg_r * ramp;
      const double yy = y_r * ramp;
      const double S = hs * hs * X[zi * ld + zi] + sg * sg;
      const double v = yy - hs * X[zi * ld + n];
      if (!(sg_r > 0.0) || !isfinite(sg_r)) atomicOr(P.flags, NUMF_SIGMA);
      if (!(S > 0.0) || !isfinite(S) || !isfinite(v)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / S;
      ll -= 0.5 * (log(6.283185307179586476925286766559 * S) + v * v * rS);
      for (int i = g.gl; i < n; i += G) cv[i] = hs * X[i * ld + zi];
      g.sync();
      if (g.gl <= n) {
        const int j = g.gl;
        const double cj = (j < n) ? -cv[j] * rS : v * rS;
#pragma unroll
        for (int i = 0; i < NR; ++i) X[i * ld + j] = fma(cv[i], cj, X[i * ld + j]);
      }
      g.sync();
      if (P.want_smooth) {
        double* kb = P.kbuf + (series * P.N + ob) * (int64_t)ks;
        for (int i = g.gl; i < n; i += G) { kb[i] = cv[i] * rS; kb[n + i] = X[i * ld + zi]; }
        if (g.gl == 0) { kb[2 * n] = S; kb[2 * n + 1] = v; kb[2 * n + 2] = X[zi * ld + n]; }
        g.sync();
      }
      // the instrument is idle after its end (reading R6)
      if (g.gl <= n) { const int j = g.gl; X[zi * ld + j] = 0.0; if (j < n) X[j * ld + zi] = 0.0; }
      g.sync();
      // the two triangles of F P F^T are rounded independently: re-symmetrised every 4th end event (the
      // asymmetry is pure rounding and grows slowly; the transposed accesses conflict in shared memory)
      if ((++nend & 3) == 0) symmetrise<G, LD>(g, T, X);
    }
    if (P.fstate) store_state<G, LD>(g, T, X, P.fstate + (series * P.K + k) * (int64_t)ss); // row a7
  }
  if (g.gl == 0) P.llpart[gid] = ll;
  if (!P.want_smooth) return;

  // ---- adjoint at the chunk's last event from the suffix information ----
  rs.issue(g, P.disc + (k1 - 1) * (int64_t)TSTRIDE, 0);
  if (P.SUF1) {
    const int ld2 = 2 * n + 1;
    // Ws = [I + J P | J | J m - eta]: J goes straight to its place, eta is parked in column 2n
    const double* sj = P.SUF1 + gid * (int64_t)ss;
    for (int j = g.gl; j <= n; j += G)
      for (int i = 0; i < n; ++i) Ws[i * ld2 + n + j] = (j < n) ? sj[n + i * n + j] : sj[i];
    g.sync();
    for (int j = g.gl; j <= n; j += G)
      for (int i = 0; i < n; ++i) {
        double acc = 0.0, cmp = 0.0; // J P cancels like the products of the dense levels: compensated (Dot2)
        for (int l = 0; l < n; ++l) dot2_step(Ws[i * ld2 + n + l], X[l * ld + j], acc, cmp);
        acc += cmp;
        if (j < n) Ws[i * ld2 + j] = acc + (i == j ? 1.0 : 0.0);
        else Ws[i * ld2 + 2 * n] = acc - Ws[i * ld2 + 2 * n];
      }
    g.sync();
    gj_solve(g, n, ld2, Ws);
    for (int j = g.gl; j <= n; j += G)
      for (int i = 0; i < n; ++i)
        X[i * ld + j] = (j < n) ? 0.5 * (Ws[i * ld2 + n + j] + Ws[j * ld2 + n + i]) : Ws[i * ld2 + 2 * n];
  } else {
    zero_fill(g, X, n * ld);
  }
  g.sync();
  zero_fill(g, Tm, NR * ld); // the solve used this region as Ws
  g.sync();
  // ---- backward ----
  // backward prefetch: meta / exposure index one event ahead, the end event's kbuf record (one entry of
  // K and of p per lane, S, v, filtered z mean) and exposure length requested before the previous step
  meta_nx = P.meta[k1 - 1];
  ob_nx = P.obs[k1 - 1];
  double kv_r = 0.0, pv_r = 0.0, S_r = 1.0, v_r = 0.0, m_r = 0.0, dlb_r = 1.0;
  if (!META_KIND(meta_nx)) {
    const double* kb = P.kbuf + (series * P.N + ob_nx) * (int64_t)ks;
    if (g.gl < n) { kv_r = kb[g.gl]; pv_r = kb[n + g.gl]; }
    S_r = kb[2 * n]; v_r = kb[2 * n + 1]; m_r = kb[2 * n + 2]; dlb_r = P.delta[k1 - 1];
  }
  for (int64_t k = k1 - 1; k >= k0; --k) {
    const double* rec = rs.wait((int)((k1 - 1 - k) & 1));
    g.sync();
    if (k > k0) rs.issue(g, P.disc + (k - 1) * (int64_t)TSTRIDE, (int)((k1 - k) & 1));
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    const double kv_c = kv_r, pv_c = pv_r, S = S_r, v = v_r, mfz = m_r, dl_c = dlb_r;
    if (k > k0) { meta_nx = P.meta[k - 1]; ob_nx = P.obs[k - 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    // components zeroed after event k pass nothing backwards (adjoint of the zeroing)
    for (int r = 0; r < TNI; ++r)
      if ((zm >> r) & 1u) {
        const int zr = d + r;
        if (g.gl <= n) { const int j = g.gl; X[zr * ld + j] = 0.0; if (j < n) X[j * ld + zr] = 0.0; }
      }
    g.sync();
    if (!kind) {
      const int zi = d + q;
      const double hs = TTAU(q) / dl_c;
      if (g.gl < n) { kv[g.gl] = kv_c; pv[g.gl] = pv_c; }
      const double rS = 1.0 / S;
      g.sync();
      double quad = 0.0, kap = 0.0;
      if (g.gl <= n) {
        const int j = g.gl;
        double a = 0.0, b = 0.0;
#pragma unroll
        for (int i = 0; i < NR; ++i) { const double x = X[i * ld + j]; a = fma(x, pv[i], a); b = fma(x, kv[i], b); }
        av[j] = a; gv[j] = b;
        if (j < n) { quad = pv[j] * a; kap = kv[j] * b; }
      }
      quad = group_sum(g, quad);
      kap = group_sum(g, kap);
      g.sync();
      if (g.gl == 0) {
        const double sm = mfz - av[n], sv = pv[zi] - quad;
        if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
        P.mean[series * P.N + ob] = ampv * hs * sm;            // H~ m^
        P.var[series * P.N + ob] = ampv * ampv * hs * hs * sv; // H~ P^ H~^T
      }
      // Lambda~ = C^T Lambda^ C + h h^T / S: only row and column z change (h = hs e_z)
      if (g.gl <= n) {
        const int j = g.gl;
        if (j < n) {
          X[zi * ld + j] -= hs * gv[j];
          X[j * ld + zi] -= hs * gv[j];
          if (j == zi) X[zi * ld + zi] += hs * hs * (kap + rS);
        } else {
          X[zi * ld + n] -= hs * (gv[n] + v * rS);
        }
      }
      g.sync();
      if ((++nend & 3) == 0) symmetrise<G, LD>(g, T, X);
    }
    if (P.binfo) store_state<G, LD>(g, T, X, P.binfo + (series * P.K + k) * (int64_t)ss);
    if (k == k0) break;
    if (!META_KIND(meta_nx)) { // request event k-1's record now: it arrives during the step below
      const double* kb = P.kbuf + (series * P.N + ob_nx) * (int64_t)ks;
      if (g.gl < n) { kv_r = kb[g.gl]; pv_r = kb[n + g.gl]; }
      S_r = kb[2 * n]; v_r = kb[2 * n + 1]; m_r = kb[2 * n + 2]; dlb_r = P.delta[k - 1];
    }
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    sandwich_Ft<G, LD>(g, T, rec, tz, X, Tm);
  }
}

struct QueryDev {
  Tab T;
  const double* p0;  // [n][n] prior covariance blkdiag(Pinf, 0) in block units (Eq. 3.19, reading R6)
  const double* discq; // [2M][stride]
  const int64_t* kp;   // [M]
  const uint32_t* meta;
  const double* fstate;
  const double* binfo;
  const double* amp;
  int64_t K, Mq, batch; // Mq: queries of this slice
  int64_t Mtot, q0;     // the outputs are [batch][Mtot]; the slice starts at query q0
  int qinst;
  double* mean; // [batch][M]
  double* var;
  int* flags;
};

__host__ __device__ inline int query_group_doubles(int n, int ld, int stride, int nblk, int G) {
  return (3 * (ld - 1) * ld + 2 * stride + 2 + nblk * G + 2 * ld + 1 + 1) & ~1;
}

template <int G, int LD>
__device__ __forceinline__ void query_body(const QueryDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  constexpr int ld = LD;
  const int n = TN;
  const size_t tb = 0;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.Mq) return;
  double* base = (double*)(smem + tb) + (size_t)(threadIdx.x / G) * query_group_doubles(n, LD, TSTRIDE, TNB, G);
  double* X = base;                 // [P* | m*]
  constexpr int NR = LD - 1;
  double* Tm = X + NR * ld;
  double* Y = Tm + NR * ld;         // [Lambda* | lambda*]
  double* recs = Y + NR * ld;
  double* U = recs + 2 * TSTRIDE + 2 + g.gl;
  double* hv = recs + 2 * TSTRIDE + 2 + TNB * G; // n: H_q in block units
  double* ph = hv + ld;                           // n: P* h
  const int ss = state_size(n);
  const int64_t series = gid / P.Mq, q = gid - series * P.Mq;
  const int64_t kp = P.kp[q];
  const double ampv = P.amp ? P.amp[series] : 1.0;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);
  RecStage rs;
  rs.init(g, recs, TSTRIDE);
  rs.issue(g, P.discq + q * (int64_t)TSTRIDE, 0);
  rs.issue(g, P.discq + (P.Mq + q) * (int64_t)TSTRIDE, 1);
  for (int i = g.gl; i < n; i += G) hv[i] = 0.0;
  g.sync();
  if (g.gl == 0)
    for (int b = 0; b < TNB; ++b) hv[TBOFF(b)] = ((P.T.bmask[b] >> P.qinst) & 1u) ? P.T.bsig[b] : 0.0; // H of the queried (virtual) instrument
  rs.wait(0);
  rs.wait(1);
  g.sync();
  // ---- state just after the last event at or before t*, predicted over Delta_1 (Eq. 3.14) ----
  if (kp >= 0) {
    load_state<G, LD>(g, T, P.fstate + (series * P.K + kp) * (int64_t)ss, X);
    g.sync();
    const uint32_t mp = P.meta[kp]; // idle through (t_kp, t_kp+1): zeroed after kp, except an instrument that just started
    const unsigned idle = META_KIND(mp) ? (META_ZMASK(mp) & ~(1u << META_INST(mp))) : META_ZMASK(mp);
    sandwich_F<G, LD, true>(g, T, recs, idle, X, Tm, U);
  } else { // before the first event: the stationary prior, idle z = 0 (retrodiction, reading R8)
    for (int j = g.gl; j <= n; j += G)
      for (int i = 0; i < n; ++i) X[i * ld + j] = (j < n) ? P.p0[i * n + j] : 0.0;
    g.sync();
  }
  // ---- adjoint at t*: the pre-update adjoint of the next event stepped back over Delta_2 ----
  const bool have_next = kp + 1 < P.K;
  if (have_next) {
    const int64_t kn = kp + 1;
    load_state<G, LD>(g, T, P.binfo + (series * P.K + kn) * (int64_t)ss, Y);
    g.sync();
    const uint32_t meta = P.meta[kn];
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = META_KIND(meta) ? zm : (zm & ~(1u << META_INST(meta)));
    sandwich_Ft<G, LD>(g, T, recs + TSTRIDE, tz, Y, Tm);
  }
  // ---- m^ = m* - P* lambda*,  P^ = P* - P* Lambda* P*, projected on H_q ----
  for (int j = g.gl; j < n; j += G) {
    double a = 0.0;
    for (int l = 0; l < n; ++l) a = fma(X[l * ld + j], hv[l], a);
    ph[j] = a;
  }
  g.sync();
  double sm = 0.0, sv = 0.0;
  for (int j = g.gl; j <= n; j += G) {
    if (j < n) {
      sm = fma(hv[j], X[j * ld + n], sm);
      sv = fma(hv[j], ph[j], sv);
    }
    if (have_next) {
      double a = 0.0;
      for (int i = 0; i < n; ++i) a = fma(Y[i * ld + j], ph[i], a);
      if (j < n) sv = fma(-ph[j], a, sv);
      else sm -= a;
    }
  }
  sm = group_sum(g, sm);
  sv = group_sum(g, sv);
  if (g.gl == 0) {
    if (!isfinite(sv) || !isfinite(sm)) atomicOr(P.flags, NUMF_BAD);
    P.mean[series * P.Mtot + P.q0 + q] = ampv * sm;
    P.var[series * P.Mtot + P.q0 + q] = ampv * ampv * sv;
  }
}


// ---------------------------------------------------------------------------------------------------
// kernel entry points: templates for the static build, fixed C names for the specialised build
// ---------------------------------------------------------------------------------------------------
#ifdef SG_JIT
#if !JT_REG /* otherwise chunk_reg.cuh provides the register-resident jit_fold0 / jit_down0 */
extern "C" __global__ void __launch_bounds__(128) jit_fold0(const __grid_constant__ ScanDev P) { fold0_body<JT_G, JT_LD>(P); }
extern "C" __global__ void __launch_bounds__(128) jit_down0(const __grid_constant__ ScanDev P) { down0_body<JT_G, JT_LD>(P); }
#endif
extern "C" __global__ void __launch_bounds__(128) jit_query(const __grid_constant__ QueryDev P) { query_body<JT_G, JT_LD>(P); }
#else
template <int G, int LD>
__global__ void __launch_bounds__(128) k_fold0(const __grid_constant__ ScanDev P) { fold0_body<G, LD>(P); }
template <int G, int LD>
__global__ void __launch_bounds__(128) k_down0(const __grid_constant__ ScanDev P) { down0_body<G, LD>(P); }
template <int G, int LD>
__global__ void __launch_bounds__(128) k_query(const __grid_constant__ QueryDev P) { query_body<G, LD>(P); }
#endif
