// chunk_reg.cuh -- REGISTER-RESIDENT per-chunk kernels (k_fold0 / k_down0 of the run-time specialised build).
//
// Same arithmetic and the same column ownership as chunk_kernels.cuh (a lane owns whole columns of
// [P | m], [Lambda | lambda], [A | b], C, [J | eta], so a product with the transition needs no cross-lane
// reduction), but every matrix entry lives in a REGISTER: lane gl of a group of G lanes owns the CPL
// columns gl, gl + G, gl + 2G (column n is the companion vector), held as double X[CPL][n] with
// compile-time indices only -- possible because the specialised build knows n, the block structure and
// (G, CPL) as constants.  What is left in shared memory is what has to cross lanes:
//   * the step's discretisation record (TMA bulk copy, two buffers; read with 128-bit broadcast loads,
//     once for all CPL columns of a lane);
//   * ONE transposed exchange per sandwich: F X F^T = F (F X)^T for a symmetric X, so lane j needs row
//     j of T = F X -- T's columns are written to a padded buffer (odd row stride: conflict-free both
//     ways) and read back as rows;
//   * the vectors of an end event (z-column of P, gain, ...), n + 1 doubles.
// G * CPL >= n + 1 with G in {4, 8, 16, 32}: for n = 21 a group is 8 lanes x 3 columns (22 of 24 slots
// used, four chunks per warp) instead of one lane per column on a 32-lane group (22 of 32).
// Round-1 ncu on the shared-memory version (profiles/r01_top_kernel_ncu.md): LSU pipe 48-52 %, FP64 pipe
// 21 %, 18 of 32 threads per instruction; every FMA was fed by a shared-memory load.
//
// The conversion of the reverse scan's suffix information into the adjoint at a chunk's last event
// (one solve per chunk) is done by k_adjD (dense_kernels.cuh) for this path, so the chunk kernels need
// no solve workspace at all.
#pragma once
#if defined(SG_JIT) && JT_REG

#define RN JT_N
#define RD JT_D
#define RLDT ((JT_N + 2) | 1)                     /* odd row stride of the exchange buffer, >= n + 2 columns (one spare): reg_ldt(n) */
#define RTM ((((JT_N * RLDT) + 7) / 16) * 16 + 8) /* its size: reg_tm(n) */
#define RVB (2 * (JT_N + 2))                      /* one vector buffer, (n + 1) pairs: reg_vb(n) */
#define SG_REG_FENCE asm volatile("" ::: "memory")
#ifndef SG_SYM_MASK
#define SG_SYM_MASK 31 /* the state is re-symmetrised every SG_SYM_MASK + 1 events (measured: 8, 32, 128 or never give the same accuracy on configs 3 and 4) */
#endif

// ---- record staging for these kernels: every lane of the group copies 16-byte pieces with cp.async (LDGSTS) ------------
// The TMA bulk copy of chunk_dev.cuh (RecStage) is issued by one elected lane through the uniform datapath and waited
// for on an mbarrier: per event that cost ~600 cycles of this latency-bound stream (clock64: "wait + sync" 263, issue
// and prefetch 339); a record is only 1.5 KB, so three cp.async per lane do the same with less ceremony.
#ifndef SG_REC_CP
#define SG_REC_CP 1
#endif
struct RecCp {
  double* buf;
  template <int G>
  __device__ __forceinline__ void init(const Grp<G>&, double* recs, int) { buf = recs; }
  template <int G>
  __device__ __forceinline__ void issue(const Grp<G>& g, const double* __restrict__ src, int b) {
    double* dst = buf + b * JT_STRIDE;
#pragma unroll
    for (int o = 2 * g.gl; o < JT_STRIDE; o += 2 * G)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(dst + o)), "l"(src + o) : "memory");
    asm volatile("cp.async.commit_group;\n" ::: "memory");
  }
  __device__ __forceinline__ const double* wait(int b) {
    asm volatile("cp.async.wait_group 0;\n" ::: "memory");
    return buf + b * JT_STRIDE; // the caller's group barrier makes the other lanes' pieces visible
  }
};
#if SG_REC_CP
typedef RecCp RegRecStage;
#else
typedef RecStage RegRecStage;
#endif

// ---- blocks of the transition on register columns -------------------------------------------------------
// v[s][.] <- F v[s][.] for the slots S0 <= s < S1 of v (in place)
template <int B, int NS, int S0, int S1>
__device__ __forceinline__ void rF_blocks(const double* rec, double (&v)[NS][RN], double (&u)[NS][JT_NB]) {
  if constexpr (B < JT_NB) {
    constexpr int DB = jt_bdim(B), OFF = jt_boff(B), RO = jt_roff(B);
    double m[DB * DB + DB];
    load_block<DB>(rec + RO, m);
#pragma unroll
    for (int s = S0; s < S1; ++s) {
      double w[DB];
#pragma unroll
      for (int l = 0; l < DB; ++l) w[l] = v[s][OFF + l];
#pragma unroll
      for (int i = 0; i < DB; ++i) {
        double acc = m[i * DB] * w[0];
#pragma unroll
        for (int l = 1; l < DB; ++l) acc = fma(m[i * DB + l], w[l], acc);
        v[s][OFF + i] = acc;
      }
      double uu = m[DB * DB] * w[0];
#pragma unroll
      for (int l = 1; l < DB; ++l) uu = fma(m[DB * DB + l], w[l], uu); // Phi-bar_b . v_b
      u[s][B] = uu;
    }
    SG_REG_FENCE; // keeps the next block's record loads from being hoisted above this block (register pressure)
    rF_blocks<B + 1, NS, S0, S1>(rec, v, u);
  }
}

template <int NS, int S0, int S1>
__device__ __forceinline__ void r_apply_F(const Tab& T, const double* rec, unsigned tz, double (&v)[NS][RN]) {
  double u[NS][JT_NB];
  rF_blocks<0, NS, S0, S1>(rec, v, u);
#pragma unroll
  for (int q = 0; q < JT_NI; ++q) {
    const bool zq = (tz >> q) & 1u;
#pragma unroll
    for (int s = S0; s < S1; ++s) {
      double acc = v[s][RD + q];
#pragma unroll
      for (int b = 0; b < JT_NB; ++b)
        if (jt_czmask(q * JT_NB + b)) acc = fma(T.cz[q * JT_NB + b], u[s][b], acc);
      v[s][RD + q] = zq ? 0.0 : acc;
    }
  }
}

// v[s][.] <- F^T v[s][.]
template <int B, int NS>
__device__ __forceinline__ void rFt_blocks(const Tab& T, const double* rec, unsigned tz, double (&v)[NS][RN]) {
  if constexpr (B < JT_NB) {
    constexpr int DB = jt_bdim(B), OFF = jt_boff(B), RO = jt_roff(B);
    double m[DB * DB + DB];
    load_block<DB>(rec + RO, m);
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      double sz = 0.0; // sum_q c_qb v_zq over the instruments that are not zeroed
#pragma unroll
      for (int q = 0; q < JT_NI; ++q)
        if (jt_czmask(q * JT_NB + B)) sz = fma(((tz >> q) & 1u) ? 0.0 : T.cz[q * JT_NB + B], v[s][RD + q], sz);
      double w[DB];
#pragma unroll
      for (int i = 0; i < DB; ++i) w[i] = v[s][OFF + i];
#pragma unroll
      for (int l = 0; l < DB; ++l) {
        double acc = m[DB * DB + l] * sz;
#pragma unroll
        for (int i = 0; i < DB; ++i) acc = fma(m[i * DB + l], w[i], acc);
        v[s][OFF + l] = acc;
      }
    }
    SG_REG_FENCE;
    rFt_blocks<B + 1, NS>(T, rec, tz, v);
  }
}
template <int NS>
__device__ __forceinline__ void r_apply_Ft(const Tab& T, const double* rec, unsigned tz, double (&v)[NS][RN]) {
  rFt_blocks<0, NS>(T, rec, tz, v);
#pragma unroll
  for (int q = 0; q < JT_NI; ++q)
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if ((tz >> q) & 1u) v[s][RD + q] = 0.0;
}

// ---- what a lane knows about its columns (fixed for the whole kernel) -----------------------------------
template <int G, int CPL>
struct Cols {
  int jc[CPL];      // column index of slot c: gl + c G
  int rbase[CPL];   // exchange read: row jc of the buffer for a matrix column (row 0, unused, otherwise)
  int myblk[CPL];   // block of an x column, -1 otherwise
  int qoff[CPL];    // record offset of column (jc - off_b) of the block's Q_xx; row stride qst
  int qst[CPL];
  int q12off[CPL];  // record offset of q12[jc - off_b]
  int wcol[CPL];    // exchange write: column jc of the buffer (the spare column n + 1 for a lane without a column)
  int vidx[CPL];    // entry of this column in an end event's vector buffers (the spare entry n + 1 without a column)
  int c0base[CPL];  // row of the shared coupling table for a z column (jc = d + q: q NB), the all-zero row otherwise
  int zq[CPL];      // q of a z column, 0 otherwise
  double czown[CPL][JT_NI]; // c_qb of the column's own block b for every instrument q (0 for a column that is not an x column)
  unsigned comp;    // bit c: slot c is the companion column n
  unsigned xcol;    // bit c: jc < n (a matrix column)
  __device__ __forceinline__ void init(int gl, const double* czs) {
    comp = 0u; xcol = 0u;
#pragma unroll
    for (int c = 0; c < CPL; ++c) {
      const int j = gl + c * G;
      jc[c] = j;
      if (j == RN) comp |= 1u << c;
      if (j < RN) xcol |= 1u << c;
      rbase[c] = (j < RN) ? j * RLDT : 0;
      wcol[c] = (j <= RN) ? j : RN + 1;
      vidx[c] = (j <= RN) ? j : RN + 1;
      const bool isz = j >= RD && j < RN;
      zq[c] = isz ? j - RD : 0;
      c0base[c] = isz ? (j - RD) * JT_NB : JT_NI * JT_NB;
      int mb = -1, qo = 0, qs = 1, q12 = 0;
#pragma unroll
      for (int b = 0; b < JT_NB; ++b) {
        const int db = jt_bdim(b), off = jt_boff(b), ro = jt_roff(b), jj = j - off;
        if (jj >= 0 && jj < db) { mb = b; qo = ro + db * db + db + jj; qs = db; q12 = ro + 2 * db * db + db + jj; }
      }
      myblk[c] = mb; qoff[c] = qo; qst[c] = qs; q12off[c] = q12;
#pragma unroll
      for (int q = 0; q < JT_NI; ++q) czown[c][q] = (mb >= 0) ? czs[q * JT_NB + mb] : 0.0;
    }
  }
};

// can slot c hold a z column / the companion for SOME lane?  (compile-time: the code for it is only emitted there)
template <int G>
__host__ __device__ constexpr bool slot_has_z(int c) { return c * G < RN && c * G + G > RD; }
template <int G>
__host__ __device__ constexpr bool slot_has_comp(int c) { return c * G <= RN && c * G + G > RN; }

// X[c][RD + q] with a run-time q (q < JT_NI): a select chain over compile-time register indices
__device__ __forceinline__ double get_z(const double (&x)[RN], int q) {
  double r = x[RD];
#pragma unroll
  for (int p = 1; p < JT_NI; ++p) r = (q == p) ? x[RD + p] : r;
  return r;
}
__device__ __forceinline__ void set_z(double (&x)[RN], int q, double val) {
#pragma unroll
  for (int p = 0; p < JT_NI; ++p) x[RD + p] = (q == p) ? val : x[RD + p];
}
__device__ __forceinline__ void add_z(double (&x)[RN], int q, double val) {
#pragma unroll
  for (int p = 0; p < JT_NI; ++p) x[RD + p] = (q == p) ? x[RD + p] + val : x[RD + p];
}

// exchange: the slots S0..S1-1 of v hold COLUMNS of a matrix T; on return the matrix slots hold the ROWS of the same
// index (the companion slot: see r_companion_back).  Two group barriers.
template <int G, int CPL, int NS, int S0>
__device__ __forceinline__ void r_exchange(const Grp<G>& g, const Cols<G, CPL>& cl, double* __restrict__ Tm, double (&v)[NS][RN]) {
  // no lane-dependent branch anywhere (a divergent branch serialises the warp behind a reconvergence barrier:
  // measured 4x on these few lines): a lane without a column writes the buffer's spare column
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
#pragma unroll
    for (int i = 0; i < RN; ++i) Tm[i * RLDT + cl.wcol[c]] = v[S0 + c][i];
  }
  g.sync();
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
#pragma unroll
    for (int l = 0; l < RN; ++l) v[S0 + c][l] = Tm[cl.rbase[c] + l];
  }
  g.sync();
}

// the companion column is not part of the second product of a sandwich: its slot gets back the column it wrote
// into the exchange buffer (no barrier needed: a lane re-reads its own stores)
template <int G, int CPL, int NS, int S0>
__device__ __forceinline__ void r_companion_back(const Cols<G, CPL>& cl, const double* __restrict__ Tm, double (&v)[NS][RN]) {
#pragma unroll
  for (int c = 0; c < CPL; ++c)
    if (slot_has_comp<G>(c)) { // compile-time
      const bool isc = (cl.comp >> c) & 1u;
#pragma unroll
      for (int i = 0; i < RN; ++i) {
        const double r = Tm[i * RLDT + RN]; // one address for the whole group: a broadcast
        v[S0 + c][i] = isc ? r : v[S0 + c][i];
      }
    }
}

// X <- (X + X^T) / 2 on the matrix columns of the slots S0.. (periodic: the two triangles are rounded independently)
template <int G, int CPL, int NS, int S0>
__device__ __forceinline__ void r_symmetrise(const Grp<G>& g, const Cols<G, CPL>& cl, double* __restrict__ Tm, double (&v)[NS][RN]) {
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
#pragma unroll
    for (int i = 0; i < RN; ++i) Tm[i * RLDT + cl.wcol[c]] = v[S0 + c][i]; // (the companion's column n is never read back)
  }
  g.sync();
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
    const bool isx = (cl.xcol >> c) & 1u;
    const int rb = cl.rbase[c];
#pragma unroll
    for (int l = 0; l < RN; ++l) {
      const double r = Tm[rb + l];
      v[S0 + c][l] = isx ? 0.5 * (v[S0 + c][l] + r) : v[S0 + c][l];
    }
  }
  g.sync();
}

// column jc of X += column jc of Q = R Q~ R^T (Eq. 3.10 P:403-405 per block; z rows / columns through c_qb).  Branch-free:
// what depends on the lane's column (its block, whether it is a z column) enters as 0 / 1 factors and per-lane
// table rows, never as a divergent branch.
template <int B>
__device__ __forceinline__ void rQ_xrows(int myblk, const double (&qv)[SG_MAXBD], double (&x)[RN]) {
  if constexpr (B < JT_NB) {
    constexpr int DB = jt_bdim(B), OFF = jt_boff(B);
    const double ind = (myblk == B) ? 1.0 : 0.0;
#pragma unroll
    for (int i = 0; i < DB; ++i) x[OFF + i] = fma(qv[i], ind, x[OFF + i]);
    rQ_xrows<B + 1>(myblk, qv, x);
  }
}
template <int B>
__device__ __forceinline__ void rQ_zcol(const Tab& T, const double* rec, const double* __restrict__ c0row, double keep, unsigned tz, double (&x)[RN]) {
  if constexpr (B < JT_NB) {
    constexpr int DB = jt_bdim(B), OFF = jt_boff(B), RO = jt_roff(B);
    const double c0 = c0row[B] * keep; // c_{q0 b} for the lane's z column q0 (0 for any other column, or when q0 is zeroed)
#pragma unroll
    for (int l = 0; l < DB; ++l) x[OFF + l] = fma(c0, rec[RO + 2 * DB * DB + DB + l], x[OFF + l]);
    const double q22 = rec[RO + 2 * DB * DB + 2 * DB];
#pragma unroll
    for (int p = 0; p < JT_NI; ++p)
      if (jt_czmask(p * JT_NB + B)) x[RD + p] = fma(((tz >> p) & 1u) ? 0.0 : c0 * T.cz[p * JT_NB + B], q22, x[RD + p]);
    rQ_zcol<B + 1>(T, rec, c0row, keep, tz, x);
  }
}
template <int G, int CPL, int NS, int S0>
__device__ __forceinline__ void r_add_Q(const Tab& T, const Cols<G, CPL>& cl, const double* rec, const double* __restrict__ czs, unsigned tz,
                                        double (&v)[NS][RN]) {
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
    double qv[SG_MAXBD];
#pragma unroll
    for (int i = 0; i < SG_MAXBD; ++i) qv[i] = rec[cl.qoff[c] + i * cl.qst[c]];
    const double q12 = rec[cl.q12off[c]];
    rQ_xrows<0>(cl.myblk[c], qv, v[S0 + c]);
#pragma unroll
    for (int q = 0; q < JT_NI; ++q) v[S0 + c][RD + q] = fma(((tz >> q) & 1u) ? 0.0 : cl.czown[c][q], q12, v[S0 + c][RD + q]);
    if (slot_has_z<G>(c)) { // compile-time: only the slots that hold a z column on some lane
      const double keep = ((tz >> cl.zq[c]) & 1u) ? 0.0 : 1.0;
      rQ_zcol<0>(T, rec, czs + cl.c0base[c], keep, tz, v[S0 + c]);
    }
  }
}

// X <- F X F^T (+ Q), x <- F x on the slots S0..S0+CPL-1
#ifdef SG_CHUNK_CLK /* debugging aid (SMOLGP_JIT_DEFS): cycles per phase of the forward sandwich, accumulated per chunk */
#define SG_CCK(i) do { const long long t_ = clock64(); sg_cck[i] += t_ - sg_ct; sg_ct = t_; } while (0)
#define SG_CCK_ARGS , long long (&sg_cck)[12], long long& sg_ct
#define SG_CCK_PASS , sg_cck, sg_ct
#else
#define SG_CCK(i) do {} while (0)
#define SG_CCK_ARGS
#define SG_CCK_PASS
#endif
template <int G, int CPL, int NS, int S0, bool ADDQ>
__device__ __forceinline__ void r_sandwich_F(const Grp<G>& g, const Tab& T, const Cols<G, CPL>& cl, const double* rec,
                                             const double* __restrict__ czs, unsigned tz, double* __restrict__ Tm, double (&v)[NS][RN] SG_CCK_ARGS) {
  r_apply_F<NS, S0, S0 + CPL>(T, rec, tz, v);
  SG_CCK(1);
  r_exchange<G, CPL, NS, S0>(g, cl, Tm, v);
  SG_CCK(2);
  r_apply_F<NS, S0, S0 + CPL>(T, rec, tz, v);
  SG_CCK(3);
  r_companion_back<G, CPL, NS, S0>(cl, Tm, v);
  if (ADDQ) r_add_Q<G, CPL, NS, S0>(T, cl, rec, czs, tz, v);
  SG_CCK(4);
}
template <int G, int CPL>
__device__ __forceinline__ void r_sandwich_Ft(const Grp<G>& g, const Tab& T, const Cols<G, CPL>& cl, const double* rec, unsigned tz,
                                              double* __restrict__ Tm, double (&v)[CPL][RN]) {
  r_apply_Ft<CPL>(T, rec, tz, v);
  r_exchange<G, CPL, CPL, 0>(g, cl, Tm, v);
  r_apply_Ft<CPL>(T, rec, tz, v);
  r_companion_back<G, CPL, CPL, 0>(cl, Tm, v);
}

// carve one group's shared memory
struct RegSmem {
  double* Tm;
  double* recs;
  double* vb0;
  double* vb1;
  double* vb2;
  __device__ __forceinline__ RegSmem(double* base) {
    recs = base;                        // 2 x stride + 2 mbarriers: first, 16-byte aligned
    Tm = base + 2 * JT_STRIDE + 2;
    vb0 = Tm + RTM;
    vb1 = vb0 + RVB;
    vb2 = vb1 + RVB;
  }
};

// ---------------------------------------------------------------------------------------------------
// k_fold0, register-resident: chunk -> element (A, b, C, eta, J).  State slots: [0, CPL) = [A | b],
// [CPL, 2 CPL) = C, [2 CPL, 3 CPL) = [J | eta].
// ---------------------------------------------------------------------------------------------------
template <int G, int CPL>
__device__ __forceinline__ void reg_fold0_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  double* czs = (double*)smem; // [(NI + 1) x NB] couplings, read with lane-dependent indices; the last row is zero
  for (int e = threadIdx.x; e < (JT_NI + 1) * JT_NB; e += blockDim.x) czs[e] = (e < JT_NI * JT_NB) ? T.cz[e] : 0.0;
  __syncthreads();
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  constexpr int CZS = ((JT_NI + 1) * JT_NB + 1) & ~1; // reg_czs
  RegSmem sm((double*)smem + CZS + (size_t)(threadIdx.x / G) * reg_group_doubles(JT_N, JT_STRIDE));
  Cols<G, CPL> cl;
  cl.init(g.gl, czs);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ramp = P.amp ? 1.0 / P.amp[series] : 1.0;
  constexpr int NS = 3 * CPL;
  double S[NS][RN];
#pragma unroll
  for (int s = 0; s < NS; ++s)
#pragma unroll
    for (int i = 0; i < RN; ++i) S[s][i] = 0.0;
#pragma unroll
  for (int c = 0; c < CPL; ++c)
#pragma unroll
    for (int i = 0; i < RN; ++i) S[c][i] = (cl.jc[c] == i) ? 1.0 : 0.0;

  RegRecStage rs;
  rs.init(g, sm.recs, JT_STRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)JT_STRIDE, 0);
  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const double* rec = rs.wait((int)((k - k0) & 1));
    g.sync();
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)JT_STRIDE, (int)((k + 1 - k0) & 1));
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    // [A | b] <- F [A | b] and T = F C with ONE pass over the record; then C <- F T^T + Q
    r_apply_F<NS, 0, 2 * CPL>(T, rec, tz, S);
    r_exchange<G, CPL, NS, CPL>(g, cl, sm.Tm, S);
    r_apply_F<NS, CPL, 2 * CPL>(T, rec, tz, S);
    r_add_Q<G, CPL, NS, CPL>(T, cl, rec, czs, tz, S);
#pragma unroll
    for (int c = 0; c < CPL; ++c) // column n of C is not part of the element: keep it zero
      if (!((cl.xcol >> c) & 1u)) {
#pragma unroll
        for (int i = 0; i < RN; ++i) S[CPL + c][i] = 0.0;
      }
    if (!kind) {
      // observe z_q / delta: h = hs e_z (Eq. 3.12); SG21 Eq. 10 with the aggregate as the earlier element
      // (rank-one J_j): Sherman-Morrison form of the combine.  a = hs A[z, :], c = hs C[:, z] (= hs C[z, :]).
      const int zi = RD + q;
      const double hs = T.tau[q] / dl_r;
      const double sg = sg_r * ramp, yy = y_r * ramp;
      double2* avcv = reinterpret_cast<double2*>(sm.vb0);
      double av_o[CPL], cv_o[CPL];
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        av_o[c] = hs * get_z(S[c], q);
        cv_o[c] = hs * get_z(S[CPL + c], q);
        avcv[cl.vidx[c]] = make_double2(av_o[c], cv_o[c]);
      }
      g.sync();
      const double Sv = hs * avcv[zi].y + sg * sg;
      if (!(Sv > 0.0) || !isfinite(Sv)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / Sv;
      const double resid = yy - avcv[RN].x;
      double aj[CPL], caj[CPL], cj[CPL];
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        const bool isx = (cl.xcol >> c) & 1u, isc = (cl.comp >> c) & 1u;
        aj[c] = isx ? av_o[c] * rS : (isc ? resid * rS : 0.0);
        caj[c] = isx ? -aj[c] : aj[c];
        cj[c] = isx ? -cv_o[c] * rS : 0.0;
      }
#pragma unroll
      for (int i = 0; i < RN; ++i) {
        const double2 ac = avcv[i];
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
          S[2 * CPL + c][i] = fma(ac.x, aj[c], S[2 * CPL + c][i]); // J += a a_j / S;  eta += a resid / S
          S[c][i] = fma(ac.y, caj[c], S[c][i]);                     // A -= c a_j / S;  b += c resid / S
          S[CPL + c][i] = fma(ac.y, cj[c], S[CPL + c][i]);          // C -= c c_j / S
        }
      }
      // the instrument is idle after its end: zero z_q (reading R6)
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        set_z(S[c], q, 0.0);
        set_z(S[CPL + c], q, 0.0);
        if (slot_has_z<G>(c)) {
          const bool kz = cl.jc[c] == zi;
#pragma unroll
          for (int i = 0; i < RN; ++i) S[CPL + c][i] = kz ? 0.0 : S[CPL + c][i];
        }
      }
      g.sync();
    }
  }
  // element out: AB [n x (n+1)] = [A | b],  C [n x n] (symmetrised),  JE [n x (n+1)] = [J | eta]
  r_symmetrise<G, CPL, NS, CPL>(g, cl, sm.Tm, S);
  double* out = P.E1 + gid * (int64_t)elem_size(RN);
  constexpr int n1 = RN + 1;
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
    const int j = cl.jc[c];
    if (j <= RN) {
#pragma unroll
      for (int i = 0; i < RN; ++i) {
        out[i * n1 + j] = S[c][i];
        out[RN * n1 + RN * RN + i * n1 + j] = S[2 * CPL + c][i];
      }
    }
    if (j < RN) {
#pragma unroll
      for (int i = 0; i < RN; ++i) out[RN * n1 + j * RN + i] = S[CPL + c][i]; // row j = column j (symmetric): contiguous
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// k_down0, register-resident: the chunk's Kalman filter from its prefix state (loglik terms, kbuf), then
// the adjoint recursion from ADJ1 (the chunk's last-event adjoint, k_adjD) with the smoothed outputs.
// ---------------------------------------------------------------------------------------------------
template <int G, int CPL>
__device__ __forceinline__ void reg_store_state(const Cols<G, CPL>& cl, const double (&X)[CPL][RN], double* __restrict__ s) {
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
    const int j = cl.jc[c];
#pragma unroll
    for (int i = 0; i < RN; ++i) {
      if (j < RN) s[RN + j * RN + i] = X[c][i]; // row j of the (symmetric up to rounding) matrix: contiguous
      else if (j == RN) s[i] = X[c][i];
    }
  }
}
template <int G, int CPL>
__device__ __forceinline__ void reg_load_state(const Cols<G, CPL>& cl, const double* __restrict__ s, double (&X)[CPL][RN]) {
#pragma unroll
  for (int c = 0; c < CPL; ++c) {
    const int j = cl.jc[c];
#pragma unroll
    for (int i = 0; i < RN; ++i) X[c][i] = (j < RN) ? s[RN + j * RN + i] : ((j == RN) ? s[i] : 0.0);
  }
}

template <int G, int CPL>
__device__ __forceinline__ void reg_down0_body(const ScanDev& P) {
  extern __shared__ __align__(16) char smem[];
  const Tab& T = P.T;
  const Grp<G> g;
  const int gpc = blockDim.x / G;
  double* czs = (double*)smem;
  for (int e = threadIdx.x; e < (JT_NI + 1) * JT_NB; e += blockDim.x) czs[e] = (e < JT_NI * JT_NB) ? T.cz[e] : 0.0;
  __syncthreads();
  const int64_t gid = (int64_t)blockIdx.x * gpc + threadIdx.x / G;
  if (gid >= P.batch * P.c1) return;
  constexpr int CZS = ((JT_NI + 1) * JT_NB + 1) & ~1; // reg_czs
  RegSmem sm((double*)smem + CZS + (size_t)(threadIdx.x / G) * reg_group_doubles(JT_N, JT_STRIDE));
  Cols<G, CPL> cl;
  cl.init(g.gl, czs);
  const int ss = state_size(RN), ks = kbuf_stride(RN);
  const int64_t series = gid / P.c1, chunk = gid - series * P.c1;
  const int64_t k0 = chunk * P.Lc, k1 = (k0 + P.Lc < P.K) ? k0 + P.Lc : P.K;
  const double ampv = P.amp ? P.amp[series] : 1.0;
  const double ramp = 1.0 / ampv;
  if (!(ampv > 0.0) || !isfinite(ampv)) atomicOr(P.flags, NUMF_AMP);

  double X[CPL][RN];
  if (P.PRE1) reg_load_state<G, CPL>(cl, P.PRE1 + gid * (int64_t)ss, X);
  else {
#pragma unroll
    for (int c = 0; c < CPL; ++c)
#pragma unroll
      for (int i = 0; i < RN; ++i) X[c][i] = (cl.jc[c] < RN) ? P.p0[cl.jc[c] * RN + i] : 0.0;
  }
  RegRecStage rs;
  rs.init(g, sm.recs, JT_STRIDE);
  rs.issue(g, P.disc + k0 * (int64_t)JT_STRIDE, 0);
  double ll = 0.0;
#ifdef SG_CHUNK_CLK
  long long sg_cck[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  long long sg_ct = clock64();
#endif
  // ---- forward ----
  uint32_t meta_nx = P.meta[k0];
  int32_t ob_nx = P.obs[k0];
  for (int64_t k = k0; k < k1; ++k) {
    const int it = (int)(k - k0);
    const double* rec = rs.wait(it & 1);
    g.sync();
    SG_CCK(0);
    if (k + 1 < k1) rs.issue(g, P.disc + (k + 1) * (int64_t)JT_STRIDE, (it + 1) & 1);
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    if (k + 1 < k1) { meta_nx = P.meta[k + 1]; ob_nx = P.obs[k + 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    double dl_r = 1.0, sg_r = 0.0, y_r = 0.0;
    if (!kind) { dl_r = P.delta[k]; sg_r = P.sigma[ob]; y_r = P.y[series * P.N + ob]; }
    SG_CCK(5);
    r_sandwich_F<G, CPL, CPL, 0, true>(g, T, cl, rec, czs, tz, sm.Tm, X SG_CCK_PASS);
    if (!kind) {
      const int zi = RD + q;
      const double hs = T.tau[q] / dl_r;
      const double sg = sg_r * ramp, yy = y_r * ramp;
      double* cvb = sm.vb0;
      double xz[CPL];
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        xz[c] = hs * get_z(X[c], q); // hs P[z, j] = hs P[j, z];  companion: hs m_z
        cvb[cl.vidx[c]] = xz[c];
      }
      g.sync();
      const double Sv = hs * cvb[zi] + sg * sg;
      const double v = yy - cvb[RN];
      if (!(sg_r > 0.0) || !isfinite(sg_r)) atomicOr(P.flags, NUMF_SIGMA);
      if (!(Sv > 0.0) || !isfinite(Sv) || !isfinite(v)) atomicOr(P.flags, NUMF_BAD);
      const double rS = 1.0 / Sv;
      ll -= 0.5 * (log(6.283185307179586476925286766559 * Sv) + v * v * rS);
      double cj[CPL];
#pragma unroll
      for (int c = 0; c < CPL; ++c) cj[c] = ((cl.xcol >> c) & 1u) ? -xz[c] * rS : (((cl.comp >> c) & 1u) ? v * rS : 0.0);
#pragma unroll
      for (int i = 0; i < RN; ++i) {
        const double ci = cvb[i];
#pragma unroll
        for (int c = 0; c < CPL; ++c) X[c][i] = fma(ci, cj[c], X[c][i]);
      }
      if (P.want_smooth) {
        double* kb = P.kbuf + (series * P.N + ob) * (int64_t)ks;
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
          const int j = cl.jc[c];
          const double pz = get_z(X[c], q); // filtered P[z, j] (m_z for the companion)
          if (j < RN) { kb[j] = xz[c] * rS; kb[RN + j] = pz; }
          else if (j == RN) { kb[2 * RN] = Sv; kb[2 * RN + 1] = v; kb[2 * RN + 2] = pz; }
        }
      }
      // the instrument is idle after its end (reading R6)
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        set_z(X[c], q, 0.0);
        if (slot_has_z<G>(c)) {
          const bool kz = cl.jc[c] == zi;
#pragma unroll
          for (int i = 0; i < RN; ++i) X[c][i] = kz ? 0.0 : X[c][i];
        }
      }
      g.sync();
    }
    SG_CCK(6);
    // the two triangles of F P F^T are rounded independently: re-symmetrised every 8th event
    if ((it & SG_SYM_MASK) == SG_SYM_MASK) r_symmetrise<G, CPL, CPL, 0>(g, cl, sm.Tm, X);
    SG_CCK(7);
    if (P.fstate) reg_store_state<G, CPL>(cl, X, P.fstate + (series * P.K + k) * (int64_t)ss); // row a7
  }
  if (g.gl == 0) P.llpart[gid] = ll;
#ifdef SG_CHUNK_CLK
  if (gid == 5 && g.gl == 0) {
    const long long ne = k1 - k0;
    printf("down0 fwd cycles/event: wait+sync %lld | meta etc %lld | F1 %lld | exchange %lld | F2 %lld | comp+Q %lld | end-event %lld | sym %lld\n", sg_cck[0] / ne,
           sg_cck[5] / ne, sg_cck[1] / ne, sg_cck[2] / ne, sg_cck[3] / ne, sg_cck[4] / ne, sg_cck[6] / ne, sg_cck[7] / ne);
  }
#endif
  if (!P.want_smooth) return;

  // ---- adjoint at the chunk's last event (k_adjD: Lambda^ = (I + J P)^-1 J, lambda^ = (I + J P)^-1 (J m - eta)) ----
  rs.issue(g, P.disc + (k1 - 1) * (int64_t)JT_STRIDE, 0);
  if (P.ADJ1) reg_load_state<G, CPL>(cl, P.ADJ1 + gid * (int64_t)ss, X);
  else {
#pragma unroll
    for (int c = 0; c < CPL; ++c)
#pragma unroll
      for (int i = 0; i < RN; ++i) X[c][i] = 0.0;
  }
  // ---- backward ----
  meta_nx = P.meta[k1 - 1];
  ob_nx = P.obs[k1 - 1];
  double kv_r[CPL], pv_r[CPL], S_r = 1.0, v_r = 0.0, m_r = 0.0, dlb_r = 1.0;
#pragma unroll
  for (int c = 0; c < CPL; ++c) { kv_r[c] = 0.0; pv_r[c] = 0.0; }
  if (!META_KIND(meta_nx)) {
    const double* kb = P.kbuf + (series * P.N + ob_nx) * (int64_t)ks;
#pragma unroll
    for (int c = 0; c < CPL; ++c)
      if (cl.jc[c] < RN) { kv_r[c] = kb[cl.jc[c]]; pv_r[c] = kb[RN + cl.jc[c]]; }
    S_r = kb[2 * RN]; v_r = kb[2 * RN + 1]; m_r = kb[2 * RN + 2]; dlb_r = P.delta[k1 - 1];
  }
  for (int64_t k = k1 - 1; k >= k0; --k) {
    const int it = (int)(k1 - 1 - k);
    const double* rec = rs.wait(it & 1);
    g.sync();
    if (k > k0) rs.issue(g, P.disc + (k - 1) * (int64_t)JT_STRIDE, (it + 1) & 1);
    const uint32_t meta = meta_nx;
    const int32_t ob = ob_nx;
    double kv_c[CPL], pv_c[CPL];
#pragma unroll
    for (int c = 0; c < CPL; ++c) { kv_c[c] = kv_r[c]; pv_c[c] = pv_r[c]; }
    const double Sv = S_r, v = v_r, mfz = m_r, dl_c = dlb_r;
    if (k > k0) { meta_nx = P.meta[k - 1]; ob_nx = P.obs[k - 1]; }
    const int kind = META_KIND(meta), q = META_INST(meta);
    const unsigned zm = META_ZMASK(meta);
    // components zeroed after event k pass nothing backwards (adjoint of the zeroing)
#pragma unroll
    for (int r = 0; r < JT_NI; ++r)
      if ((zm >> r) & 1u) {
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
          X[c][RD + r] = 0.0;
          if (slot_has_z<G>(c)) {
            const bool kz = cl.jc[c] == RD + r;
#pragma unroll
            for (int i = 0; i < RN; ++i) X[c][i] = kz ? 0.0 : X[c][i];
          }
        }
      }
    if (!kind) {
      const int zi = RD + q;
      const double hs = T.tau[q] / dl_c;
      const double rS = 1.0 / Sv;
      double2* kp = reinterpret_cast<double2*>(sm.vb1); // (K_i, p_i) pairs
      double* gvb = sm.vb2;
#pragma unroll
      for (int c = 0; c < CPL; ++c) kp[cl.vidx[c]] = make_double2(kv_c[c], pv_c[c]); // (entries n, n + 1: never read)
      g.sync();
      double a[CPL], b[CPL];
#pragma unroll
      for (int c = 0; c < CPL; ++c) { a[c] = 0.0; b[c] = 0.0; }
#pragma unroll
      for (int i = 0; i < RN; ++i) {
        const double2 t = kp[i];
#pragma unroll
        for (int c = 0; c < CPL; ++c) { a[c] = fma(X[c][i], t.y, a[c]); b[c] = fma(X[c][i], t.x, b[c]); }
      }
      double quad = 0.0, kap = 0.0, an = 0.0;
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        const bool isx = (cl.xcol >> c) & 1u, isc = (cl.comp >> c) & 1u;
        quad += isx ? pv_c[c] * a[c] : 0.0;
        kap += isx ? kv_c[c] * b[c] : 0.0;
        an += isc ? a[c] : 0.0;
        gvb[cl.vidx[c]] = b[c];
      }
      quad = group_sum(g, quad);
      kap = group_sum(g, kap);
      an = group_sum(g, an);
      g.sync();
      if (g.gl == 0) {
        const double smv = mfz - an, sv = kp[zi].y - quad;
        if (!isfinite(sv) || !isfinite(smv)) atomicOr(P.flags, NUMF_BAD);
        P.mean[series * P.N + ob] = ampv * hs * smv;            // H~ m^
        P.var[series * P.N + ob] = ampv * ampv * hs * hs * sv;  // H~ P^ H~^T
      }
      // Lambda~ = C^T Lambda^ C + h h^T / S: only row and column z change (h = hs e_z)
#pragma unroll
      for (int c = 0; c < CPL; ++c) {
        const bool isx = (cl.xcol >> c) & 1u, isc = (cl.comp >> c) & 1u;
        const double dz = isx ? -hs * b[c] : (isc ? -hs * (b[c] + v * rS) : 0.0);
        add_z(X[c], q, dz); // row z of the lane's columns
        if (slot_has_z<G>(c)) { // column z: the lane that owns it, by a 0 / 1 factor
          const double hz = (cl.jc[c] == zi) ? hs : 0.0;
#pragma unroll
          for (int j = 0; j < RN; ++j) X[c][j] = fma(-hz, gvb[j], X[c][j]);
          add_z(X[c], q, hz * hs * (kap + rS));
        }
      }
      g.sync();
    }
    if ((it & SG_SYM_MASK) == SG_SYM_MASK) r_symmetrise<G, CPL, CPL, 0>(g, cl, sm.Tm, X);
    if (P.binfo) reg_store_state<G, CPL>(cl, X, P.binfo + (series * P.K + k) * (int64_t)ss);
    if (k == k0) break;
    if (!META_KIND(meta_nx)) { // request event k-1's record now: it arrives during the step below
      const double* kb = P.kbuf + (series * P.N + ob_nx) * (int64_t)ks;
#pragma unroll
      for (int c = 0; c < CPL; ++c)
        if (cl.jc[c] < RN) { kv_r[c] = kb[cl.jc[c]]; pv_r[c] = kb[RN + cl.jc[c]]; }
      S_r = kb[2 * RN]; v_r = kb[2 * RN + 1]; m_r = kb[2 * RN + 2]; dlb_r = P.delta[k - 1];
    }
    const unsigned tz = kind ? zm : (zm & ~(1u << q));
    r_sandwich_Ft<G, CPL>(g, T, cl, rec, tz, sm.Tm, X);
  }
}

extern "C" __global__ void __launch_bounds__(JT_FTHREADS, JT_FMINB) jit_fold0(const __grid_constant__ ScanDev P) { reg_fold0_body<JT_FG, JT_FCPL>(P); }
extern "C" __global__ void __launch_bounds__(JT_RTHREADS, JT_RMINB) jit_down0(const __grid_constant__ ScanDev P) { reg_down0_body<JT_RG, JT_RCPL>(P); }

#endif // SG_JIT && JT_REG
