// grp_dev.cuh -- lane groups and the small dense solve shared by every scan kernel.  Device code
// only, no dependencies (also part of the run-time specialised source, jit.cu).
#pragma once

template <int G>
struct Grp {
  int gl;        // lane inside the group
  unsigned mask; // the group's lanes inside the warp (G <= 32)
  __device__ __forceinline__ Grp() {
    if (G > 32) { gl = threadIdx.x; mask = 0xffffffffu; } // the group is the whole CTA (blockDim.x == G)
    else {
      const int lane = threadIdx.x & 31;
      gl = lane & (G - 1);
      mask = (G == 32) ? 0xffffffffu : (((1u << (G & 31)) - 1u) << (lane & ~(G - 1)));
    }
  }
  __device__ __forceinline__ void sync() const {
    if (G > 32) __syncthreads(); else __syncwarp(mask);
  }
};

// e -> (e / nc, e % nc) for small non-negative e (exact: see DESIGN.md "index arithmetic")
__device__ __forceinline__ void divmod_small(int e, int nc, float rnc, int& i, int& j) {
  i = __float2int_rz(((float)e + 0.5f) * rnc);
  j = e - i * nc;
}

template <int G>
__device__ __forceinline__ void zero_fill(const Grp<G>& g, double* p, int cnt) {
  for (int e = g.gl; e < cnt; e += G) p[e] = 0.0;
}

// sum over the group's lanes (G <= 32)
template <int G>
__device__ __forceinline__ double group_sum(const Grp<G>& g, double v) {
#pragma unroll
  for (int o = G / 2; o; o >>= 1) v += __shfl_xor_sync(g.mask, v, o);
  return v;
}

// Compensated dot product (Ogita-Rump-Oishi "Dot2"): the products and the running sum carry their exact
// rounding errors (one FMA and one TwoSum per term), so a sum of terms that cancel by many orders of
// magnitude is as accurate as if it had been formed in twice the working precision.  The dense levels
// multiply covariances whose large entries lie in the weakly determined directions with informations
// whose large entries lie in the strongly determined ones: the products cancel.
__device__ __forceinline__ void dot2_step(double a, double b, double& s, double& c) {
  const double p = __dmul_rn(a, b); // _rn intrinsics: never contracted into an FMA, the error terms stay exact
  const double pe = fma(a, b, -p);
  const double t = __dadd_rn(s, p);
  const double z = __dadd_rn(t, -s);
  c += __dadd_rn(__dadd_rn(__dadd_rn(s, -__dadd_rn(t, -z)), __dadd_rn(p, -z)), pe);
  s = t;
}

// Gauss-Jordan elimination with partial pivoting on the augmented matrix W = [M | R] (n rows,
// ld = n + m columns) in place; on return R holds M^-1 R.  M = I + (PSD)(PSD) in every use here
// (eigenvalues >= 1), so a zero pivot cannot occur for finite input.
template <int G>
__device__ void gj_solve(const Grp<G>& g, int n, int ld, double* W) {
  for (int p = 0; p < n; ++p) {
    // pivot search in column p, rows >= p: every lane scans the column itself (broadcast reads)
    double best = -1.0;
    int bi = p;
    for (int i = p; i < n; ++i) {
      const double v = fabs(W[i * ld + p]);
      if (v > best) { best = v; bi = i; }
    }
    g.sync(); // all lanes have read column p before the swap touches it
    if (bi != p) {
      for (int j = p + g.gl; j < ld; j += G) {
        const double a = W[p * ld + j], b = W[bi * ld + j];
        W[p * ld + j] = b;
        W[bi * ld + j] = a;
      }
    }
    g.sync();
    const double rpv = 1.0 / W[p * ld + p];
    const int nc = ld - p - 1;
    const float rnc = 1.0f / (float)nc;
    const int tot = (n - 1) * nc;
    for (int e = g.gl; e < tot; e += G) {
      int i, j;
      divmod_small(e, nc, rnc, i, j);
      if (i >= p) ++i;
      j += p + 1;
      W[i * ld + j] = fma(-W[i * ld + p] * rpv, W[p * ld + j], W[i * ld + j]);
    }
    g.sync();
  }
  // scale by the diagonal
  const int m = ld - n;
  const float rm = 1.0f / (float)m;
  for (int e = g.gl; e < n * m; e += G) {
    int i, j;
    divmod_small(e, m, rm, i, j);
    W[i * ld + n + j] = W[i * ld + n + j] / W[i * ld + i];
  }
  g.sync();
}

// Gauss-Jordan with partial pivoting and NO row exchange, for a group that is a whole CTA (G > 32, n <= 32):
// the dense levels run one solve per combine on the latency-critical path, so the barriers per pivot count.
// The pivot of column p is the largest entry among the rows not yet used as a pivot; it is found by every
// warp on its own (lane l holds row l, warp-reduction arg-max, ties to the lower row, so all warps agree without
// a barrier), the row stays where it is and only its index is recorded.  Elimination p writes columns > p of
// the other rows and reads column p and row r only, so ONE barrier per pivot (before the next search) is
// enough, against three in gj_solve.  Same pivots, hence the same arithmetic per entry, as gj_solve.
// W = [M | R] (n rows, nc_all = n + m columns, row stride ld >= nc_all: an odd ld keeps the column reads of the
// pivot search and the row pairs of a warp off the same banks) is destroyed; X (n x m, row stride m) receives M^-1 R.
template <int G>
__device__ void gj_solve_np(const Grp<G>& g, int n, int nc_all, int ld, double* W, double* X) {
  __shared__ int rowof[32];
  const int lane = threadIdx.x & 31;
  unsigned used = 0u;
  for (int p = 0; p < n; ++p) {
    // arg-max of |W[., p]| over the unused rows: the bit pattern of a non-negative double orders like the value,
    // so the maximum is two 32-bit warp reductions (high word, then low word among the lanes that hold the
    // maximal high word) and a ballot; ties go to the lowest row
    const bool cand = lane < n && !((used >> lane) & 1u);
    const unsigned long long key = cand ? (unsigned long long)__double_as_longlong(fabs(W[lane * ld + p])) + 1ull : 0ull;
    const unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
    const unsigned mhi = __reduce_max_sync(0xffffffffu, hi);
    const unsigned mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? lo : 0u);
    const unsigned hit = __ballot_sync(0xffffffffu, hi == mhi && lo == mlo);
    int r = min(__ffs(hit) - 1, n - 1); // non-finite input: still one in-range row for the whole CTA
    used |= 1u << r;
    if (g.gl == 0) rowof[p] = r;
    const double rpv = 1.0 / W[r * ld + p];
    const int nc = nc_all - p - 1;
    const float rnc = 1.0f / (float)nc;
    const int tot = (n - 1) * nc;
    for (int e = g.gl; e < tot; e += G) {
      int i, j;
      divmod_small(e, nc, rnc, i, j);
      if (i >= r) ++i;
      j += p + 1;
      W[i * ld + j] = fma(-W[i * ld + p] * rpv, W[r * ld + j], W[i * ld + j]);
    }
    g.sync();
  }
  const int m = nc_all - n;
  const float rm = 1.0f / (float)m;
  for (int e = g.gl; e < n * m; e += G) {
    int i, j;
    divmod_small(e, m, rm, i, j);
    const int r = rowof[i];
    X[e] = W[r * ld + n + j] / W[r * ld + i];
  }
  g.sync();
}

// Gauss-Jordan as gj_solve_np (partial pivoting, no row exchange, same pivots and the same arithmetic per entry), with
// the augmented matrix held in REGISTERS during the elimination: thread t of the CTA owns row t / tpr and the
// columns c, c + tpr, c + 2 tpr, ... (c = t % tpr, tpr = G / n threads per row), so a pivot step touches shared
// memory only for what crosses threads -- the pivot column (n doubles, double-buffered) and the pivot row --
// instead of re-reading and re-writing every entry (round 1: 21 k of a combine's 61 k cycles, profiles/r01_dense_level_ncu.md).
// Two barriers per pivot.  W (n rows, nc_all columns, row stride ld) is read once; X (n x (nc_all - n), row
// stride nc_all - n) receives M^-1 R.  CPT >= ceil(nc_all / tpr).
#ifdef SG_JIT
#define SG_GJ_CPT ((3 * JT_N + 1 + (SG_DENSE_NT / JT_N) - 1) / (SG_DENSE_NT / JT_N))
#else
#define SG_GJ_CPT 12 /* n = 31: 8 threads per row, 94 columns */
#endif
#define SG_GJ_MAXC 96
template <int G, int CPT>
__device__ void gj_solve_reg(const Grp<G>& g, int n, int nc_all, int ld, const double* W, double* X) {
  __shared__ double colbuf[2][32];
  __shared__ double rowbuf[SG_GJ_MAXC];
  const int tpr = G / n;
  const int i = g.gl / tpr, c = g.gl - i * tpr;
  const bool act = i < n;
  double w[CPT];
#pragma unroll
  for (int s = 0; s < CPT; ++s) {
    const int j = c + s * tpr;
    w[s] = (act && j < nc_all) ? W[i * ld + j] : 0.0;
  }
  const int lane = threadIdx.x & 31;
  unsigned used = 0u;
  int outrow = 0;
  double rinv = 0.0;
  if (act && c == 0) colbuf[0][i] = w[0];
  g.sync();
  for (int p = 0; p < n; ++p) {
    const double* cb = colbuf[p & 1];
    // arg-max of |W[., p]| over the rows not yet used as a pivot: as in gj_solve_np (every warp on its own)
    const bool cand = lane < n && !((used >> lane) & 1u);
    const unsigned long long key = cand ? (unsigned long long)__double_as_longlong(fabs(cb[lane])) + 1ull : 0ull;
    const unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
    const unsigned mhi = __reduce_max_sync(0xffffffffu, hi);
    const unsigned mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? lo : 0u);
    const unsigned hit = __ballot_sync(0xffffffffu, hi == mhi && lo == mlo);
    const int r = min(__ffs(hit) - 1, n - 1);
    used |= 1u << r;
    const double rpv = 1.0 / cb[r];
    if (act && i == r) {
#pragma unroll
      for (int s = 0; s < CPT; ++s) {
        const int j = c + s * tpr;
        if (j > p && j < nc_all) rowbuf[j] = w[s];
      }
      outrow = p;
      rinv = rpv;
    }
    g.sync();
    if (act && i != r) {
      const double f = -cb[i] * rpv;
#pragma unroll
      for (int s = 0; s < CPT; ++s) {
        const int j = c + s * tpr;
        if (j > p && j < nc_all) w[s] = fma(f, rowbuf[j], w[s]);
      }
    }
    if (p + 1 < n) { // the owners of column p + 1 publish it for the next search
      const int ps = (p + 1) / tpr, pc = (p + 1) - ps * tpr;
      if (act && c == pc) {
        double v = w[0];
#pragma unroll
        for (int s = 1; s < CPT; ++s) v = (s == ps) ? w[s] : v;
        colbuf[(p + 1) & 1][i] = v;
      }
    }
    g.sync();
  }
  const int m = nc_all - n;
#pragma unroll
  for (int s = 0; s < CPT; ++s) {
    const int j = c + s * tpr;
    if (act && j >= n && j < nc_all) X[outrow * m + (j - n)] = w[s] * rinv;
  }
  g.sync();
}
