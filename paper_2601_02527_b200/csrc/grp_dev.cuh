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

#define SG_GJ_MAXC 96
#ifdef SG_JIT
#define SG_GJ_WCPT ((3 * JT_N + 1 + (SG_DENSE_NT / 32) - 1) / (SG_DENSE_NT / 32))
#else
#define SG_GJ_WCPT 12 /* 94 columns on 8 warps */
#endif

// Gauss-Jordan with partial pivoting and no row exchange, register-resident, COLUMNS PER WARP: warp w of the CTA owns
// the columns w, w + NW, w + 2 NW, ... of the augmented matrix and lane l holds row l of each of them.  A pivot
// step is then: the warp that owns column p finds the pivot row r by a warp reduction on its own registers,
// forms the multipliers f_i = W[i][p] / W[r][p] (each lane its own reciprocal candidate, so the division runs
// beside the reductions) and publishes them with r (n + 2 doubles, double-buffered): ONE barrier; every warp
// then eliminates its own columns with the pivot row's entries taken by a warp shuffle from lane r -- no shared-memory
// traffic for the matrix beyond that.  The pivot of column p is the largest entry among the rows not yet used as a
// pivot (arg-max by two 32-bit warp reductions on the bit pattern of |x|, which orders like the value, and a
// ballot; ties to the lower row); the row stays where it is and only its index is recorded, so no rows move.
// M = I + (PSD)(PSD) in every use (eigenvalues >= 1): a zero pivot cannot occur for finite input.
// W = [M | R] (n rows, nc_all columns, row stride ld: odd keeps the loads of a lane's row off one bank) is read
// once; X (n x (nc_all - n), row stride nc_all - n) receives M^-1 R.  Measured: profiles/r02_dense_level.md.
template <int G, int CPT>
__device__ void gj_solve_wcol(const Grp<G>& g, int n, int nc_all, int ld, const double* W, double* X) {
  __shared__ double fbuf[2][34];
  __shared__ __align__(16) double rowb[G / 32][CPT + (CPT & 1)];
  constexpr int NW = G / 32;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const bool act = lane < n;
  double v[CPT];
#pragma unroll
  for (int s = 0; s < CPT; ++s) {
    const int j = w + s * NW;
    v[s] = (act && j < nc_all) ? W[lane * ld + j] : 0.0;
  }
  unsigned used = 0u;
  int outrow = 0;
  double rinv = 0.0;
  for (int p = 0; p < n; ++p) {
    const int os = p / NW, ow = p - os * NW;
    double* fb = fbuf[p & 1];
    if (w == ow) {
      double a = v[0];
#pragma unroll
      for (int s = 1; s < CPT; ++s) a = (s == os) ? v[s] : a;
      const bool cand = act && !((used >> lane) & 1u);
      const unsigned long long key = cand ? (unsigned long long)__double_as_longlong(fabs(a)) + 1ull : 0ull;
      const unsigned hi = (unsigned)(key >> 32), lo = (unsigned)key;
      // every lane its own candidate reciprocal, independent of the search below.  Lanes beyond the last row hold
      // zeros: 1 / 0 would send the whole warp through the division's slow path at every pivot (measured)
      const double rc = 1.0 / (act ? a : 1.0);
      const unsigned mhi = __reduce_max_sync(0xffffffffu, hi);
      const unsigned mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? lo : 0u);
      const unsigned hit = __ballot_sync(0xffffffffu, hi == mhi && lo == mlo);
      const int r = min(__ffs(hit) - 1, n - 1);
      const double rpv = __shfl_sync(0xffffffffu, rc, r);
      fb[lane] = (lane == r) ? 0.0 : a * rpv; // multiplier of row `lane` (none for the pivot row itself)
      if (lane == 0) { fb[32] = rpv; fb[33] = (double)r; }
    }
    g.sync();
    const int r = (int)fb[33];
    const double rpv = fb[32], f = -fb[lane];
    used |= 1u << r;
    if (lane == r) { outrow = p; rinv = rpv; }
    // the pivot row's entries of this warp's columns: lane r stores them, everyone reads them back as broadcasts
    // (shuffles from lane r measured the same).  Every slot, unconditionally: the columns <= p are dead (never read again; the pivot entries
    // live on in rinv), the slots beyond nc_all hold zeros.
    double* rb = rowb[w];
    if (lane == r) {
#pragma unroll
      for (int s = 0; s < CPT; ++s) rb[s] = v[s];
    }
    __syncwarp();
#pragma unroll
    for (int s = 0; s < CPT; ++s) v[s] = fma(f, rb[s], v[s]);
  }
  const int m = nc_all - n;
#pragma unroll
  for (int s = 0; s < CPT; ++s) {
    const int j = w + s * NW;
    if (act && j >= n && j < nc_all) X[outrow * m + (j - n)] = v[s] * rinv;
  }
  g.sync();
}
