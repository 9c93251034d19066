// scan.cu -- steps a3-a6: the translation unit of the scan kernels and their host orchestration.
//
// Scan layout: the K events of a series are cut into chunks of Lc events.
//   up-sweep   k_fold0 (chunk_kernels.cuh): one group of lanes per chunk folds the chunk's primitive
//                        elements (Eq. 3.20/3.21; SG21 Eq. 10) into ONE element (A,b,C,eta,J).
//                        Folding a primitive element onto an aggregate is the associative combine
//                        with a rank-one J_j and a block-structured A_j: O(n^2 bs), not O(n^3).
//              k_foldD (dense_kernels.cuh): dense combine of g consecutive elements per level.
//   down-sweep k_downD (dense_kernels.cuh): from the top, the state (m,P) before every element (prefix)
//                        and the backward information (eta,J) after it (suffix of the SAME elements).
//              k_down0 (chunk_kernels.cuh): per chunk, the plain integrated Kalman filter (Eq. 3.14-3.15,
//                        2.22) from the chunk's prefix state -> innovations -> log-likelihood terms
//                        (Eq. 2.26); then the adjoint (modified Bryson-Frazier) recursion of that filter
//                        started from the chunk's suffix information, with the smoothed exposure average at
//                        each end event (the two-filter posterior of reading R7 without per-event solves).
// With one chunk per series (Lc >= K) only k_down0 runs: the sequential per-series filter (row a8).
// Here: the log-likelihood reduction (a5), the query locator (a7) and scan_host.cu (plan and launches).
#include <math.h>

#include "dense_kernels.cuh"
#include "chunk_sqrt.cuh" // (shared-memory sizes of the factor-form kernels for the plan; the kernels are instantiated in scan_sqrt.cu)

__global__ void k_ll_reduce(const double* __restrict__ llpart, int64_t c1, int64_t batch, int64_t N,
                            const double* __restrict__ amp, double* __restrict__ loglik, int* __restrict__ flags) {
  // one warp per series; fixed summation order (lane-strided partial sums, then a butterfly)
  const int64_t s = (int64_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
  if (s >= batch) return;
  const int lane = threadIdx.x & 31;
  double acc = 0.0;
  for (int64_t c = lane; c < c1; c += 32) acc += llpart[s * c1 + c];
  for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    const double ll = acc - (amp ? (double)N * log(amp[s]) : 0.0);
    if (!isfinite(ll)) atomicOr(flags, NUMF_BAD);
    loglik[s] = ll;
  }
}

// ---------------------------------------------------------------------------------------------------
// Row a7: prediction at arbitrary times (Algorithm 1), adjoint form of the two-filter posterior.
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

#include "scan_host.cu"
