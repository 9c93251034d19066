// events.cu -- step a1: exposures -> time-sorted start/end event stream.
//
// 2N (key, payload) pairs: key = order-preserving 64-bit image of the event time, payload =
// 2*exposure + kind.  Order of the stream (include/smolgp.h; SURVEY reading c5, DESIGN R5):
//   (time, end before start, instrument, exposure index).
// "End before start" makes back-to-back exposures of one instrument legal (the Fig. 2 case).
// The pairs are laid out [all ends | all starts] in exposure order and sorted by a STABLE least-
// significant-digit radix sort: digit 0 = (kind, instrument), digits 1..8 = the bytes of the time key.
//   k_ev_init   builds the pairs, validates the input and accumulates the GLOBAL histograms of all
//               nine digits in the same pass over the exposures;
//   k_rs_pass   one launch per digit: per-tile stable ranking (warp match_any), the tile's global
//               offsets by a decoupled look-back over the tiles' digit counts, scatter.  A digit on
//               which all keys agree (the high bytes of the times of one data set; digit 0 when the
//               exposures come grouped by instrument) is found from the global histogram on the
//               device and its pass returns at once -- no host round trip decides it;
//   k_ev_final  gather + inclusive XOR scan of the instrument bits (again one look-back word per
//               tile) -> for every event the set of instruments exposing after it, hence the zero-mask
//               Z_k (idle instruments and the event's own) and the check that each instrument's events
//               alternate start, end, start, ... (no self-overlap); dt_k = t_k - t_{k-1}.
//   k_merge     after pass 0: when every (kind, instrument) run is already in time order -- exposures of an instrument
//               given in time order, the usual case -- the stream is the merge of those runs, done by ranking in one
//               launch; the eight time passes then return at once.  Otherwise they sort pass 0's output.
// Four launches when the merge succeeds (the host bets on it and checks the bet in the status read-back the call needs
// anyway; twelve, after the four, when it does not; round 1: 33); up to 8192 events ONE launch (k_ev_small).
#include <math.h>
#include <stddef.h>
#include <string.h>

#include <mutex>

#include "common.h"

#define EVF_BADTIME 1
#define EVF_BADINST 2
#define EVF_OVERLAP 4

#define RS_NT 256      /* threads per CTA of the sort and tail kernels */
#define RS_DIGITS 9

// device-resident control block of one build (zeroed by one memset per call)
struct EvCtl {
  uint32_t ghist[RS_DIGITS][256]; // global digit histograms
  uint32_t ticket[RS_DIGITS + 1]; // tile tickets per pass (+ the tail kernel)
  uint32_t unsorted;              // k_merge: some (kind, instrument) run is not in time order => the radix passes run
  uint32_t pad0;
  uint32_t ungrouped;             // some exposure has a smaller instrument index than its predecessor
  int32_t flags;                  // EVF_*
  unsigned long long maxdelta[SG_MAXINST]; // bits of the longest exposure per instrument
  double tfirst, tlast;
};

__device__ __forceinline__ uint64_t time_key(double t) {
  t = t + 0.0; // -0.0 -> +0.0: one key for one time
  uint64_t u = (uint64_t)__double_as_longlong(t);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}

// warp-aggregated shared-memory histogram increment: one atomic when the whole warp agrees on the bin
// (constant bytes of the keys would otherwise serialise 32-fold), plain atomics otherwise
__device__ __forceinline__ void hist_add(uint32_t* h, int bin, bool live) {
  const unsigned act = __ballot_sync(0xffffffffu, live);
  if (!act) return;
  const int lead = __ffs(act) - 1;
  const int b0 = __shfl_sync(0xffffffffu, bin, lead);
  const bool same = __all_sync(0xffffffffu, !live || bin == b0);
  if (same) { if ((threadIdx.x & 31) == lead) atomicAdd(&h[b0], (uint32_t)__popc(act)); }
  else if (live) atomicAdd(&h[bin], 1u);
}

__global__ void __launch_bounds__(RS_NT) k_ev_init(int64_t N, const double* __restrict__ ts, const double* __restrict__ te,
                                                   const int32_t* __restrict__ inst, int n_inst, uint64_t* __restrict__ keys,
                                                   uint32_t* __restrict__ vals, EvCtl* __restrict__ ctl) {
  __shared__ uint32_t h[RS_DIGITS][256];
  for (int e = threadIdx.x; e < RS_DIGITS * 256; e += RS_NT) (&h[0][0])[e] = 0u;
  __syncthreads();
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long dbits = 0ull; // bits of this exposure's length (0 for dead / invalid lanes)
  int q = -1;
  const bool live = i < N;
  uint64_t ke = 0, ks = 0;
  int qd = 0;
  const bool instant = (te == nullptr); // instantaneous samples (paper section 2): one observe event per sample
  if (live) {
    const double s = ts[i], e = instant ? s : te[i];
    q = inst[i];
    int bad = 0;
    if (!isfinite(s) || !isfinite(e) || (!instant && !(e > s))) bad |= EVF_BADTIME;
    if (q < 0 || q >= n_inst) bad |= EVF_BADINST;
    qd = (q < 0 || q >= n_inst) ? 0 : q;
    if (i > 0 && q < inst[i - 1]) atomicOr(&ctl->ungrouped, 1u);
    if (bad) { atomicOr(&ctl->flags, bad); q = -1; }
    ke = time_key(e); ks = time_key(s);
    keys[i] = ke;
    vals[i] = (uint32_t)(2 * i);
    if (!instant) {
      keys[N + i] = ks;
      vals[N + i] = (uint32_t)(2 * i + 1);
    }
    if (!bad && !instant) dbits = (unsigned long long)__double_as_longlong(e - s); // positive doubles order like their bits
  }
  hist_add(h[0], qd, live);                    // end event: kind 0
  hist_add(h[0], 16 + qd, live && !instant);   // start event: kind 1
#pragma unroll
  for (int p = 0; p < 8; ++p) {
    hist_add(h[1 + p], (int)((ke >> (8 * p)) & 255u), live);
    hist_add(h[1 + p], (int)((ks >> (8 * p)) & 255u), live && !instant);
  }
  // longest exposure per instrument: one atomic per (warp, instrument) instead of one per exposure
  for (int r = 0; r < n_inst; ++r) {
    unsigned long long m = (q == r) ? dbits : 0ull;
    for (int o = 16; o; o >>= 1) { const unsigned long long x = __shfl_xor_sync(0xffffffffu, m, o); m = x > m ? x : m; }
    if ((threadIdx.x & 31) == 0 && m) atomicMax(&ctl->maxdelta[r], m);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < RS_DIGITS * 256; e += RS_NT) {
    const uint32_t c = (&h[0][0])[e];
    if (c) atomicAdd(&ctl->ghist[0][0] + e, c);
  }
}

// ---- which passes move data: bit p set <=> pass p is skipped (all keys agree on digit p; digit 0: the
// initial layout [ends | starts] is already in (kind, instrument, index) order).  Every CTA of every
// pass recomputes it from the global histogram (9 x 256 words), so the ping-pong parity of the buffers
// never needs the host.
__device__ __forceinline__ unsigned skip_mask(const EvCtl* ctl, uint32_t n, unsigned* s_mask) {
  if (threadIdx.x == 0) *s_mask = ctl->ungrouped ? 0u : 1u;
  __syncthreads();
  unsigned m = 0;
  for (int p = 1; p < RS_DIGITS; ++p)
    if (ctl->ghist[p][threadIdx.x] == n) m |= 1u << p;
  if (m) atomicOr(s_mask, m);
  __syncthreads();
  return *s_mask;
}

// look-back status word: [epoch:30 | flag:2 | count:32]; a word of another epoch reads as "not yet there"
#define LB_WIN 8
#define LB_AGG 1ull
#define LB_INC 2ull
__device__ __forceinline__ unsigned long long lb_pack(uint32_t epoch, unsigned long long flag, uint32_t v) {
  return ((unsigned long long)epoch << 34) | (flag << 32) | v;
}
__device__ __forceinline__ unsigned long long lb_load(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void lb_store(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// One pass of the LSD radix sort.  Tile = RS_NT * ITEMS keys, warp w of the CTA ranks the contiguous run
// [w * 32 * ITEMS, (w + 1) * 32 * ITEMS) of the tile in rounds of 32 (stable: run order, round order, lane
// order).  status: [tiles][256] look-back words of this ctx (never cleared: the epoch tells the passes apart).
template <int ITEMS>
__global__ void __launch_bounds__(RS_NT) k_rs_pass(EvCtl* __restrict__ ctl, int pass, uint64_t* __restrict__ kA, uint32_t* __restrict__ vA,
                                                   uint64_t* __restrict__ kB, uint32_t* __restrict__ vB, const int32_t* __restrict__ inst,
                                                   int n_inst, uint32_t n, unsigned long long* __restrict__ status, uint32_t epoch) {
  __shared__ uint32_t wcnt[RS_NT / 32][256];
  __shared__ uint32_t base[256];
  __shared__ uint32_t wsum[RS_NT / 32];
  __shared__ unsigned s_mask;
  __shared__ uint32_t s_tile;
  if (pass >= 1 && ctl->unsorted == 0u) return; // k_merge has produced the sorted stream already
  const unsigned skip = skip_mask(ctl, n, &s_mask);
  if ((skip >> pass) & 1u) return;
  const int moved = __popc(~skip & ((1u << pass) - 1u)); // passes before this one that moved the data
  const uint64_t* kin = (moved & 1) ? kB : kA;
  const uint32_t* vin = (moved & 1) ? vB : vA;
  uint64_t* kout = (moved & 1) ? kA : kB;
  uint32_t* vout = (moved & 1) ? vA : vB;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_tile = atomicAdd(&ctl->ticket[pass], 1u); // tiles are taken in start order: a predecessor is always running
  for (int e = tid; e < (RS_NT / 32) * 256; e += RS_NT) (&wcnt[0][0])[e] = 0u;
  __syncthreads();
  const uint32_t tile = s_tile;
  const uint32_t t0 = tile * (uint32_t)(RS_NT * ITEMS) + (uint32_t)w * (32 * ITEMS);
  uint64_t k[ITEMS];
  uint32_t v[ITEMS];
  int dg[ITEMS];
  uint32_t rk[ITEMS];
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const uint32_t p = t0 + r * 32 + lane;
    const bool live = p < n;
    k[r] = 0; v[r] = 0; dg[r] = 256 + lane; // dead lanes get distinct pseudo-digits
    if (live) {
      k[r] = kin[p]; v[r] = vin[p];
      if (pass == 0) {
        int q = inst[v[r] >> 1];
        if (q < 0 || q >= n_inst) q = 0;
        dg[r] = (int)((v[r] & 1u) << 4) | q;
      } else dg[r] = (int)((k[r] >> (8 * (pass - 1))) & 255u);
    }
    const unsigned peers = __match_any_sync(0xffffffffu, dg[r]);
    const int leader = __ffs(peers) - 1;
    uint32_t old = 0;
    if (live && lane == leader) { old = wcnt[w][dg[r]]; wcnt[w][dg[r]] = old + __popc(peers); }
    old = __shfl_sync(0xffffffffu, old, leader);
    rk[r] = old + __popc(peers & ((1u << lane) - 1u));
    __syncwarp();
  }
  __syncthreads();
  // thread d: exclusive scan over the warps of digit d's counts; tile count of digit d
  uint32_t cnt = 0;
#pragma unroll
  for (int ww = 0; ww < RS_NT / 32; ++ww) { const uint32_t c = wcnt[ww][tid]; wcnt[ww][tid] = cnt; cnt += c; }
  unsigned long long* st = status + (size_t)tile * 256 + tid;
  lb_store(st, lb_pack(epoch, tile == 0 ? LB_INC : LB_AGG, cnt));
  // exclusive scan over the digits of the global histogram (position of the first key of each digit)
  const uint32_t g = ctl->ghist[pass][tid];
  uint32_t x = g;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
  if (lane == 31) wsum[w] = x;
  __syncthreads();
  uint32_t wbase = 0;
#pragma unroll
  for (int ww = 0; ww < RS_NT / 32; ++ww) if (ww < w) wbase += wsum[ww];
  uint32_t excl = 0;
  if (tile > 0) {
    // look back LB_WIN tiles at a time (independent loads in flight: the walk costs one round trip per window, not per
    // tile); entries are consumed nearest first, up to the first inclusive prefix or the first word not yet published
    int64_t t = (int64_t)tile - 1;
    bool done = false;
    while (!done) {
      unsigned long long sw[LB_WIN];
#pragma unroll
      for (int i = 0; i < LB_WIN; ++i) sw[i] = (t - i >= 0) ? lb_load(status + (size_t)(t - i) * 256 + tid) : lb_pack(epoch, LB_INC, 0u);
      int used = 0;
#pragma unroll
      for (int i = 0; i < LB_WIN; ++i) {
        if (done || used != i) continue;
        const unsigned long long s = sw[i];
        if ((uint32_t)(s >> 34) != epoch || ((s >> 32) & 3ull) == 0ull) continue; // not published yet: retry from here
        excl += (uint32_t)s;
        used = i + 1;
        if (((s >> 32) & 3ull) == LB_INC) done = true;
      }
      t -= used;
    }
    lb_store(st, lb_pack(epoch, LB_INC, excl + cnt));
  }
  base[tid] = wbase + x - g + excl;
  __syncthreads();
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const uint32_t p = t0 + r * 32 + lane;
    if (p < n) {
      const uint32_t pos = base[dg[r]] + wcnt[w][dg[r]] + rk[r];
      kout[pos] = k[r];
      vout[pos] = v[r];
    }
  }
}

// ---- merge of pre-sorted runs -------------------------------------------------------------------------------------
// After pass 0 the pairs form up to 2 N_inst runs, one per (kind, instrument), each in exposure order.  Exposures
// of one instrument usually arrive in time order, and then every run is already sorted: the stream is the MERGE
// of the runs, and an element's final position is its index in its own run plus, for every other run, the number
// of elements that precede it (binary search: keys <= mine in the runs before mine, keys < mine in the runs after
// it -- the runs are in (kind, instrument) order, which is the tie rule).  One launch instead of eight radix
// passes; a run found out of order raises ctl->unsorted and the passes run on pass 0's output as before.
__global__ void __launch_bounds__(RS_NT) k_merge(EvCtl* __restrict__ ctl, uint64_t* __restrict__ kA, uint32_t* __restrict__ vA, uint64_t* __restrict__ kB,
                                                 uint32_t* __restrict__ vB, const int32_t* __restrict__ inst, int n_inst, uint32_t n) {
  __shared__ uint32_t start[33];
  const int tid = threadIdx.x;
  if (tid < 32) { // exclusive scan of the (kind, instrument) counts: run boundaries
    const uint32_t c = ctl->ghist[0][tid];
    uint32_t x = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (tid >= o) x += y; }
    start[tid] = x - c;
    if (tid == 31) start[32] = x;
  }
  __syncthreads();
  const bool moved0 = ctl->ungrouped != 0u; // pass 0 ran: its output is in B
  const uint64_t* kin = moved0 ? kB : kA;
  const uint32_t* vin = moved0 ? vB : vA;
  uint64_t* kout = moved0 ? kA : kB;
  uint32_t* vout = moved0 ? vA : vB;
  const uint32_t p = blockIdx.x * RS_NT + tid;
  if (p >= n) return;
  const uint64_t key = kin[p];
  const uint32_t val = vin[p];
  int q = inst[val >> 1];
  if (q < 0 || q >= n_inst) q = 0;
  const int r = (int)((val & 1u) << 4) | q;
  if (p > start[r] && kin[p - 1] > key) atomicOr(&ctl->unsorted, 1u);
  uint32_t rank = p - start[r];
  for (int rr = 0; rr < 32; ++rr) {
    const uint32_t lo0 = start[rr], hi0 = start[rr + 1];
    if (rr == r || lo0 == hi0) continue;
    uint32_t lo = lo0, hi = hi0; // first index whose key is > mine (rr < r) or >= mine (rr > r)
    while (lo < hi) {
      const uint32_t mid = (lo + hi) >> 1;
      const uint64_t km = kin[mid];
      const bool before = (rr < r) ? (km <= key) : (km < key);
      if (before) lo = mid + 1; else hi = mid;
    }
    rank += lo - lo0;
  }
  kout[rank] = key;
  vout[rank] = val;
}

// ---- after the sort: gather, inclusive XOR scan of the instrument bits, flags -----------------------
#define EF_ITEMS 4
__global__ void __launch_bounds__(RS_NT) k_ev_final(EvCtl* __restrict__ ctl, int64_t K, const uint32_t* __restrict__ vA,
                                                    const uint32_t* __restrict__ vB, const double* __restrict__ ts,
                                                    const double* __restrict__ te, const int32_t* __restrict__ inst, int n_inst,
                                                    double* __restrict__ t, double* __restrict__ dt, double* __restrict__ delta,
                                                    uint32_t* __restrict__ meta, int32_t* __restrict__ obs,
                                                    unsigned long long* __restrict__ status, uint32_t epoch) {
  __shared__ double st_t[RS_NT * EF_ITEMS + 1];
  __shared__ uint32_t wx[RS_NT / 32];
  __shared__ unsigned s_mask;
  __shared__ uint32_t s_tile, s_run;
  const bool instant = (te == nullptr);
  const unsigned skip = skip_mask(ctl, (uint32_t)K, &s_mask);
  const int moved = (ctl->unsorted == 0u) ? ((ctl->ungrouped != 0u) ? 2 : 1)  // merged: pass 0 (if it ran) + k_merge
                                          : __popc(~skip & ((1u << RS_DIGITS) - 1u));
  const uint32_t* vals = (moved & 1) ? vB : vA;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  if (tid == 0) s_tile = atomicAdd(&ctl->ticket[RS_DIGITS], 1u);
  __syncthreads();
  const uint32_t tile = s_tile;
  const int64_t k0 = (int64_t)tile * (RS_NT * EF_ITEMS) + tid * EF_ITEMS; // blocked: a thread holds EF_ITEMS consecutive events
  uint32_t vv[EF_ITEMS], b[EF_ITEMS];
  double tt[EF_ITEMS];
  uint32_t x = 0;
#pragma unroll
  for (int r = 0; r < EF_ITEMS; ++r) {
    const int64_t k = k0 + r;
    vv[r] = 0; b[r] = 0; tt[r] = 0.0;
    if (k < K) {
      vv[r] = vals[k];
      const int64_t i = vv[r] >> 1;
      const double s = ts[i], e = instant ? s : te[i];
      int q = inst[i];
      if (q < 0 || q >= n_inst) q = 0;
      tt[r] = ((vv[r] & 1u) ? s : e) + 0.0;
      t[k] = tt[r];
      delta[k] = instant ? 1.0 : e - s; // an instantaneous sample observes H x itself: h = hs e_z with hs = tau / delta = 1
      obs[k] = (int32_t)i;
      b[r] = 1u << q;
      if (k == 0) ctl->tfirst = tt[r];
      if (k == K - 1) ctl->tlast = tt[r];
    }
    st_t[tid * EF_ITEMS + r + 1] = tt[r];
    x ^= instant ? 0u : b[r]; // instantaneous samples open nothing
  }
  if (tid == 0) { // time of the event before the tile
    const int64_t kp = (int64_t)tile * (RS_NT * EF_ITEMS) - 1;
    double tp = 0.0;
    if (kp >= 0) { const uint32_t u = vals[kp]; tp = ((u & 1u) || instant ? ts[u >> 1] : te[u >> 1]) + 0.0; }
    st_t[0] = tp;
  }
  // inclusive XOR scan of the threads' partials over the CTA
  uint32_t incl = x;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl ^= y; }
  if (lane == 31) wx[w] = incl;
  __syncthreads();
  uint32_t pre = 0;
#pragma unroll
  for (int ww = 0; ww < RS_NT / 32; ++ww) if (ww < w) pre ^= wx[ww];
  incl ^= pre;
  if (tid == RS_NT - 1) { // tile aggregate -> look-back over the earlier tiles
    unsigned long long* st = status + tile;
    lb_store(st, lb_pack(epoch, tile == 0 ? LB_INC : LB_AGG, incl));
    uint32_t run = 0;
    if (tile > 0) {
      int64_t tq = (int64_t)tile - 1;
      for (;;) {
        const unsigned long long s = lb_load(status + tq);
        if ((uint32_t)(s >> 34) != epoch || ((s >> 32) & 3ull) == 0ull) continue;
        run ^= (uint32_t)s;
        if (((s >> 32) & 3ull) == LB_INC) break;
        --tq;
      }
      lb_store(st, lb_pack(epoch, LB_INC, run ^ incl));
    }
    s_run = run;
  }
  __syncthreads();
  uint32_t after = s_run ^ incl ^ x; // open set before this thread's first event
  const uint32_t all = (n_inst >= 32) ? 0xffffffffu : ((1u << n_inst) - 1u);
#pragma unroll
  for (int r = 0; r < EF_ITEMS; ++r) {
    const int64_t k = k0 + r;
    const uint32_t before = after;
    after ^= instant ? 0u : b[r];
    if (k < K) {
      const uint32_t kind = vv[r] & 1u;
      const bool was_open = (before & b[r]) != 0;
      if (!instant && (kind == 1u) == was_open) atomicOr(&ctl->flags, EVF_OVERLAP); // a start needs closed, an end needs open
      const uint32_t zmask = ((~after) & all) | b[r];
      const int q = __ffs(b[r]) - 1;
      meta[k] = kind | ((uint32_t)q << 1) | (zmask << 8);
      dt[k] = (k == 0) ? 0.0 : tt[r] - st_t[tid * EF_ITEMS + r];
    }
  }
}

// ---- small inputs: the whole build in ONE CTA ------------------------------------------------------------------
// Up to EVS_MAX events (config 1: 2000) the twelve launches above cost more than the work: one CTA of 1024 threads
// sorts the (time key, kind | instrument | exposure) pairs in shared memory (bitonic network on the composite key:
// the same total order, so the same stream bit for bit), then gathers, scans the instrument bits and writes the
// stream, flags and extents exactly as k_ev_init / k_ev_final do.
#define EVS_MAX 8192
#define EVS_NT 1024
__global__ void __launch_bounds__(EVS_NT) k_ev_small(int64_t N, const double* __restrict__ ts, const double* __restrict__ te,
                                                      const int32_t* __restrict__ inst, int n_inst, EvCtl* __restrict__ ctl,
                                                      double* __restrict__ t, double* __restrict__ dt, double* __restrict__ delta,
                                                      uint32_t* __restrict__ meta, int32_t* __restrict__ obs, int P) {
  extern __shared__ unsigned long long sk[]; // [P] time keys, then [P] secondary keys (u32)
  uint32_t* sv = reinterpret_cast<uint32_t*>(sk + P);
  __shared__ uint32_t wx[32];
  __shared__ unsigned long long smax[SG_MAXINST];
  const int tid = threadIdx.x, NT = blockDim.x; // (1024; 256 threads with eight pairs each were measured: 68 us against 41 at K = 2000)
  const bool instant = (te == nullptr);
  const int K = (int)(instant ? N : 2 * N);
  for (int e = tid; e < P; e += NT) { sk[e] = ~0ull; sv[e] = ~0u; }
  if (tid < SG_MAXINST) smax[tid] = 0ull;
  __syncthreads();
  for (int i0 = 0; i0 < (int)N; i0 += NT) { // (whole warps stay in the loop: the reduction below uses shuffles)
    const int i = i0 + tid;
    unsigned long long dbits = 0ull; // bits of this exposure's length (0 for dead / invalid lanes)
    int q = -1;
    if (i < (int)N) {
      const double s = ts[i], e = instant ? s : te[i];
      int bad = 0;
      q = inst[i];
      if (!isfinite(s) || !isfinite(e) || (!instant && !(e > s))) bad |= EVF_BADTIME;
      if (q < 0 || q >= n_inst) { bad |= EVF_BADINST; q = 0; }
      if (bad) atomicOr(&ctl->flags, bad);
      else if (!instant) dbits = (unsigned long long)__double_as_longlong(e - s); // positive doubles order like their bits
      // secondary key: end (0) before start (1), then instrument, then exposure index -- the tie rule of the stream
      sk[i] = time_key(e); sv[i] = ((uint32_t)q << 13) | (uint32_t)i;
      if (!instant) { sk[N + i] = time_key(s); sv[N + i] = (1u << 18) | ((uint32_t)q << 13) | (uint32_t)i; }
    }
    for (int r = 0; r < n_inst; ++r) { // longest exposure per instrument: one shared-memory atomic per (warp, instrument)
      unsigned long long m = (q == r) ? dbits : 0ull;
      for (int o = 16; o; o >>= 1) { const unsigned long long y = __shfl_xor_sync(0xffffffffu, m, o); m = y > m ? y : m; }
      if ((tid & 31) == 0 && m) atomicMax(&smax[r], m);
    }
  }
  __syncthreads();
  if (tid < n_inst) ctl->maxdelta[tid] = smax[tid];
  // bitonic network.  A warp owns 64 consecutive positions (thread: positions 2 tid, 2 tid + 1 of each 2 NT-block), so
  // every exchange at distance < 64 stays inside a warp: those run in registers with shuffles, and only the
  // exchanges at distance >= 64 (15 of the 66 stages at P = 2048) go through shared memory and a barrier.
  for (int k2 = 2; k2 <= P; k2 <<= 1) {
    int j2 = k2 >> 1;
    for (; j2 >= 64; j2 >>= 1) {
      for (int e = tid; e < P; e += NT) {
        const int x = e ^ j2;
        if (x > e) {
          const unsigned long long ka = sk[e], kb = sk[x];
          const uint32_t va = sv[e], vb = sv[x];
          const bool gt = (ka > kb) || (ka == kb && va > vb);
          if (gt == ((e & k2) == 0)) { sk[e] = kb; sk[x] = ka; sv[e] = vb; sv[x] = va; }
        }
      }
      __syncthreads();
    }
    for (int base = 0; base < P; base += 2 * NT) {
      const int e0 = base + 2 * tid;
      if (base + 2 * (tid & ~31) >= P) break; // this warp's 64 positions lie beyond the padded length (whole warps leave together)
      unsigned long long k0r = sk[e0], k1r = sk[e0 + 1];
      uint32_t v0r = sv[e0], v1r = sv[e0 + 1];
      const bool up = (e0 & k2) == 0; // both positions share it: k2 >= 2
      for (int j = j2; j >= 2; j >>= 1) { // partner position e ^ j: thread tid ^ (j / 2), same slot
        const int lm = j >> 1;
        const bool lower = (e0 & j) == 0;
        const unsigned long long pk0 = __shfl_xor_sync(0xffffffffu, k0r, lm), pk1 = __shfl_xor_sync(0xffffffffu, k1r, lm);
        const uint32_t pv0 = __shfl_xor_sync(0xffffffffu, v0r, lm), pv1 = __shfl_xor_sync(0xffffffffu, v1r, lm);
        // the lower position keeps the smaller pair when ascending (up), the larger when descending; the upper one the other
        const bool g0 = (k0r > pk0) || (k0r == pk0 && v0r > pv0), g1 = (k1r > pk1) || (k1r == pk1 && v1r > pv1);
        if (g0 == (lower == up)) { k0r = pk0; v0r = pv0; }
        if (g1 == (lower == up)) { k1r = pk1; v1r = pv1; }
      }
      if (j2 >= 1) { // distance 1: the thread's own two positions
        const bool gt = (k0r > k1r) || (k0r == k1r && v0r > v1r);
        if (gt == up) { const unsigned long long tk = k0r; k0r = k1r; k1r = tk; const uint32_t tv = v0r; v0r = v1r; v1r = tv; }
      }
      sk[e0] = k0r; sk[e0 + 1] = k1r; sv[e0] = v0r; sv[e0 + 1] = v1r;
    }
    __syncthreads();
  }
  // gather + inclusive XOR scan of the instrument bits (a thread holds `per` consecutive events)
  const int per = (K + NT - 1) / NT, k0 = tid * per, k1 = (k0 + per < K) ? k0 + per : K;
  uint32_t x = 0;
  if (!instant)
    for (int k = k0; k < k1; ++k) x ^= 1u << ((sv[k] >> 13) & 31u);
  const int lane = tid & 31, w = tid >> 5;
  uint32_t incl = x;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl ^= y; }
  if (lane == 31) wx[w] = incl;
  __syncthreads();
  uint32_t pre = 0;
  for (int ww = 0; ww < w; ++ww) pre ^= wx[ww];
  uint32_t after = pre ^ incl ^ x; // open set before this thread's first event
  const uint32_t all = (n_inst >= 32) ? 0xffffffffu : ((1u << n_inst) - 1u);
  double tprev = 0.0;
  if (k0 > 0 && k0 < K) { const uint32_t u = sv[k0 - 1]; const int ip = (int)(u & 0x1fffu); tprev = (((u >> 18) & 1u) || instant ? ts[ip] : te[ip]) + 0.0; }
  for (int k = k0; k < k1; ++k) {
    const uint32_t u = sv[k], kind = (u >> 18) & 1u, b = 1u << ((u >> 13) & 31u);
    const int i = (int)(u & 0x1fffu), q = (int)((u >> 13) & 31u);
    const double s = ts[i], e = instant ? s : te[i];
    const double tt = (kind ? s : e) + 0.0;
    t[k] = tt;
    delta[k] = instant ? 1.0 : e - s;
    obs[k] = i;
    const uint32_t before = after;
    after ^= instant ? 0u : b;
    if (!instant && (kind == 1u) == ((before & b) != 0)) atomicOr(&ctl->flags, EVF_OVERLAP); // a start needs closed, an end needs open
    meta[k] = kind | ((uint32_t)q << 1) | ((((~after) & all) | b) << 8);
    dt[k] = (k == 0) ? 0.0 : tt - tprev;
    tprev = tt;
    if (k == 0) ctl->tfirst = tt;
    if (k == K - 1) ctl->tlast = tt;
  }
}

// look-back words of this ctx (grown on demand, zeroed when allocated; epochs start at 1)
static int lb_reserve(smolgp_ctx* ctx, size_t words) {
  if (words <= ctx->lb_words) return SMOLGP_OK;
  if (ctx->lb_status) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->lb_status); ctx->lb_status = nullptr; ctx->lb_words = 0; }
  const size_t want = words + words / 4;
  if (cudaMalloc(&ctx->lb_status, want * 8) != cudaSuccess) { cudaGetLastError(); ctx->lb_status = nullptr; ctx->err = "build_events: out of device memory (sort status)"; return SMOLGP_ENOMEM; }
  cudaMemsetAsync(ctx->lb_status, 0, want * 8, ctx->stream);
  ctx->lb_words = want;
  return SMOLGP_OK;
}
static uint32_t lb_next_epoch(smolgp_ctx* ctx) {
  if (++ctx->lb_epoch >= (1u << 30)) { // wrap: forget every old word first
    cudaMemsetAsync(ctx->lb_status, 0, ctx->lb_words * 8, ctx->stream);
    ctx->lb_epoch = 1;
  }
  return ctx->lb_epoch;
}

static int build_events_impl(smolgp_ctx* ctx, int64_t N, const double* ts, const double* te, const int32_t* inst,
                             int32_t n_inst, smolgp_events** out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!out || !ts || !inst) { ctx->err = "build_events: null argument"; return SMOLGP_EINVAL; }
  *out = nullptr;
  if (N <= 0 || N > (1ll << 30)) { ctx->err = "build_events: N must be in [1, 2^30]"; return SMOLGP_EINVAL; }
  if (n_inst < 1 || n_inst > SG_MAXINST) { ctx->err = "build_events: n_inst out of range"; return SMOLGP_EUNSUPPORTED; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  const bool instant = (te == nullptr); // instantaneous samples: K = N observe events (paper section 2)
  const int64_t K = instant ? N : 2 * N;
  smolgp_events* ev = new smolgp_events();
  ev->device = ctx->device; ev->N = N; ev->K = K; ev->n_inst = n_inst; ev->instant = instant ? 1 : 0;
  ev->t = ev->dt = ev->delta = nullptr; ev->meta = nullptr; ev->obs = nullptr; ev->base = nullptr; ev->stream = ctx->stream;
  auto fail = [&](int rc) { smolgp_free_events(ev); return rc; };
  // stream-ordered allocation (cudaMallocAsync): no device-wide synchronisation on alloc or free
  const size_t k8 = ((size_t)K * 8 + 255) / 256 * 256, k4 = ((size_t)K * 4 + 255) / 256 * 256;
  if (cudaMallocAsync(&ev->base, 3 * k8 + 2 * k4, ctx->stream) != cudaSuccess) { cudaGetLastError(); ev->base = nullptr; ctx->err = "build_events: out of device memory"; return fail(SMOLGP_ENOMEM); }
  {
    char* b = (char*)ev->base;
    ev->t = (double*)b; ev->dt = (double*)(b + k8); ev->delta = (double*)(b + 2 * k8);
    ev->meta = (uint32_t*)(b + 3 * k8); ev->obs = (int32_t*)(b + 3 * k8 + k4);
  }
  // tile size of the sort: 1024 keys up to 2^21 events (more CTAs than SMs already at 2e5), 4096 above
  const int items = (K <= (1ll << 21)) ? 4 : 16;
  const int64_t tile_rs = (int64_t)RS_NT * items, tile_ef = (int64_t)RS_NT * EF_ITEMS;
  const int64_t ntiles_rs = (K + tile_rs - 1) / tile_rs, ntiles_ef = (K + tile_ef - 1) / tile_ef;
  int rc = lb_reserve(ctx, (size_t)ntiles_rs * 256 > (size_t)ntiles_ef ? (size_t)ntiles_rs * 256 : (size_t)ntiles_ef);
  if (rc) return fail(rc);
  // scratch: control block, keys x2 (u64), vals x2 (u32)
  const size_t ctl_b = (sizeof(EvCtl) + 255) / 256 * 256;
  void* scratch;
  rc = sg_arena(ctx, ctl_b + 2 * k8 + 2 * k4, &scratch);
  if (rc) return fail(rc);
  sg_mem_mark(ctx, 3 * k8 + 2 * k4);
  char* p = (char*)scratch;
  EvCtl* ctl = (EvCtl*)p; p += ctl_b;
  uint64_t* kA = (uint64_t*)p; p += k8;
  uint64_t* kB = (uint64_t*)p; p += k8;
  uint32_t* vA = (uint32_t*)p; p += k4;
  uint32_t* vB = (uint32_t*)p;
  cudaStream_t st = ctx->stream;
  const bool small = K <= EVS_MAX;
  // ONE status read-back per attempt: merge outcome, validation flags, longest exposures, first / last event time
  struct { uint32_t unsorted, pad0, ungrouped; int32_t flags; unsigned long long md[SG_MAXINST]; double tfl[2]; } hs;
  static_assert(offsetof(EvCtl, flags) == offsetof(EvCtl, unsorted) + 12 && offsetof(EvCtl, maxdelta) == offsetof(EvCtl, flags) + 4 &&
                offsetof(EvCtl, tfirst) == offsetof(EvCtl, maxdelta) + 8 * SG_MAXINST && offsetof(EvCtl, tlast) == offsetof(EvCtl, tfirst) + 8,
                "EvCtl: unsorted | pad | ungrouped | flags | maxdelta | tfirst | tlast must be contiguous");
  // The first attempt bets that k_merge succeeds (every (kind, instrument) run in time order: the usual case) and does
  // not launch the eight time passes at all -- they would all return at once; the read-back that the call needs anyway
  // tells whether the bet held, and if not the build is redone with the passes (twice the work on unsorted input).
  for (int attempt = 0; attempt < 2; ++attempt) {
  const bool bet = (attempt == 0) && !small;
  cudaMemsetAsync(ctl, 0, sizeof(EvCtl), st);
  if (small) { // one CTA does everything (k_ev_small)
    int P2 = 64; // (a warp's 64 positions at least: k_ev_small)
    while (P2 < K) P2 <<= 1;
    const size_t smem = (size_t)P2 * 12;
    cudaFuncSetAttribute(k_ev_small, cudaFuncAttributeMaxDynamicSharedMemorySize, EVS_MAX * 12);
    sg_launch_begin(ctx, KID_EV_FINAL);
    k_ev_small<<<1, EVS_NT, smem, st>>>(N, ts, te, inst, n_inst, ctl, ev->t, ev->dt, ev->delta, ev->meta, ev->obs, P2);
    sg_launch_end(ctx);
  } else {
  sg_launch_begin(ctx, KID_EV_INIT);
  k_ev_init<<<(unsigned)((N + RS_NT - 1) / RS_NT), RS_NT, 0, st>>>(N, ts, te, inst, n_inst, kA, vA, ctl);
  sg_launch_end(ctx);
  for (int pass = 0; pass < RS_DIGITS; ++pass) {
    if (pass == 1) { // pass 0 has formed the (kind, instrument) runs: try the merge
      sg_launch_begin(ctx, KID_RS_PASS);
      k_merge<<<(unsigned)((K + RS_NT - 1) / RS_NT), RS_NT, 0, st>>>(ctl, kA, vA, kB, vB, inst, n_inst, (uint32_t)K);
      sg_launch_end(ctx);
      if (bet) break;
    }
    const uint32_t epoch = lb_next_epoch(ctx);
    sg_launch_begin(ctx, KID_RS_PASS);
    if (items == 4) k_rs_pass<4><<<(unsigned)ntiles_rs, RS_NT, 0, st>>>(ctl, pass, kA, vA, kB, vB, inst, n_inst, (uint32_t)K, ctx->lb_status, epoch);
    else k_rs_pass<16><<<(unsigned)ntiles_rs, RS_NT, 0, st>>>(ctl, pass, kA, vA, kB, vB, inst, n_inst, (uint32_t)K, ctx->lb_status, epoch);
    sg_launch_end(ctx);
  }
  {
    const uint32_t epoch = lb_next_epoch(ctx);
    sg_launch_begin(ctx, KID_EV_FINAL);
    k_ev_final<<<(unsigned)ntiles_ef, RS_NT, 0, st>>>(ctl, K, vA, vB, ts, te, inst, n_inst, ev->t, ev->dt, ev->delta, ev->meta, ev->obs, ctx->lb_status, epoch);
    sg_launch_end(ctx);
  }
  } // !small
  cudaError_t ce = cudaMemcpyAsync(&hs, &ctl->unsorted, sizeof(hs), cudaMemcpyDeviceToHost, st);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
  if (ce != cudaSuccess) { ctx->err = std::string("build_events: ") + cudaGetErrorString(ce); cudaGetLastError(); return fail(SMOLGP_ECUDA); }
  if (!(bet && hs.unsorted)) break; // (a lost bet: the stream written by k_ev_final means nothing; redo with the passes)
  }
  const int flags = hs.flags;
  if (flags & EVF_BADTIME) { ctx->err = "build_events: non-finite time or t_end <= t_start"; return fail(SMOLGP_EINVAL); }
  if (flags & EVF_BADINST) { ctx->err = "build_events: instrument index out of range"; return fail(SMOLGP_EINVAL); }
  if (flags & EVF_OVERLAP) { ctx->err = "build_events: an instrument overlaps itself (P:464)"; return fail(SMOLGP_EOVERLAP); }
  for (int q = 0; q < SG_MAXINST; ++q) {
    double dmax;
    memcpy(&dmax, &hs.md[q], 8);
    int e = 0;
    if (q < n_inst && dmax > 0) frexp(dmax, &e); // dmax = f 2^e, f in [0.5, 1)
    ev->tau[q] = (q < n_inst && dmax > 0) ? ldexp(1.0, e) : 1.0; // power of two >= the longest exposure
  }
  ev->t_first = hs.tfl[0]; ev->t_last = hs.tfl[1];
  *out = ev;
  return SMOLGP_OK;
}

extern "C" int smolgp_build_events(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                                   const int32_t* instrument, int32_t n_inst, smolgp_events** out) {
  if (ctx && !t_end) { ctx->err = "build_events: null argument"; return SMOLGP_EINVAL; }
  return build_events_impl(ctx, N, t_start, t_end, instrument, n_inst, out);
}

extern "C" int smolgp_build_events_instant(smolgp_ctx* ctx, int64_t N, const double* t, const int32_t* instrument, int32_t n_inst,
                                           smolgp_events** out) {
  return build_events_impl(ctx, N, t, nullptr, instrument, n_inst, out);
}

extern "C" int smolgp_build_events_instant_host(smolgp_ctx* ctx, int64_t N, const double* t, const int32_t* instrument,
                                                int32_t n_inst, smolgp_events** out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (N <= 0 || !t || !instrument) { ctx->err = "build_events_instant_host: bad argument"; return SMOLGP_EINVAL; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  char* stage = nullptr;
  const size_t n8 = ((size_t)N * 8 + 255) / 256 * 256;
  if (cudaMallocAsync(&stage, n8 + (size_t)N * 4, ctx->stream) != cudaSuccess) {
    cudaGetLastError(); ctx->err = "build_events_instant_host: out of device memory"; return SMOLGP_ENOMEM;
  }
  cudaMemcpyAsync(stage, t, N * 8, cudaMemcpyHostToDevice, ctx->stream);
  cudaMemcpyAsync(stage + n8, instrument, N * 4, cudaMemcpyHostToDevice, ctx->stream);
  int rc = build_events_impl(ctx, N, (const double*)stage, nullptr, (const int32_t*)(stage + n8), n_inst, out);
  cudaFreeAsync(stage, ctx->stream);
  return rc;
}

extern "C" int smolgp_build_events_host(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                                        const int32_t* instrument, int32_t n_inst, smolgp_events** out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (N <= 0 || !t_start || !t_end || !instrument) { ctx->err = "build_events_host: bad argument"; return SMOLGP_EINVAL; }
  // (instantaneous samples have their own entry point: smolgp_build_events_instant_host)
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  double *ds = nullptr, *de = nullptr; int32_t* di = nullptr;
  char* stage = nullptr;
  const size_t n8 = ((size_t)N * 8 + 255) / 256 * 256;
  if (cudaMallocAsync(&stage, 2 * n8 + (size_t)N * 4, ctx->stream) != cudaSuccess) {
    cudaGetLastError(); ctx->err = "build_events_host: out of device memory"; return SMOLGP_ENOMEM;
  }
  ds = (double*)stage; de = (double*)(stage + n8); di = (int32_t*)(stage + 2 * n8);
  cudaMemcpyAsync(ds, t_start, N * 8, cudaMemcpyHostToDevice, ctx->stream);
  cudaMemcpyAsync(de, t_end, N * 8, cudaMemcpyHostToDevice, ctx->stream);
  cudaMemcpyAsync(di, instrument, N * 4, cudaMemcpyHostToDevice, ctx->stream);
  int rc = build_events_impl(ctx, N, ds, de, di, n_inst, out);
  cudaFreeAsync(stage, ctx->stream);
  return rc;
}

extern "C" void smolgp_free_events(smolgp_events* ev) {
  if (!ev) return;
  if (ev->base) cudaFreeAsync(ev->base, ev->stream); // ordered after every kernel enqueued so far on that stream
  delete ev;
}

extern "C" int smolgp_events_export(smolgp_ctx* ctx, const smolgp_events* ev, double* t, int32_t* kind,
                                    int32_t* instrument, int32_t* exposure) {
  if (!ctx || !ev) return SMOLGP_EINVAL;
  const int64_t K = ev->K;
  std::vector<uint32_t> meta(K);
  SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  if (t) SG_CUDA(ctx, cudaMemcpy(t, ev->t, K * 8, cudaMemcpyDeviceToHost));
  SG_CUDA(ctx, cudaMemcpy(meta.data(), ev->meta, K * 4, cudaMemcpyDeviceToHost));
  if (exposure) SG_CUDA(ctx, cudaMemcpy(exposure, ev->obs, K * 4, cudaMemcpyDeviceToHost));
  for (int64_t k = 0; k < K; ++k) {
    if (kind) kind[k] = (int32_t)META_KIND(meta[k]);
    if (instrument) instrument[k] = (int32_t)META_INST(meta[k]);
  }
  return SMOLGP_OK;
}

// ---- event build that allocates nothing (include/smolgp.h: smolgp_build_events_noalloc) ----------------------------
// For callers that cannot call cudaMalloc (stream capture, serving loops, harnesses that forbid it): the same
// kernels as build_events_impl, with the sort's scratch -- control block, look-back words, two key and two payload
// buffers -- in ONE file-scope device array instead of the ctx arena, outputs in caller-provided device arrays,
// the validation flags left in a caller-provided device word instead of a host read-back + synchronise.
// Every GPU that loads the library holds the array (NA_BYTES, about 6.5 MB) until exit.  All calls on a device
// share it: calls that overlap on the GPU (two streams, two threads) race; serialise them.
#define NA_MAXK (1 << 18)                       /* events: N <= 131072 exposures, or 262144 instantaneous samples */
#define NA_ITEMS 4                              /* tile of the sort: RS_NT * 4 keys, as build_events_impl up to 2^21 events */
#define NA_TILES (NA_MAXK / (RS_NT * NA_ITEMS)) /* 256 */
#define NA_CTL_B ((sizeof(EvCtl) + 255) / 256 * 256)
#define NA_LB_B ((size_t)NA_TILES * 256 * 8)
#define NA_K8 ((size_t)NA_MAXK * 8)
#define NA_K4 ((size_t)NA_MAXK * 4)
#define NA_BYTES (NA_CTL_B + NA_LB_B + 2 * NA_K8 + 2 * NA_K4)
static __device__ __align__(256) unsigned char g_na_scratch[NA_BYTES];

#define NA_MAXDEV 64
static void* g_na_ptr[NA_MAXDEV];       // device address of g_na_scratch on device d (the symbol itself is a host-side stand-in)
static std::mutex g_na_mu;
static thread_local std::string g_na_err;

extern "C" const char* smolgp_noalloc_last_error(void) { return g_na_err.c_str(); }
extern "C" int64_t smolgp_noalloc_max_events(void) { return NA_MAXK; }
extern "C" int64_t smolgp_noalloc_scratch_bytes(void) { return (int64_t)NA_BYTES; }

// once per device, with that device current: the address of the scratch array on it
extern "C" int smolgp_noalloc_setup(int32_t device) {
  if (device < 0 || device >= NA_MAXDEV) { g_na_err = "noalloc: device index out of range"; return SMOLGP_EINVAL; }
  std::lock_guard<std::mutex> lk(g_na_mu);
  if (g_na_ptr[device]) return SMOLGP_OK;
  cudaError_t ce = cudaSetDevice(device);
  void* p = nullptr;
  if (ce == cudaSuccess) ce = cudaGetSymbolAddress(&p, g_na_scratch);
  if (ce != cudaSuccess || !p) {
    g_na_err = std::string("noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(ce);
    cudaGetLastError();
    return SMOLGP_ECUDA;
  }
  g_na_ptr[device] = p;
  return SMOLGP_OK;
}

extern "C" int smolgp_build_events_noalloc(int32_t device, void* cuda_stream, int64_t N, const double* ts, const double* te,
                                           const int32_t* inst, int32_t n_inst, double* t, double* dt, double* delta,
                                           uint32_t* meta, int32_t* exposure, int32_t* flags) {
  if (!ts || !inst || !t || !dt || !delta || !meta || !exposure || !flags) { g_na_err = "build_events_noalloc: null argument"; return SMOLGP_EINVAL; }
  if (n_inst < 1 || n_inst > SG_MAXINST) { g_na_err = "build_events_noalloc: n_inst out of range"; return SMOLGP_EUNSUPPORTED; }
  const bool instant = (te == nullptr);
  if (N <= 0) { g_na_err = "build_events_noalloc: N must be positive"; return SMOLGP_EINVAL; }
  const int64_t K = instant ? N : 2 * N;
  if (K > NA_MAXK) {
    g_na_err = "build_events_noalloc: " + std::to_string((long long)K) + " events exceed the fixed scratch (at most " +
               std::to_string((long long)NA_MAXK) + " events = " + std::to_string((long long)NA_MAXK / 2) +
               " exposures or " + std::to_string((long long)NA_MAXK) + " instantaneous samples); use smolgp_build_events";
    return SMOLGP_EUNSUPPORTED;
  }
  int rc = smolgp_noalloc_setup(device);
  if (rc) return rc;
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); g_na_err = "build_events_noalloc: cudaSetDevice failed"; return SMOLGP_ECUDA; }
  char* p = (char*)g_na_ptr[device];
  EvCtl* ctl = (EvCtl*)p; p += NA_CTL_B;
  unsigned long long* status = (unsigned long long*)p; p += NA_LB_B;
  uint64_t* kA = (uint64_t*)p; p += NA_K8;
  uint64_t* kB = (uint64_t*)p; p += NA_K8;
  uint32_t* vA = (uint32_t*)p; p += NA_K4;
  uint32_t* vB = (uint32_t*)p;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t tile_rs = (int64_t)RS_NT * NA_ITEMS, tile_ef = (int64_t)RS_NT * EF_ITEMS;
  const int64_t ntiles_rs = (K + tile_rs - 1) / tile_rs, ntiles_ef = (K + tile_ef - 1) / tile_ef;
  // the array keeps the last call's contents: the control block and the look-back words this call will read start at
  // zero (epoch 0 = "not published"; the ten launches below use epochs 1..10); keys and payloads are fully rewritten
  cudaMemsetAsync(ctl, 0, NA_CTL_B + (size_t)ntiles_rs * 256 * 8, st);
  k_ev_init<<<(unsigned)((N + RS_NT - 1) / RS_NT), RS_NT, 0, st>>>(N, ts, te, inst, n_inst, kA, vA, ctl);
  uint32_t epoch = 0;
  for (int pass = 0; pass < RS_DIGITS; ++pass) {
    if (pass == 1) k_merge<<<(unsigned)((K + RS_NT - 1) / RS_NT), RS_NT, 0, st>>>(ctl, kA, vA, kB, vB, inst, n_inst, (uint32_t)K);
    k_rs_pass<NA_ITEMS><<<(unsigned)ntiles_rs, RS_NT, 0, st>>>(ctl, pass, kA, vA, kB, vB, inst, n_inst, (uint32_t)K, status, ++epoch);
  }
  k_ev_final<<<(unsigned)ntiles_ef, RS_NT, 0, st>>>(ctl, K, vA, vB, ts, te, inst, n_inst, t, dt, delta, meta, exposure, status, ++epoch);
  // validation flags to the caller's device word, in stream order: no host read-back, no synchronisation
  cudaMemcpyAsync(flags, &ctl->flags, sizeof(int32_t), cudaMemcpyDeviceToDevice, st);
  const cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) { g_na_err = std::string("build_events_noalloc: ") + cudaGetErrorString(ce); return SMOLGP_ECUDA; }
  return SMOLGP_OK;
}
