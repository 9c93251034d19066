// events.cu -- step a1: exposures -> time-sorted start/end event stream.
//
// 2N (key, payload) pairs: key = order-preserving 64-bit image of the event time, payload =
// 2*exposure + kind.  The pairs are laid out [all ends | all starts] and sorted by a STABLE
// least-significant-digit radix sort (8 passes of 8 bits), so equal times keep "end before start"
// (reading R5: needed for back-to-back exposures, the Fig. 2 case P:543).  An inclusive XOR scan
// of the instrument bits gives, for every event, the set of instruments that are exposing after
// it; from it come the zero-mask Z_k (idle instruments and the event's own) and the check that
// each instrument's events alternate start, end, start, ... (no self-overlap).
#include <math.h>

#include "common.h"

#define EVF_BADTIME 1
#define EVF_BADINST 2
#define EVF_OVERLAP 4

__device__ __forceinline__ uint64_t time_key(double t) {
  uint64_t u = (uint64_t)__double_as_longlong(t);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}

__global__ void k_ev_init(int64_t N, const double* __restrict__ ts, const double* __restrict__ te,
                          const int32_t* __restrict__ inst, int n_inst, uint64_t* __restrict__ keys,
                          uint32_t* __restrict__ vals, int* __restrict__ flags,
                          unsigned long long* __restrict__ maxdelta) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long dbits = 0ull; // bits of this exposure's length (0 for dead / invalid lanes)
  int q = -1;
  if (i < N) {
    const double s = ts[i], e = te[i];
    q = inst[i];
    int bad = 0;
    if (!isfinite(s) || !isfinite(e) || !(e > s)) bad |= EVF_BADTIME;
    if (q < 0 || q >= n_inst) bad |= EVF_BADINST;
    if (bad) { atomicOr(flags, bad); q = -1; }
    keys[i] = time_key(e);
    vals[i] = (uint32_t)(2 * i);
    keys[N + i] = time_key(s);
    vals[N + i] = (uint32_t)(2 * i + 1);
    if (!bad) dbits = (unsigned long long)__double_as_longlong(e - s); // positive doubles order like their bits
  }
  // longest exposure per instrument: one atomic per (warp, instrument) instead of one per exposure
  for (int r = 0; r < n_inst; ++r) {
    unsigned long long m = (q == r) ? dbits : 0ull;
    for (int o = 16; o; o >>= 1) { const unsigned long long x = __shfl_xor_sync(0xffffffffu, m, o); m = x > m ? x : m; }
    if ((threadIdx.x & 31) == 0 && m) atomicMax(maxdelta + r, m);
  }
}

// ---- LSD radix sort, 8 bits per pass.  One warp per tile of RS_TILE keys, RS_WPB tiles per CTA. ----
// hist: per-tile digit counts (digit-major) + global digit totals; scan: one CTA per digit turns its
// row into global positions (base = total of the smaller digits); scatter: stable, warp-serial
// ranking with match_any (equal keys keep their order: ends stay before starts, reading R5).
#define RS_TILE 512
#define RS_WPB 4
__global__ void __launch_bounds__(32 * RS_WPB) k_rs_hist(const uint64_t* __restrict__ keys, int64_t n, int shift,
                                                         uint32_t* __restrict__ hist, int ntiles, uint32_t* __restrict__ gcnt) {
  __shared__ uint32_t cnt_all[RS_WPB][256];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int tile = blockIdx.x * RS_WPB + w;
  uint32_t* cnt = cnt_all[w];
  for (int b = lane; b < 256; b += 32) cnt[b] = 0;
  __syncwarp();
  if (tile < ntiles) {
    const int64_t base = (int64_t)tile * RS_TILE;
    for (int i = lane; i < RS_TILE; i += 32) {
      const int64_t p = base + i;
      if (p < n) atomicAdd(&cnt[(keys[p] >> shift) & 255u], 1u);
    }
    __syncwarp();
    for (int b = lane; b < 256; b += 32) {
      const uint32_t c = cnt[b];
      hist[(int64_t)b * ntiles + tile] = c; // digit-major
      if (c) atomicAdd(&gcnt[b], c);
    }
  }
}
// exclusive scan of the digit-major histogram: CTA d scans row d, starting at the total of digits < d
__global__ void __launch_bounds__(256) k_rs_scan(uint32_t* __restrict__ hist, int ntiles, const uint32_t* __restrict__ gcnt) {
  __shared__ uint32_t sm[256];
  __shared__ uint32_t carry;
  const int d = blockIdx.x, tid = threadIdx.x;
  sm[tid] = (tid < d) ? gcnt[tid] : 0u;
  __syncthreads();
  for (int off = 128; off; off >>= 1) { if (tid < off) sm[tid] += sm[tid + off]; __syncthreads(); }
  if (tid == 0) carry = sm[0];
  __syncthreads();
  uint32_t* row = hist + (int64_t)d * ntiles;
  for (int t0 = 0; t0 < ntiles; t0 += 256) {
    const int t = t0 + tid;
    const uint32_t v = (t < ntiles) ? row[t] : 0u;
    const uint32_t run0 = carry;
    __syncthreads();
    sm[tid] = v;
    __syncthreads();
    for (int off = 1; off < 256; off <<= 1) {
      const uint32_t x = (tid >= off) ? sm[tid - off] : 0u;
      __syncthreads();
      sm[tid] += x;
      __syncthreads();
    }
    if (t < ntiles) row[t] = run0 + sm[tid] - v;
    if (tid == 255) carry = run0 + sm[255];
    __syncthreads();
  }
}
__global__ void __launch_bounds__(32 * RS_WPB) k_rs_scatter(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ vals,
                                                            uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out,
                                                            int64_t n, int shift, const uint32_t* __restrict__ hist, int ntiles) {
  __shared__ uint32_t pos_all[RS_WPB][256];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int tile = blockIdx.x * RS_WPB + w;
  if (tile >= ntiles) return;
  uint32_t* pos = pos_all[w];
  for (int b = lane; b < 256; b += 32) pos[b] = hist[(int64_t)b * ntiles + tile];
  __syncwarp();
  const int64_t base = (int64_t)tile * RS_TILE;
  for (int i0 = 0; i0 < RS_TILE; i0 += 32) {
    const int64_t p = base + i0 + lane;
    const bool live = p < n;
    uint64_t k = 0;
    uint32_t v = 0;
    int dg = 256 + lane; // dead lanes get distinct pseudo-digits
    if (live) { k = keys[p]; v = vals[p]; dg = (int)((k >> shift) & 255u); }
    const unsigned peers = __match_any_sync(0xffffffffu, dg);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    const int leader = __ffs(peers) - 1;
    uint32_t basepos = 0;
    if (live && lane == leader) { basepos = pos[dg]; pos[dg] = basepos + __popc(peers); }
    basepos = __shfl_sync(0xffffffffu, basepos, leader);
    if (live) { keys_out[basepos + rank] = k; vals_out[basepos + rank] = v; }
    __syncwarp();
  }
}

// gcnt: 8 x 256 counters (one slice per pass)
int sg_sort_pairs(smolgp_ctx* ctx, uint64_t* keys, uint32_t* vals, uint64_t* keys_tmp, uint32_t* vals_tmp,
                  int64_t n, uint32_t* hist, uint32_t* gcnt) {
  const int ntiles = (int)((n + RS_TILE - 1) / RS_TILE);
  const unsigned blocks = (unsigned)((ntiles + RS_WPB - 1) / RS_WPB);
  uint64_t* kin = keys; uint32_t* vin = vals; uint64_t* kout = keys_tmp; uint32_t* vout = vals_tmp;
  cudaMemsetAsync(gcnt, 0, 8 * 256 * sizeof(uint32_t), ctx->stream);
  for (int pass = 0; pass < 8; ++pass) {
    const int shift = 8 * pass;
    uint32_t* gc = gcnt + pass * 256;
    sg_launch_begin(ctx, KID_RS_HIST);
    k_rs_hist<<<blocks, 32 * RS_WPB, 0, ctx->stream>>>(kin, n, shift, hist, ntiles, gc);
    sg_launch_end(ctx);
    sg_launch_begin(ctx, KID_RS_SCAN);
    k_rs_scan<<<256, 256, 0, ctx->stream>>>(hist, ntiles, gc);
    sg_launch_end(ctx);
    sg_launch_begin(ctx, KID_RS_SCATTER);
    k_rs_scatter<<<blocks, 32 * RS_WPB, 0, ctx->stream>>>(kin, vin, kout, vout, n, shift, hist, ntiles);
    sg_launch_end(ctx);
    uint64_t* tk = kin; kin = kout; kout = tk;
    uint32_t* tv = vin; vin = vout; vout = tv;
  }
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK; // 8 passes: the result is back in (keys, vals)
}

// ---- after the sort --------------------------------------------------------------------------------
__global__ void k_ev_gather(int64_t K, const uint32_t* __restrict__ vals, const double* __restrict__ ts,
                            const double* __restrict__ te, const int32_t* __restrict__ inst, int n_inst,
                            double* __restrict__ t, double* __restrict__ delta, int32_t* __restrict__ obs,
                            uint32_t* __restrict__ bits) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= K) return;
  const uint32_t v = vals[k];
  const int64_t i = v >> 1;
  const double s = ts[i], e = te[i];
  int q = inst[i];
  if (q < 0 || q >= n_inst) q = 0;
  t[k] = (v & 1u) ? s : e;
  delta[k] = e - s;
  obs[k] = (int32_t)i;
  bits[k] = 1u << q;
}

// inclusive XOR scan, three kernels (tile reduce, scan of tile sums, apply)
#define XS_TILE 1024
__global__ void __launch_bounds__(256) k_xs_reduce(const uint32_t* __restrict__ bits, int64_t K, uint32_t* __restrict__ tile) {
  __shared__ uint32_t sm[8];
  const int64_t base = (int64_t)blockIdx.x * XS_TILE;
  uint32_t x = 0;
  for (int i = threadIdx.x; i < XS_TILE; i += 256) if (base + i < K) x ^= bits[base + i];
  for (int o = 16; o; o >>= 1) x ^= __shfl_xor_sync(0xffffffffu, x, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = x;
  __syncthreads();
  if (threadIdx.x == 0) { uint32_t r = 0; for (int w = 0; w < 8; ++w) r ^= sm[w]; tile[blockIdx.x] = r; }
}
__global__ void k_xs_tiles(uint32_t* __restrict__ tile, int ntiles) { // exclusive, serial: ntiles <= a few thousand
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    uint32_t run = 0;
    for (int i = 0; i < ntiles; ++i) { uint32_t v = tile[i]; tile[i] = run; run ^= v; }
  }
}
__global__ void __launch_bounds__(32) k_ev_final(int64_t K, const uint32_t* __restrict__ bits, const uint32_t* __restrict__ tile,
                                                 const uint32_t* __restrict__ vals, const double* __restrict__ t,
                                                 int n_inst, uint32_t* __restrict__ meta, double* __restrict__ dt,
                                                 int* __restrict__ flags) {
  const int lane = threadIdx.x;
  const int64_t base = (int64_t)blockIdx.x * XS_TILE;
  uint32_t run = tile[blockIdx.x];
  const uint32_t all = (n_inst >= 32) ? 0xffffffffu : ((1u << n_inst) - 1u);
  for (int i0 = 0; i0 < XS_TILE; i0 += 32) {
    const int64_t k = base + i0 + lane;
    const uint32_t b = (k < K) ? bits[k] : 0u;
    uint32_t x = b;
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x ^= y; }
    const uint32_t after = run ^ x, before = after ^ b;
    if (k < K) {
      const uint32_t kind = vals[k] & 1u;
      const bool was_open = (before & b) != 0;
      if ((kind == 1u) == was_open) atomicOr(flags, EVF_OVERLAP); // a start needs closed, an end needs open
      const uint32_t zmask = ((~after) & all) | b;
      const int q = __ffs(b) - 1;
      meta[k] = kind | ((uint32_t)q << 1) | (zmask << 8);
      dt[k] = (k == 0) ? 0.0 : t[k] - t[k - 1];
    }
    run ^= __shfl_sync(0xffffffffu, x, 31);
  }
}

static int build_events_impl(smolgp_ctx* ctx, int64_t N, const double* ts, const double* te, const int32_t* inst,
                             int32_t n_inst, smolgp_events** out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!out || !ts || !te || !inst) { ctx->err = "build_events: null argument"; return SMOLGP_EINVAL; }
  *out = nullptr;
  if (N <= 0 || N > (1ll << 30)) { ctx->err = "build_events: N must be in [1, 2^30]"; return SMOLGP_EINVAL; }
  if (n_inst < 1 || n_inst > SG_MAXINST) { ctx->err = "build_events: n_inst out of range"; return SMOLGP_EUNSUPPORTED; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  const int64_t K = 2 * N;
  smolgp_events* ev = new smolgp_events();
  ev->device = ctx->device; ev->N = N; ev->K = K; ev->n_inst = n_inst;
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
  // scratch: keys, keys_tmp (u64), vals, vals_tmp, bits (u32), hist, tiles, maxdelta
  const int ntiles_rs = (int)((K + RS_TILE - 1) / RS_TILE), ntiles_xs = (int)((K + XS_TILE - 1) / XS_TILE);
  size_t bytes = (size_t)K * (8 + 8 + 4 + 4 + 4) + (size_t)256 * ntiles_rs * 4 + (size_t)ntiles_xs * 4 + SG_MAXINST * 8 + 8 * 256 * 4 + 1024;
  void* scratch;
  int rc = sg_arena(ctx, bytes, &scratch);
  if (rc) return fail(rc);
  char* p = (char*)scratch;
  uint64_t* keys = (uint64_t*)p; p += K * 8;
  uint64_t* keys_tmp = (uint64_t*)p; p += K * 8;
  unsigned long long* maxdelta = (unsigned long long*)p; p += SG_MAXINST * 8;
  uint32_t* vals = (uint32_t*)p; p += K * 4;
  uint32_t* vals_tmp = (uint32_t*)p; p += K * 4;
  uint32_t* bits = (uint32_t*)p; p += K * 4;
  uint32_t* hist = (uint32_t*)p; p += (size_t)256 * ntiles_rs * 4;
  uint32_t* gcnt = (uint32_t*)p; p += 8 * 256 * 4;
  uint32_t* tiles = (uint32_t*)p;
  cudaStream_t st = ctx->stream;
  cudaMemsetAsync(ctx->d_flags, 0, sizeof(int), st);
  cudaMemsetAsync(maxdelta, 0, SG_MAXINST * 8, st);
  sg_launch_begin(ctx, KID_EV_INIT);
  k_ev_init<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, ts, te, inst, n_inst, keys, vals, ctx->d_flags, maxdelta);
  sg_launch_end(ctx);
  rc = sg_sort_pairs(ctx, keys, vals, keys_tmp, vals_tmp, K, hist, gcnt);
  if (rc) return fail(rc);
  sg_launch_begin(ctx, KID_EV_GATHER);
  k_ev_gather<<<(unsigned)((K + 255) / 256), 256, 0, st>>>(K, vals, ts, te, inst, n_inst, ev->t, ev->delta, ev->obs, bits);
  sg_launch_end(ctx);
  sg_launch_begin(ctx, KID_XS_REDUCE);
  k_xs_reduce<<<ntiles_xs, 256, 0, st>>>(bits, K, tiles);
  sg_launch_end(ctx);
  sg_launch_begin(ctx, KID_XS_TILES);
  k_xs_tiles<<<1, 32, 0, st>>>(tiles, ntiles_xs);
  sg_launch_end(ctx);
  sg_launch_begin(ctx, KID_EV_FINAL);
  k_ev_final<<<ntiles_xs, 32, 0, st>>>(K, bits, tiles, vals, ev->t, n_inst, ev->meta, ev->dt, ctx->d_flags);
  sg_launch_end(ctx);
  int flags = 0;
  unsigned long long md[SG_MAXINST];
  double tfl[2];
  if (cudaMemcpyAsync(&flags, ctx->d_flags, sizeof(int), cudaMemcpyDeviceToHost, st) ||
      cudaMemcpyAsync(md, maxdelta, sizeof(md), cudaMemcpyDeviceToHost, st) ||
      cudaMemcpyAsync(&tfl[0], ev->t, 8, cudaMemcpyDeviceToHost, st) ||
      cudaMemcpyAsync(&tfl[1], ev->t + (K - 1), 8, cudaMemcpyDeviceToHost, st) || cudaStreamSynchronize(st)) {
    ctx->err = std::string("build_events: ") + cudaGetErrorString(cudaGetLastError());
    return fail(SMOLGP_ECUDA);
  }
  if (flags & EVF_BADTIME) { ctx->err = "build_events: non-finite time or t_end <= t_start"; return fail(SMOLGP_EINVAL); }
  if (flags & EVF_BADINST) { ctx->err = "build_events: instrument index out of range"; return fail(SMOLGP_EINVAL); }
  if (flags & EVF_OVERLAP) { ctx->err = "build_events: an instrument overlaps itself (P:464)"; return fail(SMOLGP_EOVERLAP); }
  for (int q = 0; q < SG_MAXINST; ++q) {
    double dmax;
    memcpy(&dmax, &md[q], 8);
    int e = 0;
    if (q < n_inst && dmax > 0) frexp(dmax, &e); // dmax = f 2^e, f in [0.5, 1)
    ev->tau[q] = (q < n_inst && dmax > 0) ? ldexp(1.0, e) : 1.0; // power of two >= the longest exposure
  }
  ev->t_first = tfl[0]; ev->t_last = tfl[1];
  *out = ev;
  return SMOLGP_OK;
}

extern "C" int smolgp_build_events(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                                   const int32_t* instrument, int32_t n_inst, smolgp_events** out) {
  return build_events_impl(ctx, N, t_start, t_end, instrument, n_inst, out);
}

extern "C" int smolgp_build_events_host(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                                        const int32_t* instrument, int32_t n_inst, smolgp_events** out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (N <= 0 || !t_start || !t_end || !instrument) { ctx->err = "build_events_host: bad argument"; return SMOLGP_EINVAL; }
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
