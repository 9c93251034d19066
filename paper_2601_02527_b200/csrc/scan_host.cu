#include <stddef.h>
#include <stdio.h>

#include "jit.h"
#include "scan_plan.h"
// scan_host.cu -- host orchestration of the scan kernels (level plan, workspace carving, launches).
// Included at the end of scan.cu (same translation unit as the kernels it launches).

struct LevelPlan {
  int T;                // number of dense levels (0 = single chunk per series)
  int64_t cnt[40];      // cnt[l] = elements per series at level l (l = 1..T)
};

static int pick_lanes(const smolgp_ctx* ctx, int n) {
  const int need = n + 1 <= 8 ? 8 : (n + 1 <= 16 ? 16 : 32); // one lane per column of [X | x]
  if ((ctx->opt_lanes == 8 || ctx->opt_lanes == 16 || ctx->opt_lanes == 32) && ctx->opt_lanes >= need) return (int)ctx->opt_lanes;
  return need;
}

// ---- which level-0 (chunk) kernels run ---------------------------------------------------------------
// Run-time specialised kernels (jit.cu): always when asked for; by default from 1e5 events per call, or once the
// same structure has been evaluated a few dozen times (tiered: sg_jit_hot).  The one-off compilation (a few
// seconds per model structure) is cached in the ctx.  A specialised module holds the REGISTER-RESIDENT
// k_fold0 / k_down0 (chunk_reg.cuh) when the state fits the register file (n <= SG_REG_NMAX), else the
// shared-memory ones with n as a constant.
#define SG_REG_NMAX 24
struct L0Plan {
  const SgJitKernels* jk; // nullptr: the statically compiled generic kernels
  SgJitCfg cfg;
};

// lanes x columns-per-lane of the register-resident k_down0: G * CPL >= n + 1 with the least idle slots, at most
// 63 state doubles per lane; ties go to fewer columns per lane (register pressure)
static void pick_reg_shape(int n, int max_doubles, int mats, int* G, int* CPL) {
  int bestG = 32, bestC = 1, bestW = 1 << 30;
  for (int c = 1; c <= 3; ++c) {
    if (c > 1 && mats * c * n > max_doubles) break;
    for (int gsz = 4; gsz <= 32; gsz *= 2) {
      if (gsz * c < n + 1) continue;
      const int waste = gsz * c - (n + 1);
      if (waste < bestW) { bestW = waste; bestG = gsz; bestC = c; }
      break;
    }
  }
  *G = bestG; *CPL = bestC;
}

static SgJitCfg make_cfg(smolgp_ctx* ctx, const Tab& T, int G) {
  SgJitCfg c;
  c.G = G; c.LD = (T.n + 1) | 1; // the specialised shared-memory kernels take the tightest odd stride
  c.reg = (T.n <= SG_REG_NMAX && ctx->opt_reg >= 0) ? 1 : 0;
  // one column per lane for both kernels: measured on config 3 (profiles/r02_sweeps.md), more columns per lane lose
  // more to the smaller number of resident warps than they gain from the denser packing (the chunk count is bound
  // by the dense levels, so it cannot grow with the packing); "cpl" overrides k_down0's shape for sweeps
  pick_reg_shape(T.n, 0, 1, &c.rG, &c.rCPL);
  pick_reg_shape(T.n, 0, 3, &c.fG, &c.fCPL);
  if (ctx->opt_rcpl >= 1 && ctx->opt_rcpl <= 3) { // tuning override: columns per lane of k_down0
    c.rCPL = (int)ctx->opt_rcpl;
    c.rG = 4;
    while (c.rG * c.rCPL < T.n + 1) c.rG *= 2;
  }
  c.dot2 = (ctx->opt_dot2 >= 0 && ctx->opt_dot2 <= 3) ? (int)ctx->opt_dot2 : 1;
  c.rMinB = (ctx->opt_rminb > 0) ? (int)ctx->opt_rminb : 8;
  c.fMinB = (ctx->opt_fminb > 0) ? (int)ctx->opt_fminb : 8;
  if (!c.reg) { c.rG = c.rCPL = c.fG = c.fCPL = c.rMinB = c.fMinB = 0; }
  return c;
}

static L0Plan plan_l0(smolgp_ctx* ctx, const Tab& T, int G, int64_t events, bool count) {
  L0Plan p;
  p.cfg = make_cfg(ctx, T, G);
  p.jk = nullptr;
  bool want;
  if (ctx->opt_jit != 0) want = ctx->opt_jit > 0;
  else {
    const bool hot = sg_jit_hot(ctx, T, p.cfg, count); // counted once per API call (sg_run_scan)
    want = events >= 100000 || hot || sg_jit_prebuilt(ctx, T, p.cfg); // an ahead-of-time module costs nothing to use
  }
  if (want) p.jk = sg_jit_get(ctx, T, p.cfg);
  return p;
}
static int l0_ld(const L0Plan& p, int n) { return p.jk ? p.cfg.LD : chunk_ld(n); } // row stride of the shared-memory kernels in effect

static int launch_jit(smolgp_ctx* ctx, cudaKernel_t k, int kid, unsigned blocks, unsigned threads, size_t smem, const void* params) {
  SG_CUDA(ctx, cudaFuncSetAttribute((const void*)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  void* args[1] = {const_cast<void*>(params)};
  sg_launch_begin(ctx, kid);
  cudaError_t e = cudaLaunchKernel((const void*)k, dim3(blocks), dim3(threads), args, smem, ctx->stream);
  sg_launch_end(ctx);
  SG_CUDA(ctx, e);
  return SMOLGP_OK;
}

// register-resident kernels: one warp per CTA, 32 / G chunks per warp
static size_t reg_cta_smem(const ModelDev* hm, int G) {
  return ((size_t)reg_czs(hm->n_inst, hm->nblk) + (size_t)(32 / G) * reg_group_doubles(hm->n, hm->disc_stride)) * 8;
}
// chunks resident per SM (shared memory, registers, 32 CTAs)
static int reg_groups_per_sm(const ModelDev* hm, int G, int regs) {
  const size_t cta = reg_cta_smem(hm, G);
  int ctas = (int)((228 * 1024) / (cta + 1024));
  if (ctas > 32) ctas = 32;
  const int by_regs = 65536 / (((regs + 7) / 8 * 8) * 32);
  if (ctas > by_regs) ctas = by_regs;
  if (ctas < 1) ctas = 1;
  return ctas * (32 / G);
}

template <int G, int LD>
static int launch_level0(smolgp_ctx* ctx, const ScanDev& P, const ModelDev* hm, bool fold) {
  const int n = hm->n;
  const int gd = fold ? fold0_group_doubles(n, LD, hm->disc_stride, hm->nblk, G) : down0_group_doubles(n, LD, hm->disc_stride, hm->nblk, G);
  const size_t per_group = (size_t)gd * 8;
  const int gpc = groups_per_cta(per_group, G);
  const size_t smem = per_group * gpc;
  if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  const int64_t groups = P.batch * P.c1;
  const unsigned blocks = (unsigned)((groups + gpc - 1) / gpc);
  if (fold) {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_fold0<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_FOLD0);
    k_fold0<G, LD><<<blocks, gpc * G, smem, ctx->stream>>>(P);
  } else {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_down0<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_DOWN0);
    k_down0<G, LD><<<blocks, gpc * G, smem, ctx->stream>>>(P);
  }
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}

static int launch_level0_any(smolgp_ctx* ctx, const ScanDev& P, const ModelDev* hm, bool fold, int G, const L0Plan& lp) {
  const SgJitKernels* jk = lp.jk;
  const int64_t groups = P.batch * P.c1;
  if (jk && jk->cfg.reg) {
    const int rg = fold ? jk->cfg.fG : jk->cfg.rG, gpc = 32 / rg;
    const size_t smem = reg_cta_smem(hm, rg);
    if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
    return launch_jit(ctx, fold ? jk->fold0 : jk->down0, fold ? KID_FOLD0 : KID_DOWN0, (unsigned)((groups + gpc - 1) / gpc), 32, smem, &P);
  }
  const int LD = l0_ld(lp, hm->n);
  if (jk) {
    const int n = hm->n;
    const int gd = fold ? fold0_group_doubles(n, LD, hm->disc_stride, hm->nblk, G) : down0_group_doubles(n, LD, hm->disc_stride, hm->nblk, G);
    const size_t per_group = (size_t)gd * 8;
    const int gpc = groups_per_cta(per_group, G);
    const size_t smem = per_group * gpc;
    if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
    return launch_jit(ctx, fold ? jk->fold0 : jk->down0, fold ? KID_FOLD0 : KID_DOWN0, (unsigned)((groups + gpc - 1) / gpc), gpc * G, smem, &P);
  }
#define SG_CALL_L0(g_, ld_) return launch_level0<g_, ld_>(ctx, P, hm, fold)
  SG_DISPATCH_GL(G, LD, SG_CALL_L0);
#undef SG_CALL_L0
  return SMOLGP_EUNSUPPORTED;
}

static int launch_dense(smolgp_ctx* ctx, const DenseArgs& D, int n, const SgJitKernels* jk, bool fold) {
  const int gd = fold ? foldD_group_doubles(n) : downD_group_doubles(n);
  const size_t smem = (size_t)gd * 8;
  if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  const int64_t groups = D.batch * D.cout;
  dim3 grid((unsigned)groups, fold ? 1 : (D.want_suffix ? 2 : 1));
  if (jk) {
    cudaKernel_t k = fold ? jk->foldD : jk->downD;
    SG_CUDA(ctx, cudaFuncSetAttribute((const void*)k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    void* args[1] = {const_cast<DenseArgs*>(&D)};
    sg_launch_begin(ctx, fold ? KID_FOLDD : KID_DOWND);
    cudaError_t e = cudaLaunchKernel((const void*)k, grid, dim3(SG_DENSE_NT), args, smem, ctx->stream);
    sg_launch_end(ctx);
    SG_CUDA(ctx, e);
    return SMOLGP_OK;
  }
  if (fold) {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_foldD<SG_DENSE_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_FOLDD);
    k_foldD<SG_DENSE_NT><<<grid, SG_DENSE_NT, smem, ctx->stream>>>(D);
  } else {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_downD<SG_DENSE_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_DOWND);
    k_downD<SG_DENSE_NT><<<grid, SG_DENSE_NT, smem, ctx->stream>>>(D);
  }
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}

int sg_run_scan(smolgp_ctx* ctx, const ScanArgs& a) {
  const ModelDev* hm = a.h_model;
  const int n = hm->n;
  const int64_t K = a.ev->K, N = a.ev->N, batch = a.batch;
  const int G = pick_lanes(ctx, n);
  Tab T0;
  tab_build(hm, &T0);
  const bool sq = hm->sqrt_form != 0; // square-root form: the generic factor-form kernels (chunk_sqrt.cuh, dense_sqrt.cuh)
  L0Plan lp;
  if (sq) { lp.jk = nullptr; lp.cfg = make_cfg(ctx, T0, G); }
  else lp = plan_l0(ctx, T0, G, batch * K, true); // specialised kernels for this model's structure, or the generic ones
  const SgJitKernels* jk0 = lp.jk;
  const bool reg = jk0 && jk0->cfg.reg;
  const int ld0 = l0_ld(lp, n);
  const int Gd = reg ? jk0->cfg.rG : G; // lanes per chunk of k_down0
  int g = (ctx->opt_group >= 2) ? (int)ctx->opt_group : 0; // 0: automatic, set once the chunk count is known

  // chunk length: enough chunks to fill the machine about twice, within [16, 512]; a batch that
  // already fills it runs one chunk per series (the sequential filter, row a8)
  int64_t Lc = ctx->opt_chunk;
  if (Lc <= 0) {
    // one full wave: as many chunks as groups can be resident at once (equal work per chunk, no tail);
    // a batch that already fills the machine runs one chunk per series (the sequential filter, row a8)
    int per_sm = 1, per_sm_f = 1;
    if (reg) {
      per_sm = reg_groups_per_sm(hm, jk0->cfg.rG, jk0->regs_down0);
      per_sm_f = reg_groups_per_sm(hm, jk0->cfg.fG, jk0->regs_fold0);
    } else if (sq) {
      groups_per_cta((size_t)sqrt_group_doubles(n, chunk_ld(n), hm->disc_stride, hm->nblk, G) * 8, G, &per_sm);
      groups_per_cta((size_t)fold0s_group_doubles(n, chunk_ld(n), hm->disc_stride, hm->nblk, G) * 8, G, &per_sm_f);
    } else {
      groups_per_cta((size_t)down0_group_doubles(n, ld0, hm->disc_stride, hm->nblk, G) * 8, G, &per_sm);
      groups_per_cta((size_t)fold0_group_doubles(n, ld0, hm->disc_stride, hm->nblk, G) * 8, G, &per_sm_f);
    }
    if (per_sm_f < per_sm) per_sm = per_sm_f;
    const int64_t resident = (int64_t)ctx->sm_count * per_sm;
    // measured on config 5 (profiles/r01_sweeps.md): once the batch alone gives every SM >= 4 warps, one
    // chunk per series wins, because chunking costs the extra fold pass (~ +70 % arithmetic)
    if (batch >= resident || batch * Gd >= (int64_t)ctx->sm_count * 4 * 32) Lc = K;
    else {
      const int64_t per_series = (resident + batch - 1) / batch; // chunks per series
      Lc = (K + per_series - 1) / per_series;
      // floor of 16 events per chunk (below it the dense levels cost more than the chunks save: config 2),
      // relaxed down to 4 for series so short that 16 would leave most SMs idle (config 1)
      int64_t lc_min = (batch * K) / (2 * (int64_t)ctx->sm_count);
      lc_min = lc_min < 4 ? 4 : (lc_min > 16 ? 16 : lc_min);
      if (Lc < lc_min) Lc = lc_min;
    }
  }
  if (Lc > K) Lc = K;
  if (Lc < 2) Lc = 2;
  LevelPlan pl;
  pl.T = 0;
  const int64_t c1 = (K + Lc - 1) / Lc;
  // measured (profiles/r01_sweeps.md): fan-in 2-4 is a flat optimum; 2 where a combine is long (n >= 12:
  // the chain length matters), 4 where it is short and the launches dominate
  if (g == 0) g = (n >= 12) ? 2 : 4;
  if (c1 > 1) {
    pl.T = 1;
    pl.cnt[1] = c1;
    // the tree stops once a level holds <= gtop elements: the top down-sweep walks them sequentially in one
    // CTA per direction.  A level costs two latency-bound launches, a step of the walk about one; measured
    // (profiles/r01_sweeps.md, sweep "top"): 3-8 is a flat optimum at n = 21 / 17, 8-16 for short series of small n
    int gtop = (ctx->opt_top >= 2) ? (int)ctx->opt_top : ((n >= 12) ? 4 : 8);
    if (gtop < g) gtop = g;
    while (pl.cnt[pl.T] > gtop) { pl.cnt[pl.T + 1] = (pl.cnt[pl.T] + g - 1) / g; pl.T++; }
  }
  const int es = elem_size(n), ss = state_size(n);
  // workspace
  size_t bytes = 256;
  auto add = [&](size_t b) { size_t o = bytes; bytes += (b + 255) / 256 * 256; return o; };
  size_t oE[40], oPRE[40], oSUF[40];
  for (int l = 1; l <= pl.T; ++l) {
    oE[l] = add((size_t)batch * pl.cnt[l] * es * 8);
    oPRE[l] = add((size_t)batch * pl.cnt[l] * ss * 8);
    oSUF[l] = a.want_smooth ? add((size_t)batch * pl.cnt[l] * ss * 8) : 0;
  }
  const size_t oX = a.want_smooth ? add((size_t)batch * N * kbuf_stride(n) * 8) : 0;
  const bool use_adj = reg && pl.T && a.want_smooth; // the register k_down0 takes the chunk-end adjoint from k_adjD
  const size_t oADJ = use_adj ? add((size_t)batch * c1 * ss * 8) : 0;
  const size_t oLL = add((size_t)batch * c1 * 8);
  void* ws;
  int rc = sg_arena(ctx, bytes, &ws);
  if (rc) return rc;
  char* w = (char*)ws;

  ScanDev P;
  P.T = T0;
  P.p0 = (const double*)((const char*)a.d_model + offsetof(ModelDev, p0)); P.disc = a.disc; P.dt = a.ev->dt; P.delta = a.ev->delta; P.meta = a.ev->meta; P.obs = a.ev->obs;
  P.y = a.y; P.sigma = a.sigma; P.amp = a.amp; P.K = K; P.N = N; P.batch = batch; P.Lc = (int)Lc; P.c1 = c1;
  P.E1 = pl.T ? (double*)(w + oE[1]) : nullptr;
  P.PRE1 = pl.T ? (const double*)(w + oPRE[1]) : nullptr;
  P.SUF1 = (pl.T && a.want_smooth) ? (const double*)(w + oSUF[1]) : nullptr;
  P.kbuf = a.want_smooth ? (double*)(w + oX) : nullptr;
  P.llpart = (double*)(w + oLL);
  P.mean = a.mean; P.var = a.var; P.flags = ctx->d_flags; P.want_smooth = a.want_smooth;
  P.fstate = a.fstate; P.binfo = a.binfo;
  P.ADJ1 = use_adj ? (const double*)(w + oADJ) : nullptr;

  if (pl.T) {
    rc = sq ? sg_launch_sqrt_chunk(ctx, P, hm, G, true) : launch_level0_any(ctx, P, hm, true, G, lp);
    if (rc) return rc;
    for (int l = 1; l < pl.T; ++l) {
      DenseArgs D = {};
      D.n = n; D.p0 = (const double*)((const char*)a.d_model + offsetof(ModelDev, p0)); D.Ein = (const double*)(w + oE[l]); D.Eout = (double*)(w + oE[l + 1]);
      D.cin = pl.cnt[l]; D.cout = pl.cnt[l + 1]; D.batch = batch; D.g = g;
      rc = sq ? sg_launch_sqrt_dense(ctx, D, n, true) : launch_dense(ctx, D, n, jk0, true);
      if (rc) return rc;
    }
    for (int l = pl.T; l >= 1; --l) {
      DenseArgs D = {};
      D.n = n; D.p0 = (const double*)((const char*)a.d_model + offsetof(ModelDev, p0)); D.Ein = (const double*)(w + oE[l]); D.cin = pl.cnt[l]; D.batch = batch;
      D.want_suffix = a.want_smooth;
      if (l == pl.T) { D.cout = 1; D.g = (int)pl.cnt[l]; D.PREup = nullptr; D.SUFup = nullptr; }
      else { D.cout = pl.cnt[l + 1]; D.g = g; D.PREup = (const double*)(w + oPRE[l + 1]); D.SUFup = a.want_smooth ? (const double*)(w + oSUF[l + 1]) : nullptr; }
      D.PRE = (double*)(w + oPRE[l]); D.SUF = a.want_smooth ? (double*)(w + oSUF[l]) : nullptr;
      rc = sq ? sg_launch_sqrt_dense(ctx, D, n, false) : launch_dense(ctx, D, n, jk0, false);
      if (rc) return rc;
    }
  }
  if (use_adj) {
    AdjArgs A;
    A.n = n; A.PRE = P.PRE1; A.SUF = P.SUF1; A.ADJ = (double*)(w + oADJ); A.c1 = c1; A.batch = batch;
    const size_t smem = (size_t)adjD_group_doubles(n) * 8;
    SG_CUDA(ctx, cudaFuncSetAttribute((const void*)jk0->adjD, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    void* args[1] = {&A};
    sg_launch_begin(ctx, KID_DOWND); // accounted with the dense down-sweep
    cudaError_t e = cudaLaunchKernel((const void*)jk0->adjD, dim3((unsigned)(batch * c1)), dim3(SG_DENSE_NT), args, smem, ctx->stream);
    sg_launch_end(ctx);
    SG_CUDA(ctx, e);
  }
  rc = sq ? sg_launch_sqrt_chunk(ctx, P, hm, G, false) : launch_level0_any(ctx, P, hm, false, G, lp);
  if (rc) return rc;
  {
    char buf[256];
    snprintf(buf, sizeof buf, "n=%d batch=%lld K=%lld chunk=%lld chunks=%lld levels=%d fanin=%d lanes=%d cpl=%d fold_lanes=%d jit=%d kernels=%s regs=%d/%d prebuilt=%d form=%s", n,
             (long long)batch, (long long)K, (long long)Lc, (long long)c1, pl.T, g, Gd, reg ? jk0->cfg.rCPL : 1, reg ? jk0->cfg.fG : G,
             jk0 ? 1 : 0, reg ? "reg" : "smem", jk0 ? jk0->regs_fold0 : 0, jk0 ? jk0->regs_down0 : 0, jk0 ? jk0->prebuilt : 0, sq ? "sqrt" : "cov");
    ctx->plan = buf;
  }
  if (a.loglik) {
    const int wpb = 4;
    sg_launch_begin(ctx, KID_LL_REDUCE);
    k_ll_reduce<<<(unsigned)((batch + wpb - 1) / wpb), wpb * 32, 0, ctx->stream>>>(P.llpart, c1, batch, N, a.amp, a.loglik, ctx->d_flags);
    sg_launch_end(ctx);
    SG_CUDA(ctx, cudaGetLastError());
  }
  return SMOLGP_OK;
}

template <int G, int LD>
static int launch_query(smolgp_ctx* ctx, const QueryDev& Q, const ModelDev* hm) {
  const size_t per_group = (size_t)query_group_doubles(hm->n, LD, hm->disc_stride, hm->nblk, G) * 8;
  const int gpc = groups_per_cta(per_group, G);
  const size_t smem = per_group * gpc;
  if (smem > ctx->smem_optin) { ctx->err = "query: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  const int64_t groups = Q.batch * Q.Mq;
  SG_CUDA(ctx, cudaFuncSetAttribute(k_query<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  sg_launch_begin(ctx, KID_QUERY);
  k_query<G, LD><<<(unsigned)((groups + gpc - 1) / gpc), gpc * G, smem, ctx->stream>>>(Q);
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}

// Row a7.  Scratch (kp, dtq, discq) comes from the arena: the scan's workspace is dead by now (stream order),
// fstate/binfo live outside it.  The queries are processed in slices so that the scratch (two discretisation
// records per query) stays below SG_QUERY_SCRATCH bytes whatever M is (M = 100 N in the paper's third benchmark
// column, would otherwise need 2 M records: 29 GB on config 3).
#define SG_QUERY_SCRATCH ((size_t)256 << 20)
int sg_run_query(smolgp_ctx* ctx, const QueryArgs& a) {
  const ModelDev* hm = a.h_model;
  const int n = hm->n;
  const size_t per_query = (size_t)2 * hm->disc_stride * 8 + 24;
  int64_t slice = (int64_t)(SG_QUERY_SCRATCH / per_query);
  if (slice < 4096) slice = 4096;
  if (slice > a.M) slice = a.M;
  const size_t o_kp = 0, o_dt = ((size_t)slice * 8 + 255) / 256 * 256, o_disc = o_dt + ((size_t)2 * slice * 8 + 255) / 256 * 256;
  void* ws;
  int rc = sg_arena(ctx, o_disc + (size_t)2 * slice * hm->disc_stride * 8, &ws);
  if (rc) return rc;
  int64_t* kp = (int64_t*)((char*)ws + o_kp);
  double* dtq = (double*)((char*)ws + o_dt);
  double* discq = (double*)((char*)ws + o_disc);
  QueryDev Q;
  tab_build(hm, &Q.T);
  Q.p0 = (const double*)((const char*)a.d_model + offsetof(ModelDev, p0)); Q.discq = discq; Q.kp = kp; Q.meta = a.ev->meta; Q.fstate = a.fstate; Q.binfo = a.binfo; Q.amp = a.amp;
  Q.K = a.ev->K; Q.batch = a.batch; Q.qinst = a.qinst; Q.mean = a.mean; Q.var = a.var; Q.flags = ctx->d_flags; Q.Mtot = a.M;
  const int G = pick_lanes(ctx, n);
  const bool sq = hm->sqrt_form != 0;
  L0Plan lp;
  if (sq) { lp.jk = nullptr; lp.cfg = make_cfg(ctx, Q.T, G); }
  else lp = plan_l0(ctx, Q.T, G, Q.batch * Q.K, false);
  const SgJitKernels* jk = lp.jk;
  const int LD = l0_ld(lp, n);
  for (int64_t q0 = 0; q0 < a.M; q0 += slice) {
    const int64_t M = (a.M - q0 < slice) ? a.M - q0 : slice;
    Q.Mq = M; Q.q0 = q0;
    sg_launch_begin(ctx, KID_QLOCATE);
    k_query_locate<<<(unsigned)((M + 127) / 128), 128, 0, ctx->stream>>>(M, a.tq + q0, a.ev->K, a.ev->t, kp, dtq);
    sg_launch_end(ctx);
    SG_CUDA(ctx, cudaGetLastError());
    rc = sg_launch_disc(ctx, a.d_model, hm, dtq, 2 * M, discq);
    if (rc) return rc;
    if (sq) rc = sg_launch_sqrt_query(ctx, Q, hm, G);
    else if (jk) {
      const size_t per_group = (size_t)query_group_doubles(n, LD, hm->disc_stride, hm->nblk, G) * 8;
      const int gpc = groups_per_cta(per_group, G);
      const int64_t groups = Q.batch * Q.Mq;
      rc = launch_jit(ctx, jk->query, KID_QUERY, (unsigned)((groups + gpc - 1) / gpc), gpc * G, per_group * gpc, &Q);
    } else {
#define SG_CALL_Q(g_, ld_) rc = launch_query<g_, ld_>(ctx, Q, hm)
      SG_DISPATCH_GL(G, LD, SG_CALL_Q);
#undef SG_CALL_Q
    }
    if (rc) return rc;
  }
  return SMOLGP_OK;
}
