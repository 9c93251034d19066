// api.cu -- the C ABI of include/smolgp.h: context, workspace, and the entry points that chain
// discretisation (disc.cu) and the scans (scan.cu).  No CPU fallback anywhere: every entry point
// needs a CUDA device and fails with SMOLGP_ECUDA without one.
#include <math.h>
#include <string.h>

#include "common.h"
#include "jit.h"

int sg_arena(smolgp_ctx* ctx, size_t bytes, void** out) {
  if (bytes > ctx->arena_bytes) {
    if (ctx->arena) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->arena); ctx->arena = nullptr; ctx->arena_bytes = 0; }
    size_t want = bytes + bytes / 8;
    if (cudaMalloc(&ctx->arena, want) != cudaSuccess) {
      cudaGetLastError();
      want = bytes;
      if (cudaMalloc(&ctx->arena, want) != cudaSuccess) { cudaGetLastError(); ctx->arena = nullptr; ctx->err = "out of device memory (workspace)"; return SMOLGP_ENOMEM; }
    }
    ctx->arena_bytes = want;
  }
  sg_mem_mark(ctx);
  *out = ctx->arena;
  return SMOLGP_OK;
}

extern "C" int smolgp_create(smolgp_ctx** out, int device, void* cuda_stream) {
  if (!out) return SMOLGP_EINVAL;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return SMOLGP_ECUDA; }
  if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return SMOLGP_ECUDA; }
  smolgp_ctx* c = new smolgp_ctx();
  c->device = device; c->stream = (cudaStream_t)cuda_stream; c->launches = 0; c->prof_on = 0; c->prof_cur = 0;
  c->opt_chunk = 0; c->opt_group = 0; c->opt_top = 0; c->opt_jit = 0; c->opt_reg = 0; c->opt_rcpl = 0; c->opt_rminb = 0; c->opt_fminb = 0; c->opt_dot2 = -1; c->opt_form = 0; c->jit = nullptr; c->opt_lanes = 0; c->arena = nullptr; c->arena_bytes = 0; c->d_flags = nullptr; c->pers = nullptr; c->pers_bytes = 0; c->hmodel = nullptr;
  c->lb_status = nullptr; c->lb_words = 0; c->lb_epoch = 0; c->mem_extra = 0; c->mem_peak = 0;
  // pinned: the per-call model upload is a true asynchronous copy
  if (cudaMallocHost((void**)&c->hmodel, sizeof(ModelDev)) != cudaSuccess) { cudaGetLastError(); delete c; return SMOLGP_ENOMEM; }
  int v = 0;
  cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, device); c->sm_count = v;
  cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device); c->smem_optin = (size_t)v;
  {
    // keep freed stream-ordered allocations in the pool instead of returning them at every synchronise
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
      unsigned long long thr = ~0ull;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
    }
    cudaGetLastError();
  }
  if (cudaMalloc(&c->d_flags, 64) != cudaSuccess) { cudaGetLastError(); cudaFreeHost(c->hmodel); delete c; return SMOLGP_ENOMEM; }
  cudaMemset(c->d_flags, 0, 64);
  *out = c;
  return SMOLGP_OK;
}

extern "C" void smolgp_destroy(smolgp_ctx* ctx) {
  if (!ctx) return;
  cudaSetDevice(ctx->device);
  cudaStreamSynchronize(ctx->stream);
  sg_jit_destroy(ctx);
  cudaFree(ctx->arena);
  cudaFree(ctx->pers);
  cudaFree(ctx->d_flags);
  cudaFree(ctx->lb_status);
  for (auto& r : ctx->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto& e : ctx->evpool) cudaEventDestroy(e);
  cudaFreeHost(ctx->hmodel);
  delete ctx;
}

extern "C" const char* smolgp_last_error(const smolgp_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
extern "C" int64_t smolgp_launch_count(const smolgp_ctx* ctx) { return ctx ? ctx->launches : 0; }

static const char* const KNAMES[KID_COUNT] = {"k_ev_init", "k_rs_pass", "k_ev_final", "k_disc", "k_fold0", "k_foldD",
                                               "k_downD", "k_down0", "k_ll_reduce", "k_query_locate", "k_query"};
static_assert(KID_COUNT == SMOLGP_NKERNELS, "smolgp.h: SMOLGP_NKERNELS out of step with the kernel ids");
extern "C" const char* smolgp_kernel_name(int32_t id) { return (id >= 0 && id < KID_COUNT) ? KNAMES[id] : nullptr; }

extern "C" int smolgp_profile(smolgp_ctx* ctx, int32_t enable) {
  if (!ctx) return SMOLGP_EINVAL;
  for (auto& r : ctx->prof) { ctx->evpool.push_back(r.a); ctx->evpool.push_back(r.b); }
  ctx->prof.clear();
  if (enable < 0 || enable >= 2 + KID_COUNT) return SMOLGP_EINVAL;
  ctx->prof_on = enable;
  return SMOLGP_OK;
}

extern "C" int smolgp_profile_read(smolgp_ctx* ctx, double* ms, int64_t* launches) {
  if (!ctx || !ms || !launches) return SMOLGP_EINVAL;
  SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  for (int i = 0; i < KID_COUNT; ++i) { ms[i] = 0.0; launches[i] = 0; }
  for (auto& r : ctx->prof) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) { ms[r.id] += t; launches[r.id]++; }
    else cudaGetLastError();
    ctx->evpool.push_back(r.a); ctx->evpool.push_back(r.b);
  }
  ctx->prof.clear();
  return SMOLGP_OK;
}

extern "C" const char* smolgp_jit_log(smolgp_ctx* ctx) { return ctx ? sg_jit_log(ctx) : ""; }
extern "C" const char* smolgp_plan_info(const smolgp_ctx* ctx) { return ctx ? ctx->plan.c_str() : ""; }
extern "C" int smolgp_memory_info(smolgp_ctx* ctx, int64_t* current_bytes, int64_t* peak_bytes, int32_t reset_peak) {
  if (!ctx) return SMOLGP_EINVAL;
  if (current_bytes) *current_bytes = (int64_t)sg_mem_now(ctx);
  if (peak_bytes) *peak_bytes = (int64_t)ctx->mem_peak;
  if (reset_peak) ctx->mem_peak = sg_mem_now(ctx);
  return SMOLGP_OK;
}

extern "C" int smolgp_set_option(smolgp_ctx* ctx, const char* name, int64_t value) {
  if (!ctx || !name) return SMOLGP_EINVAL;
  if (!strcmp(name, "chunk")) ctx->opt_chunk = value;
  else if (!strcmp(name, "group")) ctx->opt_group = value;
  else if (!strcmp(name, "top")) ctx->opt_top = value;
  else if (!strcmp(name, "lanes")) ctx->opt_lanes = value;
  else if (!strcmp(name, "jit")) ctx->opt_jit = value;
  else if (!strcmp(name, "reg")) ctx->opt_reg = value;
  else if (!strcmp(name, "cpl")) ctx->opt_rcpl = value;
  else if (!strcmp(name, "rminb")) ctx->opt_rminb = value;
  else if (!strcmp(name, "dot2")) ctx->opt_dot2 = value;
  else if (!strcmp(name, "fminb")) ctx->opt_fminb = value;
  else if (!strcmp(name, "form")) {
    if (value != 0 && value != 1) { ctx->err = "option form: 0 (covariance) or 1 (square-root)"; return SMOLGP_EINVAL; }
    ctx->opt_form = value;
  }
  else { ctx->err = std::string("unknown option ") + name; return SMOLGP_EINVAL; }
  return SMOLGP_OK;
}

// validation of sigma > 0 and amp > 0 happens on the device inside the filter (NUMF_SIGMA / NUMF_AMP flags)
struct QuerySpec { int64_t M = 0; const double* tq = nullptr; int qinst = 0; double* mean = nullptr; double* var = nullptr; };

static int run_path(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                    const double* y, const double* sigma, const double* amp, double* mean, double* var,
                    double* loglik, int want_smooth, const QuerySpec& qs = QuerySpec()) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!ev || !kernel || !y || !sigma || batch <= 0) { ctx->err = "null or empty argument"; return SMOLGP_EINVAL; }
  if (want_smooth && (!mean || !var)) { ctx->err = "condition: mean_obs and var_obs are required"; return SMOLGP_EINVAL; }
  if (!want_smooth && !loglik) { ctx->err = "loglik: output pointer is null"; return SMOLGP_EINVAL; }
  if (ev->device != ctx->device) { ctx->err = "events belong to another device"; return SMOLGP_EINVAL; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  ModelDev& hm = *ctx->hmodel;
  int rc = sg_build_model(ctx, kernel, ev->n_inst, ev->tau, ev->instant, &hm);
  if (rc) return rc;
  hm.sqrt_form = (ctx->opt_form == 1) ? 1 : 0;
  const size_t model_b = (sizeof(ModelDev) + 255) / 256 * 256;
  const size_t disc_b = ((size_t)ev->K * hm.disc_stride * 8 + 255) / 256 * 256;
  if (ctx->pers_bytes < model_b + disc_b) {
    if (ctx->pers) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->pers); ctx->pers = nullptr; ctx->pers_bytes = 0; }
    if (cudaMalloc(&ctx->pers, model_b + disc_b) != cudaSuccess) { cudaGetLastError(); ctx->pers = nullptr; ctx->err = "out of device memory (discretisation)"; return SMOLGP_ENOMEM; }
    ctx->pers_bytes = model_b + disc_b;
  }
  const size_t ev_bytes = (size_t)ev->K * 28; // the caller's event stream: counted with the call that uses it
  sg_mem_mark(ctx, ev_bytes);
  void* pers = ctx->pers;
  ModelDev* dm = (ModelDev*)pers;
  double* disc = (double*)((char*)pers + model_b);
  SG_CUDA(ctx, cudaMemcpyAsync(dm, &hm, sizeof(ModelDev), cudaMemcpyHostToDevice, ctx->stream));
  SG_CUDA(ctx, cudaMemsetAsync(ctx->d_flags, 0, sizeof(int), ctx->stream));
  rc = sg_launch_disc(ctx, dm, &hm, ev->dt, ev->K, disc);
  if (rc) return rc;
  ScanArgs a;
  a.d_model = dm; a.h_model = &hm; a.ev = ev; a.disc = disc; a.batch = batch; a.y = y; a.sigma = sigma; a.amp = amp;
  a.loglik = loglik; a.mean = mean; a.var = var; a.want_smooth = want_smooth;
  a.fstate = a.binfo = nullptr;
  double* qstore = nullptr; // all 2N filtered states and backward informations, only when queries are asked for
  if (qs.M > 0) {
    if (!qs.tq || !qs.mean || !qs.var) { ctx->err = "condition: t_query, mean_query and var_query are required when M > 0"; return SMOLGP_EINVAL; }
    if (qs.qinst < 0 || qs.qinst >= 32) { ctx->err = "condition: query_instrument must be a mask bit in [0, 32)"; return SMOLGP_EINVAL; }
    const size_t one = (size_t)batch * ev->K * (hm.n + hm.n * hm.n) * 8;
    if (cudaMallocAsync(&qstore, 2 * one, ctx->stream) != cudaSuccess) { cudaGetLastError(); ctx->err = "out of device memory (states for query-time prediction)"; return SMOLGP_ENOMEM; }
    a.fstate = qstore; a.binfo = (double*)((char*)qstore + one);
    ctx->mem_extra += 2 * one;
    sg_mem_mark(ctx, ev_bytes);
  }
  rc = sg_run_scan(ctx, a);
  if (rc == SMOLGP_OK && qs.M > 0) {
    QueryArgs q;
    q.d_model = dm; q.h_model = &hm; q.ev = ev; q.batch = batch; q.M = qs.M; q.tq = qs.tq; q.qinst = qs.qinst; q.amp = amp;
    q.fstate = a.fstate; q.binfo = a.binfo; q.mean = qs.mean; q.var = qs.var;
    rc = sg_run_query(ctx, q);
  }
  sg_mem_mark(ctx, ev_bytes);
  if (qstore) ctx->mem_extra -= 2 * (size_t)batch * ev->K * (hm.n + hm.n * hm.n) * 8;
  if (rc) { if (qstore) cudaFreeAsync(qstore, ctx->stream); return rc; }
  int flags = 0;
  cudaError_t ce = cudaMemcpyAsync(&flags, ctx->d_flags, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(ctx->stream);
  if (qstore) cudaFreeAsync(qstore, ctx->stream);
  SG_CUDA(ctx, ce);
  if (flags & NUMF_SIGMA) { ctx->err = "noise_sigma must be finite and > 0 at every exposure"; return SMOLGP_EINVAL; }
  if (flags & NUMF_AMP) { ctx->err = "amp must be finite and > 0 for every series"; return SMOLGP_EINVAL; }
  if (flags) { ctx->err = "non-finite value or non-positive innovation variance (check noise_sigma > 0, amp > 0, finite y)"; return SMOLGP_ENUMERIC; }
  return SMOLGP_OK;
}

extern "C" int smolgp_loglik(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                             const double* y, const double* noise_sigma, const double* amp, double* loglik) {
  return run_path(ctx, ev, kernel, batch, y, noise_sigma, amp, nullptr, nullptr, loglik, 0);
}

extern "C" int smolgp_condition(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                                const double* y, const double* noise_sigma, const double* amp, int64_t M,
                                const double* t_query, int32_t query_instrument, double* mean_obs, double* var_obs,
                                double* mean_query, double* var_query, double* loglik) {
  if (!ctx) return SMOLGP_EINVAL;
  if (M < 0) { ctx->err = "condition: M < 0"; return SMOLGP_EINVAL; }
  QuerySpec qs;
  qs.M = M; qs.tq = t_query; qs.qinst = query_instrument; qs.mean = mean_query; qs.var = var_query;
  return run_path(ctx, ev, kernel, batch, y, noise_sigma, amp, mean_obs, var_obs, loglik, 1, qs);
}

// ---- host-pointer variants: copies inside the call, on the ctx stream -------------------------------
struct HostStage {
  double *y = nullptr, *sigma = nullptr, *amp = nullptr, *mean = nullptr, *var = nullptr, *ll = nullptr;
  double *tq = nullptr, *mq = nullptr, *vq = nullptr;
  cudaStream_t st = 0;
  ~HostStage() { for (double* p : {y, sigma, amp, mean, var, ll, tq, mq, vq}) if (p) cudaFreeAsync(p, st); }
};

static int host_path(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                     const double* y, const double* sigma, const double* amp, double* mean, double* var,
                     double* loglik, int want_smooth, const QuerySpec& hq = QuerySpec()) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!ev || !y || !sigma || batch <= 0) { ctx->err = "null or empty argument"; return SMOLGP_EINVAL; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  const int64_t N = ev->N;
  HostStage s;
  s.st = ctx->stream;
  const size_t bn = (size_t)batch * N * 8;
  auto am = [&](double** p, size_t b) { return cudaMallocAsync(p, b, ctx->stream) != cudaSuccess; };
  if (am(&s.y, bn) || am(&s.sigma, N * 8) || (amp && am(&s.amp, batch * 8)) ||
      (want_smooth && (am(&s.mean, bn) || am(&s.var, bn))) || am(&s.ll, batch * 8)) {
    cudaGetLastError(); ctx->err = "out of device memory (host staging)"; return SMOLGP_ENOMEM;
  }
  cudaStream_t st = ctx->stream;
  QuerySpec qs;
  const size_t bm = (size_t)batch * (hq.M > 0 ? hq.M : 0) * 8;
  if (hq.M > 0) {
    if (!hq.tq || !hq.mean || !hq.var) { ctx->err = "condition: t_query, mean_query and var_query are required when M > 0"; return SMOLGP_EINVAL; }
    if (am(&s.tq, hq.M * 8) || am(&s.mq, bm) || am(&s.vq, bm)) { cudaGetLastError(); ctx->err = "out of device memory (host staging)"; return SMOLGP_ENOMEM; }
    SG_CUDA(ctx, cudaMemcpyAsync(s.tq, hq.tq, hq.M * 8, cudaMemcpyHostToDevice, st));
    qs.M = hq.M; qs.tq = s.tq; qs.qinst = hq.qinst; qs.mean = s.mq; qs.var = s.vq;
  }
  SG_CUDA(ctx, cudaMemcpyAsync(s.y, y, bn, cudaMemcpyHostToDevice, st));
  SG_CUDA(ctx, cudaMemcpyAsync(s.sigma, sigma, N * 8, cudaMemcpyHostToDevice, st));
  if (amp) SG_CUDA(ctx, cudaMemcpyAsync(s.amp, amp, batch * 8, cudaMemcpyHostToDevice, st));
  int rc = run_path(ctx, ev, kernel, batch, s.y, s.sigma, amp ? s.amp : nullptr, s.mean, s.var, s.ll, want_smooth, qs);
  if (rc) return rc;
  if (hq.M > 0) {
    SG_CUDA(ctx, cudaMemcpyAsync(hq.mean, s.mq, bm, cudaMemcpyDeviceToHost, st));
    SG_CUDA(ctx, cudaMemcpyAsync(hq.var, s.vq, bm, cudaMemcpyDeviceToHost, st));
  }
  if (want_smooth) {
    SG_CUDA(ctx, cudaMemcpyAsync(mean, s.mean, bn, cudaMemcpyDeviceToHost, st));
    SG_CUDA(ctx, cudaMemcpyAsync(var, s.var, bn, cudaMemcpyDeviceToHost, st));
  }
  if (loglik) SG_CUDA(ctx, cudaMemcpyAsync(loglik, s.ll, batch * 8, cudaMemcpyDeviceToHost, st));
  SG_CUDA(ctx, cudaStreamSynchronize(st));
  return SMOLGP_OK;
}

extern "C" int smolgp_loglik_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                                  const double* y, const double* noise_sigma, const double* amp, double* loglik) {
  if (ctx && !loglik) { ctx->err = "loglik: output pointer is null"; return SMOLGP_EINVAL; }
  return host_path(ctx, ev, kernel, batch, y, noise_sigma, amp, nullptr, nullptr, loglik, 0);
}

extern "C" int smolgp_condition_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                                     int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                                     int64_t M, const double* t_query, int32_t query_instrument, double* mean_obs,
                                     double* var_obs, double* mean_query, double* var_query, double* loglik) {
  if (!ctx) return SMOLGP_EINVAL;
  if (M < 0) { ctx->err = "condition: M < 0"; return SMOLGP_EINVAL; }
  if (!mean_obs || !var_obs) { ctx->err = "condition: mean_obs and var_obs are required"; return SMOLGP_EINVAL; }
  QuerySpec qs;
  qs.M = M; qs.tq = t_query; qs.qinst = query_instrument; qs.mean = mean_query; qs.var = var_query;
  return host_path(ctx, ev, kernel, batch, y, noise_sigma, amp, mean_obs, var_obs, loglik, 1, qs);
}

// ---- gradient of the log-likelihood w.r.t. the hyper-parameters ---------------
// d loglik / d theta for theta in (sigma, p0, p1, p2) of every component, per series, by Richardson-extrapolated
// central differences IN LOG theta of the exact log-likelihood this library computes (relative error of loglik
// ~1e-15, include/smolgp.h):  with D(h) = (L(theta e^h) - L(theta e^-h)) / 2h,
//   dL/dlog theta = (4 D(h) - D(2h)) / 3 + O(h^4),   dL/dtheta = that / theta.
// Four likelihood evaluations per parameter, all on the device; the event stream and the data stay where they
// are.  (The adjoint form -- one forward and one backward pass for all parameters -- is not built: DESIGN.md 12.)
static int family_params(int family) { // bit i: parameter i of (sigma, p0, p1, p2) is used by the family
  switch (family) {
    case SMOLGP_MATERN32: case SMOLGP_MATERN52: return 0x3;
    case SMOLGP_SHO: return 0x7;
    case SMOLGP_MATERN32_X_PERIODIC: return 0xF;
    default: return 0;
  }
}

static int grad_path(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch, const double* y,
                     const double* sigma, const double* amp, double rel_step, double* loglik_h, double* grad_h) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!ev || !kernel || kernel->n_comp <= 0 || !kernel->comp || !y || !sigma || batch <= 0 || !grad_h) { ctx->err = "loglik_grad: null or empty argument"; return SMOLGP_EINVAL; }
  const double h = (rel_step > 0 && rel_step < 0.1) ? rel_step : 1e-3;
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  double* dll = nullptr;
  if (cudaMallocAsync(&dll, batch * 8, ctx->stream) != cudaSuccess) { cudaGetLastError(); ctx->err = "loglik_grad: out of device memory"; return SMOLGP_ENOMEM; }
  std::vector<smolgp_component> comp(kernel->comp, kernel->comp + kernel->n_comp);
  smolgp_kernel kk; kk.n_comp = kernel->n_comp; kk.comp = comp.data();
  std::vector<double> f[4];
  for (auto& v : f) v.resize(batch);
  auto eval = [&](double* out_h) -> int {
    int rc = run_path(ctx, ev, &kk, batch, y, sigma, amp, nullptr, nullptr, dll, 0); // synchronises the stream
    if (rc) return rc;
    if (cudaMemcpy(out_h, dll, batch * 8, cudaMemcpyDeviceToHost) != cudaSuccess) { ctx->err = "loglik_grad: read-back failed"; cudaGetLastError(); return SMOLGP_ECUDA; }
    return SMOLGP_OK;
  };
  int rc = SMOLGP_OK;
  if (loglik_h) rc = eval(loglik_h);
  for (int c = 0; c < kernel->n_comp && rc == SMOLGP_OK; ++c) {
    const int used = family_params(comp[c].family);
    double* theta[4] = {&comp[c].sigma, &comp[c].p0, &comp[c].p1, &comp[c].p2};
    for (int p = 0; p < 4 && rc == SMOLGP_OK; ++p) {
      double* g = grad_h + ((size_t)c * 4 + p);
      if (!((used >> p) & 1)) { for (int64_t s = 0; s < batch; ++s) g[(size_t)s * kernel->n_comp * 4] = 0.0; continue; }
      const double t0 = *theta[p];
      const double mult[4] = {exp(h), exp(-h), exp(2 * h), exp(-2 * h)};
      for (int e = 0; e < 4 && rc == SMOLGP_OK; ++e) { *theta[p] = t0 * mult[e]; rc = eval(f[e].data()); }
      *theta[p] = t0;
      for (int64_t s = 0; s < batch && rc == SMOLGP_OK; ++s) {
        const double d1 = (f[0][s] - f[1][s]) / (2 * h), d2 = (f[2][s] - f[3][s]) / (4 * h);
        g[(size_t)s * kernel->n_comp * 4] = (4 * d1 - d2) / 3 / t0;
      }
    }
  }
  cudaFreeAsync(dll, ctx->stream);
  return rc;
}

extern "C" int smolgp_loglik_grad(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                                  const double* y, const double* noise_sigma, const double* amp, double rel_step,
                                  double* loglik, double* grad) {
  return grad_path(ctx, ev, kernel, batch, y, noise_sigma, amp, rel_step, loglik, grad);
}

extern "C" int smolgp_loglik_grad_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel, int64_t batch,
                                       const double* y, const double* noise_sigma, const double* amp, double rel_step,
                                       double* loglik, double* grad) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!ev || !y || !noise_sigma || batch <= 0) { ctx->err = "loglik_grad: null or empty argument"; return SMOLGP_EINVAL; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  HostStage s;
  s.st = ctx->stream;
  const int64_t N = ev->N;
  const size_t bn = (size_t)batch * N * 8;
  auto am = [&](double** p, size_t b) { return cudaMallocAsync(p, b, ctx->stream) != cudaSuccess; };
  if (am(&s.y, bn) || am(&s.sigma, N * 8) || (amp && am(&s.amp, batch * 8))) { cudaGetLastError(); ctx->err = "out of device memory (host staging)"; return SMOLGP_ENOMEM; }
  SG_CUDA(ctx, cudaMemcpyAsync(s.y, y, bn, cudaMemcpyHostToDevice, ctx->stream));
  SG_CUDA(ctx, cudaMemcpyAsync(s.sigma, noise_sigma, N * 8, cudaMemcpyHostToDevice, ctx->stream));
  if (amp) SG_CUDA(ctx, cudaMemcpyAsync(s.amp, amp, batch * 8, cudaMemcpyHostToDevice, ctx->stream));
  return grad_path(ctx, ev, kernel, batch, s.y, s.sigma, amp ? s.amp : nullptr, rel_step, loglik, grad);
}

// ---- step a2 alone (tests): A~ and Q~ of one step in raw state units ---------------------------------
extern "C" int smolgp_discretise_host(smolgp_ctx* ctx, const smolgp_kernel* kernel, int32_t n_inst, double dt,
                                      double* A, double* Q, int32_t* n_out) {
  if (!ctx) return SMOLGP_EINVAL;
  if (!A || !Q || !(dt >= 0) || !isfinite(dt)) { ctx->err = "discretise: bad argument"; return SMOLGP_EINVAL; }
  SG_CUDA(ctx, cudaSetDevice(ctx->device));
  ModelDev& hm = *ctx->hmodel;
  double tau[SG_MAXINST];
  for (int q = 0; q < SG_MAXINST; ++q) tau[q] = 1.0;
  int rc = sg_build_model(ctx, kernel, n_inst, tau, 0, &hm);
  if (rc) return rc;
  const int n = hm.n, d = hm.d;
  if (n_out) *n_out = n;
  void* ws;
  const size_t model_b = (sizeof(ModelDev) + 255) / 256 * 256;
  rc = sg_arena(ctx, model_b + 256 + (size_t)hm.disc_stride * 8, &ws);
  if (rc) return rc;
  ModelDev* dm = (ModelDev*)ws;
  double* ddt = (double*)((char*)ws + model_b);
  double* drec = ddt + 32;
  SG_CUDA(ctx, cudaMemcpyAsync(dm, &hm, sizeof(ModelDev), cudaMemcpyHostToDevice, ctx->stream));
  SG_CUDA(ctx, cudaMemcpyAsync(ddt, &dt, 8, cudaMemcpyHostToDevice, ctx->stream));
  rc = sg_launch_disc(ctx, dm, &hm, ddt, 1, drec);
  if (rc) return rc;
  std::vector<double> rec(hm.disc_stride);
  SG_CUDA(ctx, cudaMemcpyAsync(rec.data(), drec, hm.disc_stride * 8, cudaMemcpyDeviceToHost, ctx->stream));
  SG_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // block units -> raw units: x_i = s_i x''_i with s = sigma_b lambda^(derivative order); z = tau z' (tau = 1)
  std::vector<double> sc(n, 1.0);
  const double* sigb = hm.bsig; // sigma_b of every block (model.cu)
  for (int b = 0; b < hm.nblk; ++b) {
    const BlockConst& B = hm.blk[b];
    for (int i = 0; i < B.dim; ++i) {
      const int order = (B.family == BLK_M32ROT) ? i / 2 : i;
      sc[B.off + i] = sigb[b] * pow(B.inv_T, order);
    }
  }
  for (int i = 0; i < n * n; ++i) { A[i] = 0; Q[i] = 0; }
  for (int b = 0; b < hm.nblk; ++b) {
    const BlockConst& B = hm.blk[b];
    const int db = B.dim, o = B.off;
    const double* r = rec.data() + hm.disc_off[b];
    const double Tb = 1.0 / B.inv_T;
    for (int i = 0; i < db; ++i)
      for (int j = 0; j < db; ++j) {
        A[(o + i) * n + o + j] = sc[o + i] * r[i * db + j] / sc[o + j];
        Q[(o + i) * n + o + j] = sc[o + i] * r[db * db + db + i * db + j] * sc[o + j];
      }
    for (int q = 0; q < n_inst; ++q) {
      if (hm.cz[q][b] == 0.0) continue;
      const double c = sigb[b] * Tb; // I = sigma_b T_b I''
      for (int j = 0; j < db; ++j) {
        A[(d + q) * n + o + j] = c * r[db * db + j] / sc[o + j];
        const double v = c * r[2 * db * db + db + j] * sc[o + j];
        Q[(d + q) * n + o + j] = v;
        Q[(o + j) * n + d + q] = v;
      }
      for (int q2 = 0; q2 < n_inst; ++q2)
        if (hm.cz[q2][b] != 0.0) Q[(d + q) * n + d + q2] += c * c * r[2 * db * db + 2 * db];
    }
  }
  for (int q = 0; q < n_inst; ++q) A[(d + q) * n + d + q] = 1.0;
  return SMOLGP_OK;
}
