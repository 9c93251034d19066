/* smolgp.h -- C ABI of the B200-native (sm_100a) integrated-GP state-space library.
 *
 * What it computes: exact Gaussian-process inference for exposure-integrated, possibly
 * overlapping measurements (arXiv:2601.02527) through the augmented linear-Gaussian state-space
 * model of the paper: one integral state z_i per instrument (Eq. 3.17), reset at each
 * exposure start (Eq. 3.11/3.18) and observed as z_i/delta_n at each exposure end
 * (Eq. 3.12).  Inference is the parallel-in-time (associative-scan) Kalman filter and
 * smoother of section 3.4 with the log marginal likelihood of Eq. 2.26.
 * "P:<n>" = line n of the paper text; DESIGN.md lists the readings taken where the
 * text is silent or garbled.
 *
 * Conventions
 *  - Every function returns SMOLGP_OK (0) or a negative smolgp_status; nothing throws, exits or
 *    prints.  smolgp_last_error(ctx) gives a ctx-owned NUL-terminated message for the last failure.
 *  - Array arguments are DEVICE pointers (8-byte aligned, caller-owned, not retained after the
 *    call returns unless stated) in the entry points without suffix, and HOST pointers in the
 *    *_host entry points, which copy in and out on the ctx stream and synchronise before
 *    returning.  Kernel descriptions (smolgp_kernel) are always small HOST structs.
 *  - All times are in one unit (seconds in the shipped workloads); all arithmetic is fp64.
 *  - Outputs are in the caller's exposure order (the order of t_start/t_end), per series.
 *  - Work is enqueued on the ctx stream; the device entry points return after the work is
 *    enqueued except where a status needs a read-back (smolgp_build_events; the numeric flag of
 *    smolgp_loglik/smolgp_condition, which is read after a stream synchronise).
 *  - There is no CPU fallback: without a CUDA device smolgp_create fails with SMOLGP_ECUDA.
 */
#ifndef SMOLGP_H
#define SMOLGP_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  SMOLGP_OK = 0,
  SMOLGP_EINVAL = -1,       /* bad argument: N<=0, non-finite time, t_end<=t_start, instrument out of range, sigma<=0, amp<=0 */
  SMOLGP_EOVERLAP = -2,     /* an instrument overlaps itself (t_n^e > t_{n+1}^s) */
  SMOLGP_EUNSUPPORTED = -3, /* augmented dimension above SMOLGP_MAX_DIM, unknown family, too many instruments */
  SMOLGP_ENOMEM = -4,
  SMOLGP_ECUDA = -5,
  SMOLGP_ENUMERIC = -6      /* a non-finite value or a non-positive innovation variance was met */
} smolgp_status;

#define SMOLGP_MAX_DIM 31  /* max augmented state dimension n = d + N_inst (n + 1 columns, one lane each) */
#define SMOLGP_MAX_INST 16 /* max number of instruments */

/* kernel families (state-space forms: DESIGN.md "Models"; SHO: App. B) */
enum {
  SMOLGP_MATERN32 = 0,           /* p0 = ell                                   d = 2 */
  SMOLGP_MATERN52 = 1,           /* p0 = ell                                   d = 3 */
  SMOLGP_SHO = 2,                /* p0 = omega0 [rad/time], p1 = Q             d = 2 */
  SMOLGP_MATERN32_X_PERIODIC = 3 /* p0 = ell, p1 = period, p2 = ell_periodic, order = J:
                                    Matern-3/2 times the order-J cosine series of the periodic
                                    kernel (products of kernels: App. C.2)  d = 2 + 4J */
};

/* one additive component of the kernel (sums of kernels: App. C.1) */
typedef struct {
  int32_t family;
  int32_t order;      /* J for MATERN32_X_PERIODIC, else ignored */
  uint32_t inst_mask; /* bit i set <=> the component enters instrument i's integrand H_i (Eq. 3.2) */
  double sigma;       /* amplitude: k(0) = sigma^2 (times the series' sum for the periodic product) */
  double p0, p1, p2;
} smolgp_component;

typedef struct {
  int32_t n_comp;
  const smolgp_component* comp; /* host memory */
} smolgp_kernel;

typedef struct smolgp_ctx smolgp_ctx;       /* device id, stream, workspace arena */
typedef struct smolgp_events smolgp_events; /* immutable device-resident event stream */

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (NULL = the legacy
 * default stream); the caller keeps ownership of the stream. */
int smolgp_create(smolgp_ctx** out, int device, void* cuda_stream);
void smolgp_destroy(smolgp_ctx* ctx);
const char* smolgp_last_error(const smolgp_ctx* ctx);

/* Tuning knobs (all optional).  name = "chunk": events per scan chunk at the leaf level
 * (0 = automatic; >= the series length selects the sequential one-group-per-series filter of
 * SURVEY 8(a) row a8); "group": dense-combine fan-in of the upper scan levels (0 = automatic: 2 for n >= 12, else 4);
 * "top": the level tree of the scan stops once a level holds <= top elements, which the top down-sweep
 * walks sequentially (0 = automatic: 4 for n >= 12, else 8; values below the fan-in act as the fan-in);
 * "lanes": threads cooperating on one chunk (0 = automatic; 8, 16 or 32);
 * "jit": run-time specialisation of the chunk kernels for the kernel's structure with NVRTC
 * (0 = automatic: from 1e5 events per call, or after 32 calls with the same structure; 1 = always;
 * -1 = never); "reg": -1 = the specialised chunk kernels in their shared-memory form instead of the register-resident
 * one (default for n <= 24); "cpl": columns of the state per lane of the register-resident k_down0 (0 = automatic, 1-3);
 * "rminb" / "fminb": minimum resident CTAs per SM asked of the two register-resident kernels (caps their registers;
 * 0 = 8); "dot2": which products of the dense levels are compensated (bit 0: those forming a solve's matrix,
 * bit 1: the others; -1 = default 1) -- sweep knobs, see profiles/r02_sweeps.md;
 * "form": 0 = covariance form (default); 1 = SQUARE-ROOT (Cholesky-factor) form of the whole scan, the paper's remedy for
 * the conditioning of the covariance recursions: covariances, informations and adjoint matrices are carried
 * as factors (P = S S^T, J = Z Z^T) and re-triangularised, in the chunk recursions and in the dense combines alike; nothing
 * is subtracted from a covariance, no I + C J is formed or inverted, no product is compensated (csrc/chunk_sqrt.cuh,
 * csrc/dense_sqrt.cuh).  Same inputs, outputs, tolerances and scan plans ("chunk", "group", "top", "lanes"
 * apply); the kernels are the generic shared-memory ones ("jit" / "reg" are ignored), about ten times slower than the
 * covariance form and one to three orders more accurate; query times (M > 0) are served from the stored factors.
 * A structure is compiled once per ctx (a few seconds) and serves every hyper-parameter value; when NVRTC is missing or a
 * compilation fails the generic kernels run and smolgp_jit_log says why. */
int smolgp_set_option(smolgp_ctx* ctx, const char* name, int64_t value);
const char* smolgp_jit_log(smolgp_ctx* ctx);
/* The scan plan of the last smolgp_loglik / smolgp_condition call of this ctx, as a ctx-owned string
 * "n=21 batch=1 K=200000 chunk=136 chunks=1471 levels=10 fanin=2 lanes=8 cpl=3 jit=1 kernels=reg": which kernels
 * ran (jit=1: the run-time specialised ones) and how the events were cut.  For bench.py and the tests. */
const char* smolgp_plan_info(const smolgp_ctx* ctx);
/* Device memory held by the ctx: bytes now, and the high-water mark since creation or the last reset (the
 * workspace arena, the model + discretisation array, the event-build status words and, inside a call, the
 * event stream it was given and the state store of query-time prediction: 2 batch K (n + n^2) doubles
 * "all 2N states").  The per-query scratch of smolgp_condition is bounded (256 MB) whatever M is.  HOST outputs,
 * either may be NULL. */
int smolgp_memory_info(smolgp_ctx* ctx, int64_t* current_bytes, int64_t* peak_bytes, int32_t reset_peak);

/* Step a1.  Turns N exposures [t_start[n], t_end[n]] of instrument
 * instrument[n] in [0, n_inst) into the time-sorted stream of K = 2N events (one reset event per
 * start, one observe event per end).  ORDER OF THE STREAM: by (time, end before start, instrument,
 * exposure index), whatever the order of the input arrays -- ends come before starts at equal times so
 * that back-to-back exposures of one instrument, the Fig. 2 case P:543, are legal; simultaneous events
 * of the same kind are ordered by instrument, then by exposure index (-0.0 and +0.0 are one time).  Device radix sort (stable, least significant digit
 * first: (kind, instrument), then the bytes of the order-preserving 64-bit image of the times; digits on
 * which all keys agree are skipped); the reset/observe flags, the per-event set of idle instruments and
 * the validation that no instrument overlaps itself come from an XOR scan of the instrument bits.  The three inputs are DEVICE pointers; the result
 * is owned by the caller (smolgp_free_events; free it before destroying the ctx whose stream it was
 * allocated on) and can be reused across kernels and data.
 * Errors: EINVAL, EOVERLAP, EUNSUPPORTED (n_inst > SMOLGP_MAX_INST), ENOMEM, ECUDA. */
int smolgp_build_events(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                        const int32_t* instrument, int32_t n_inst, smolgp_events** out);
int smolgp_build_events_host(smolgp_ctx* ctx, int64_t N, const double* t_start, const double* t_end,
                             const int32_t* instrument, int32_t n_inst, smolgp_events** out);
void smolgp_free_events(smolgp_events* ev);

/* Instantaneous data -- the paper's section 2 (Fig. 1, Fig. 4 workloads P:561): y_n is a noisy
 * sample of the latent of instrument instrument[n] AT time t[n], not an exposure average.  The stream has K = N
 * observe events ordered by (time, instrument, sample index); simultaneous samples are legal.  Every other call
 * (smolgp_loglik, smolgp_condition incl. query times) takes the result unchanged: mean_obs / var_obs are then the
 * posterior of the noise-free latent H_i x at the sample times.  Internally the per-instrument state z_i carries
 * H_i x at the instrument's samples instead of an integral, so the kernels are the
 * same.  A data set is either exposure-integrated or instantaneous: the two kinds cannot be mixed in one stream.
 * Errors: EINVAL (N <= 0, non-finite time, instrument out of range), EUNSUPPORTED, ENOMEM, ECUDA. */
int smolgp_build_events_instant(smolgp_ctx* ctx, int64_t N, const double* t, const int32_t* instrument,
                                int32_t n_inst, smolgp_events** out);
int smolgp_build_events_instant_host(smolgp_ctx* ctx, int64_t N, const double* t, const int32_t* instrument,
                                     int32_t n_inst, smolgp_events** out);

/* Step a1 WITHOUT ANY ALLOCATION -- for callers that cannot call cudaMalloc: code under CUDA stream capture, tight
 * serving loops, harnesses that forbid it.  Same kernels, same stream order (the tie rule
 * above) as smolgp_build_events, but
 *   - the sort's scratch (control block, look-back words, two key and two payload buffers) is ONE file-scope device
 *     array of fixed size, smolgp_noalloc_scratch_bytes() = about 6.5 MB, which every GPU that loads the library holds
 *     until exit.  LIMIT: K <= smolgp_noalloc_max_events() = 262144 events, i.e. N <= 131072 exposures (or 262144
 *     instantaneous samples); beyond it the call returns SMOLGP_EUNSUPPORTED and smolgp_noalloc_last_error() says so;
 *   - no ctx, no smolgp_events object: the caller owns the outputs.  All pointers are DEVICE pointers.
 *     inputs  t_start[N], t_end[N] (NULL = instantaneous samples at t_start, K = N), instrument[N] in [0, n_inst);
 *     outputs, each of length K (= 2N, or N): t = event time; dt[k] = t[k] - t[k-1] (dt[0] = 0); delta = length of the
 *             event's exposure (1 for an instantaneous sample); meta = kind | instrument << 1 | zmask << 8 with kind
 *             1 = start/reset, 0 = end/observe, and bit i of zmask set when z_i is zero after the event (instrument i
 *             idle, or the event's own); exposure = index n of the event's exposure;
 *             flags[1] = 0 when the input is valid, else bits 1 (non-finite time or t_end <= t_start), 2 (instrument
 *             out of range), 4 (an instrument overlaps itself) -- the other outputs then mean nothing.  It is
 *             written in stream order like the rest: there is no host read-back and no synchronisation;
 *   - device = CUDA device ordinal (made current), cuda_stream = cudaStream_t (NULL = default stream).
 * The call makes no cudaMalloc / cudaFree / cudaMallocAsync and calls no allocating library routine: one memset of the
 * control block and look-back words (the array keeps the last call's contents), twelve kernel launches, one 4-byte
 * device-to-device copy.  smolgp_noalloc_setup(device) looks the array's address up (once per device; the first call
 * does it if the caller has not -- call it before starting a stream capture).
 * ALL CALLS ON ONE DEVICE SHARE THE ARRAY: calls that overlap on the GPU (two streams, two host threads, two graph
 * launches in flight) race and produce garbage; serialise them.  Calls in one stream are ordered and safe.
 * Errors (return value; text from smolgp_noalloc_last_error(), per host thread): EINVAL (null pointer, N <= 0, device
 * ordinal), EUNSUPPORTED (size above the limit, n_inst > SMOLGP_MAX_INST), ECUDA. */
int smolgp_build_events_noalloc(int32_t device, void* cuda_stream, int64_t N, const double* t_start,
                                const double* t_end, const int32_t* instrument, int32_t n_inst, double* t, double* dt,
                                double* delta, uint32_t* meta, int32_t* exposure, int32_t* flags);
int smolgp_noalloc_setup(int32_t device);
int64_t smolgp_noalloc_max_events(void);
int64_t smolgp_noalloc_scratch_bytes(void);
const char* smolgp_noalloc_last_error(void);

/* Read back the event stream (HOST output arrays of length K = 2N, or N for instantaneous data; any may be NULL): event time,
 * kind (1 = start/reset, 0 = end/observe), instrument, exposure index.  For tests. */
int smolgp_events_export(smolgp_ctx* ctx, const smolgp_events* ev, double* t, int32_t* kind,
                         int32_t* instrument, int32_t* exposure);

/* Steps a2 + a3 + a5 (Eq. 2.17-2.19, 3.7-3.10; Eq. 3.20-3.21 + forward scan; Eq. 2.26).
 * y: [batch][N] data; noise_sigma: [N] per-exposure white-noise standard deviation (> 0);
 * amp: [batch] per-series kernel amplitude scale (k_p = amp_p^2 k) or NULL (= 1);
 * loglik: [batch] output, Eq. 2.26 including the N log(2 pi)/2 constant. */
int smolgp_loglik(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                  int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                  double* loglik);
int smolgp_loglik_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                       int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                       double* loglik);

/* Gradient of Eq. 2.26 w.r.t. the hyper-parameters (its stated use is optimisation / MCMC).  grad is a HOST
 * array [batch][n_comp][4]: d loglik / d (sigma, p0, p1, p2) of every component (0 for a parameter the family does
 * not use); loglik is a HOST array [batch] or NULL; y, noise_sigma, amp as in smolgp_loglik (device pointers; HOST in
 * the _host variant).  Computed by Richardson-extrapolated central differences in log theta of the exact
 * log-likelihood (four evaluations per parameter, relative step rel_step; <= 0 selects 1e-3): relative accuracy
 * ~1e-8 of the gradient's scale.  The one-pass adjoint form is not built. */
int smolgp_loglik_grad(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                       int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                       double rel_step, double* loglik, double* grad);
int smolgp_loglik_grad_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                            int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                            double rel_step, double* loglik, double* grad);

/* Steps a2-a6 (+ a7 when M > 0).  As smolgp_loglik, plus the posterior of the noise-free exposure
 * average at every observation (mean_obs, var_obs: [batch][N]; H~ m^, H~ P^ H~^T of P:460) and,
 * when M > 0, the posterior of the instantaneous latent of instrument query_instrument at the
 * M query times (Algorithm 1; mean_query, var_query: [batch][M]).  loglik may be NULL.
 * query_instrument is a bit of the components' inst_mask: a bit < n_inst selects that instrument's
 * integrand H_q (Eq. 3.2); a bit in [n_inst, 32) is a VIRTUAL instrument that takes no data: setting it
 * on some components and querying it gives the component-wise predictive mean and variance of
 * App. C.3 (H^m of Eq. C13-C14). */
int smolgp_condition(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                     int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                     int64_t M, const double* t_query, int32_t query_instrument,
                     double* mean_obs, double* var_obs, double* mean_query, double* var_query,
                     double* loglik);
int smolgp_condition_host(smolgp_ctx* ctx, const smolgp_events* ev, const smolgp_kernel* kernel,
                          int64_t batch, const double* y, const double* noise_sigma, const double* amp,
                          int64_t M, const double* t_query, int32_t query_instrument,
                          double* mean_obs, double* var_obs, double* mean_query, double* var_query,
                          double* loglik);

/* Step a2 alone, for tests: the augmented transition A~ = [Phi 0; Phi-bar I] and process noise
 * Q~ (Eq. 3.7-3.10; Eq. 3.17-3.19 for several instruments) of one step of length dt,
 * in raw (unscaled) state units, row-major n x n, HOST outputs.  n_out receives n = d + n_inst. */
int smolgp_discretise_host(smolgp_ctx* ctx, const smolgp_kernel* kernel, int32_t n_inst, double dt,
                           double* A, double* Q, int32_t* n_out);

/* Launch accounting for bench.py: number of kernels this ctx has launched so far. */
int64_t smolgp_launch_count(const smolgp_ctx* ctx);

/* Per-kernel device timing for bench.py's roofline block.  smolgp_profile(ctx, 1) starts a window in
 * which every kernel this ctx launches is bracketed by CUDA events on the ctx stream (two event records per
 * launch: about 0.25 ms per step of config 3, so a headline is not timed in this mode);
 * smolgp_profile(ctx, 2 + id) brackets only the launches of kernel id (EINVAL outside [0, SMOLGP_NKERNELS));
 * smolgp_profile_read synchronises the stream, writes the summed milliseconds and launch counts per
 * kernel id (HOST arrays of SMOLGP_NKERNELS entries; names from smolgp_kernel_name) and clears the
 * window; smolgp_profile(ctx, 0) stops.  smolgp_kernel_name returns NULL outside [0, SMOLGP_NKERNELS). */
#define SMOLGP_NKERNELS 11
int smolgp_profile(smolgp_ctx* ctx, int32_t enable);
int smolgp_profile_read(smolgp_ctx* ctx, double* ms, int64_t* launches);
const char* smolgp_kernel_name(int32_t id);

#ifdef __cplusplus
}
#endif
#endif /* SMOLGP_H */
