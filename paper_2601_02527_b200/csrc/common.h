// Internal declarations shared by the translation units of libsmolgp_b200.so (CUDA product path).
// Nothing here is used by, or shared with, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "../../include/smolgp.h"
#include "dev_consts.h"

static_assert(SG_NMAX >= SMOLGP_MAX_DIM + 1 && SG_MAXINST == SMOLGP_MAX_INST, "dev_consts.h out of step with smolgp.h");
#define SG_KT 18     /* Taylor order of the small-step discretisation */
#define SG_BE (SG_MAXBD + 1)

enum { BLK_M32 = 0, BLK_M52 = 1, BLK_SHO = 2, BLK_M32ROT = 3 };

// One block-diagonal block of the base model in its own non-dimensional units ("block units"):
// time in units of T_b (1/lambda or 1/omega0), state x''_i = x_i / (sigma_b lambda^i), so that all
// constants below are O(1).  The block is augmented with its own integral I'' = int H'' x'' dt''
// (Eq. 3.3-3.6): F~'' = [F'' 0; H'' 0], L~ Qc L~^T = [W'' 0; 0 0].
struct BlockConst {
  int family, dim, off; // off = offset of the block inside x
  int sho_case;         // SHO: 0 underdamped (Q > 1/2), 1 critical, 2 overdamped
  double inv_T;         // 1 / T_b
  double rho;           // inf-norm of F~''  (step size control of the Taylor regime)
  double a, b;          // SHO: a = 1/(2Q), b = sqrt(|1 - a^2|);  M32ROT: b = omega'' = j omega_p T_b
  double pinf[SG_MAXBD * SG_MAXBD];             // stationary covariance in block units
  double tayA[SG_KT + 1][SG_BE * SG_BE];        // F~''^k / k!
  double tayQ[SG_KT + 1][SG_BE * SG_BE];        // Gamma_k / k!, Gamma_1 = W~'', Gamma_{k+1} = F~ Gamma_k + Gamma_k F~^T
};

// Whole model, device resident (built on the host by model.cu for each call's kernel).
struct ModelDev {
  int n, d, n_inst, nblk;
  int instant;                     // 1: instantaneous-data mode: the "integral" rows of a record hold H Phi, Q H^T, H Q H^T (disc.cu)
  int sqrt_form;                   // 1: square-root form: a record's (Qxx, q12, q22) slots hold the block's Cholesky factor (Lxx, Lzx, Lzz) (disc.cu, chunk_sqrt.cuh)
  int disc_stride;                 // doubles per event in the discretisation array
  int disc_off[SG_MAXBLK];         // offset of block b inside one event's record
  double cz[SG_MAXINST][SG_MAXBLK]; // c_qb: coupling of block b's integral into z_q (equilibrated units), 0 if masked out
  double tau[SG_MAXINST];          // z_q is carried as z_q / tau_q
  double bsig[SG_MAXBLK];          // amplitude sigma_b of block b (H_b = sigma_b e_0 in block units)
  uint32_t bmask[SG_MAXBLK];       // the component's inst_mask: bit v set <=> block b is in the integrand of (virtual) instrument v
  double p0[SG_NMAX * SG_NMAX];    // prior covariance blkdiag(Pinf'', 0) (Eq. 3.19, reading R6)
  BlockConst blk[SG_MAXBLK];
};

// per-event record layout inside the discretisation array, block b at disc_off[b]:
//   Phi (dim*dim, row-major) | phibar (dim) | Qxx (dim*dim) | q12 (dim) | q22 (1) | pad (1)      [block units]
static inline int disc_block_size(int dim) { return 2 * dim * dim + 2 * dim + 2; } // + 1 pad: every block 16-byte aligned

struct smolgp_events {
  int device;
  int64_t N, K;
  int n_inst;
  int instant;     // 1: instantaneous samples (paper section 2): K = N observe events, z_i carries H_i x at its sample
  double* t;       // [K] event time
  double* dt;      // [K] t_k - t_{k-1}, dt_0 = 0
  double* delta;   // [K] exposure length of the event's exposure
  uint32_t* meta;  // [K]
  int32_t* obs;    // [K] exposure index
  double tau[SG_MAXINST]; // per-instrument power-of-two scale of z (host copy)
  void* base;            // one stream-ordered allocation holds all five arrays
  cudaStream_t stream;   // the ctx stream the allocation is ordered on
  double t_first, t_last;
};

// kernel ids for launch accounting / per-kernel timing (smolgp_profile_read)
enum { KID_EV_INIT = 0, KID_RS_PASS, KID_EV_FINAL, KID_DISC, KID_FOLD0, KID_FOLDD, KID_DOWND, KID_DOWN0, KID_LL_REDUCE,
       KID_QLOCATE, KID_QUERY, KID_COUNT };
struct ProfRec { int id; cudaEvent_t a, b; };

struct smolgp_ctx {
  int device;
  cudaStream_t stream;
  std::string err;
  std::string plan; // smolgp_plan_info
  int64_t launches;
  int prof_on;   // 0 off, 1 every kernel, 2 + id: only kernel id (smolgp_profile)
  int prof_cur;  // the launch in flight is being timed
  std::vector<ProfRec> prof;       // open records of the current profiling window
  std::vector<cudaEvent_t> evpool; // recycled events
  int64_t opt_chunk, opt_group, opt_lanes, opt_top, opt_jit; // opt_jit: 0 automatic, 1 always, -1 never
  int64_t opt_dot2; // -1 default (3)
  int64_t opt_rminb, opt_fminb; // tuning: min CTAs per SM of the register kernels
  int64_t opt_form; // 0 covariance form, 1 square-root (Cholesky-factor) form of the chunk recursions (chunk_sqrt.cuh)
  int64_t opt_reg, opt_rcpl; // opt_reg: -1 = specialised kernels in their shared-memory form; opt_rcpl: columns per lane of the register k_down0 (0 auto)
  void* jit;       // run-time specialised kernels (jit.cu)
  // workspace arena (grown on demand, reused across calls)
  void* arena;
  size_t arena_bytes;
  int* d_flags; // device status word(s)
  void* pers;   // model + discretisation array of the current call (kept across calls)
  size_t pers_bytes;
  ModelDev* hmodel; // host copy of the current model
  int sm_count;
  size_t smem_optin;
  size_t mem_extra;  // stream-ordered allocations alive inside the current call (query state store, host staging)
  size_t mem_peak;   // high-water mark of the device memory this ctx holds (smolgp_memory_info)
  // decoupled look-back words of the event build (events.cu): persistent, told apart by epoch
  unsigned long long* lb_status;
  size_t lb_words;
  uint32_t lb_epoch;
};

// bracket a kernel launch: counts it and, when profiling is on, times it with CUDA events on the ctx stream
static inline void sg_launch_begin(smolgp_ctx* ctx, int id) {
  ctx->launches++;
  ctx->prof_cur = ctx->prof_on == 1 || ctx->prof_on == 2 + id;
  if (!ctx->prof_cur) return;
  ProfRec r; r.id = id;
  cudaEvent_t* e[2] = {&r.a, &r.b};
  for (int i = 0; i < 2; ++i) {
    if (!ctx->evpool.empty()) { *e[i] = ctx->evpool.back(); ctx->evpool.pop_back(); }
    else cudaEventCreate(e[i]);
  }
  cudaEventRecord(r.a, ctx->stream);
  ctx->prof.push_back(r);
}
static inline void sg_launch_end(smolgp_ctx* ctx) {
  if (ctx->prof_cur && !ctx->prof.empty()) cudaEventRecord(ctx->prof.back().b, ctx->stream);
  ctx->prof_cur = 0;
}

#define SG_CUDA(ctx, call)                                                            \
  do {                                                                                \
    cudaError_t e__ = (call);                                                         \
    if (e__ != cudaSuccess) {                                                         \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);               \
      return SMOLGP_ECUDA;                                                            \
    }                                                                                 \
  } while (0)

// model.cu
int sg_build_model(smolgp_ctx* ctx, const smolgp_kernel* kern, int n_inst, const double* tau, int instant, ModelDev* out);
// disc.cu
int sg_launch_disc(smolgp_ctx* ctx, const ModelDev* d_model, const ModelDev* h_model, const double* dt,
                   int64_t K, double* disc);
// scan.cu
struct ScanArgs {
  const ModelDev* d_model;
  const ModelDev* h_model;
  const smolgp_events* ev;
  const double* disc;
  int64_t batch;
  const double* y;     // [batch][N]
  const double* sigma; // [N]
  const double* amp;   // [batch] or NULL
  double* loglik;      // [batch] or NULL
  double* mean;        // [batch][N] or NULL
  double* var;         // [batch][N] or NULL
  int want_smooth;
  double* fstate;      // [batch][K][n + n^2] or NULL: post-event filtered states (row a7)
  double* binfo;       // [batch][K][n + n^2] or NULL: pre-update backward information
};
int sg_run_scan(smolgp_ctx* ctx, const ScanArgs& a);
struct QueryArgs {
  const ModelDev* d_model;
  const ModelDev* h_model;
  const smolgp_events* ev;
  int64_t batch, M;
  const double* tq;    // [M] device
  int qinst;
  const double* amp;
  const double* fstate;
  const double* binfo;
  double* mean;        // [batch][M]
  double* var;
};
int sg_run_query(smolgp_ctx* ctx, const QueryArgs& a);
// arena helper
int sg_arena(smolgp_ctx* ctx, size_t bytes, void** out);
// device bytes held by the ctx right now (workspace arena, model + discretisation array, sort status, flags, in-call extras)
static inline size_t sg_mem_now(const smolgp_ctx* ctx) { return ctx->arena_bytes + ctx->pers_bytes + ctx->lb_words * 8 + 64 + ctx->mem_extra; }
static inline void sg_mem_mark(smolgp_ctx* ctx, size_t also = 0) { const size_t v = sg_mem_now(ctx) + also; if (v > ctx->mem_peak) ctx->mem_peak = v; }
