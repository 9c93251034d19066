// scan_plan.h -- host-side helpers shared by the translation units that launch the scan kernels (scan.cu, scan_sqrt.cu)
#pragma once
#include "common.h"

// groups per CTA: the count that puts the most groups on one SM (228 KB of shared memory per SM,
// 1 KB reserved per CTA, at most 128 threads per CTA); ties go to the smaller CTA
static inline int groups_per_cta(size_t per_group, int G, int* groups_per_sm = nullptr) {
  int best = 1, best_sm = 0;
  for (int gpc = 1; gpc <= 128 / G; ++gpc) {
    const size_t cta = per_group * gpc;
    if (cta > 227 * 1024) break;
    int ctas = (int)((228 * 1024) / (cta + 1024));
    if (ctas > 32) ctas = 32;
    const int warps = (gpc * G + 31) / 32;
    if (ctas * warps > 64) ctas = 64 / warps;
    if (ctas * gpc > best_sm) { best_sm = ctas * gpc; best = gpc; }
  }
  if (groups_per_sm) *groups_per_sm = best_sm > 0 ? best_sm : 1;
  return best;
}


// (lanes, row stride) variants compiled: lanes = 8/16/32 for n + 1 <= 8/16/33 columns, stride = chunk_ld(n)
#define SG_DISPATCH_GL(G, LD, CALL)                                                      \
  do {                                                                                   \
    if (G == 8 && LD == 5) { CALL(8, 5); }                                               \
    else if (G == 8 && LD == 9) { CALL(8, 9); }                                          \
    else if (G == 16 && LD == 5) { CALL(16, 5); }                                        \
    else if (G == 16 && LD == 9) { CALL(16, 9); }                                        \
    else if (G == 16 && LD == 13) { CALL(16, 13); }                                      \
    else if (G == 16 && LD == 17) { CALL(16, 17); }                                      \
    else if (G == 32 && LD == 5) { CALL(32, 5); }                                        \
    else if (G == 32 && LD == 9) { CALL(32, 9); }                                        \
    else if (G == 32 && LD == 13) { CALL(32, 13); }                                      \
    else if (G == 32 && LD == 17) { CALL(32, 17); }                                      \
    else if (G == 32 && LD == 21) { CALL(32, 21); }                                      \
    else if (G == 32 && LD == 25) { CALL(32, 25); }                                      \
    else if (G == 32 && LD == 29) { CALL(32, 29); }                                      \
    else if (G == 32 && LD == 33) { CALL(32, 33); }                                      \
    else { ctx->err = "scan: unsupported (lanes, n) combination"; return SMOLGP_EUNSUPPORTED; } \
  } while (0)


struct ScanDev;
struct DenseArgs;
struct QueryDev;
// square-root form: kernels and launchers live in scan_sqrt.cu (a translation unit of its own: the fourteen (lanes, stride)
// variants of three chunk kernels compile in parallel with scan.cu)
int sg_launch_sqrt_chunk(smolgp_ctx* ctx, const ScanDev& P, const ModelDev* hm, int G, bool fold);
int sg_launch_sqrt_dense(smolgp_ctx* ctx, const DenseArgs& D, int n, bool fold);
int sg_launch_sqrt_query(smolgp_ctx* ctx, const QueryDev& Q, const ModelDev* hm, int G);
