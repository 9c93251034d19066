// scan_sqrt.cu -- the square-root (Cholesky-factor) form of the scan: kernels (chunk_sqrt.cuh, dense_sqrt.cuh) and their
// launchers, called from scan_host.cu when the model asks for factor form.
#include <math.h>

#include "dense_sqrt.cuh"
#include "scan_plan.h"

// square-root form (chunk_sqrt.cuh, dense_sqrt.cuh): generic kernels
template <int G, int LD>
static int launch_sqrt(smolgp_ctx* ctx, const ScanDev& P, const ModelDev* hm, bool fold) {
  const size_t per_group = (size_t)(fold ? fold0s_group_doubles(hm->n, LD, hm->disc_stride, hm->nblk, G) : sqrt_group_doubles(hm->n, LD, hm->disc_stride, hm->nblk, G)) * 8;
  const int gpc = groups_per_cta(per_group, G);
  const size_t smem = per_group * gpc;
  if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  if (hm->n + hm->d + hm->nblk > sqrt_ldm(LD)) { ctx->err = "scan: model too wide for the square-root kernel"; return SMOLGP_EUNSUPPORTED; }
  const int64_t groups = P.batch * P.c1;
  if (fold) {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_fold0_sqrt<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_FOLD0);
    k_fold0_sqrt<G, LD><<<(unsigned)((groups + gpc - 1) / gpc), gpc * G, smem, ctx->stream>>>(P);
  } else {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_down0_sqrt<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_DOWN0);
    k_down0_sqrt<G, LD><<<(unsigned)((groups + gpc - 1) / gpc), gpc * G, smem, ctx->stream>>>(P);
  }
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}


int sg_launch_sqrt_dense(smolgp_ctx* ctx, const DenseArgs& D, int n, bool fold) {
  const size_t smem = (size_t)(fold ? foldDs_group_doubles(n) : downDs_group_doubles(n)) * 8;
  if (smem > ctx->smem_optin) { ctx->err = "scan: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  dim3 grid((unsigned)(D.batch * D.cout), fold ? 1 : (D.want_suffix ? 2 : 1));
  if (fold) {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_foldD_sqrt<SG_DENSE_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_FOLDD);
    k_foldD_sqrt<SG_DENSE_NT><<<grid, SG_DENSE_NT, smem, ctx->stream>>>(D);
  } else {
    SG_CUDA(ctx, cudaFuncSetAttribute(k_downD_sqrt<SG_DENSE_NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    sg_launch_begin(ctx, KID_DOWND);
    k_downD_sqrt<SG_DENSE_NT><<<grid, SG_DENSE_NT, smem, ctx->stream>>>(D);
  }
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}


template <int G, int LD>
static int launch_query_sqrt(smolgp_ctx* ctx, const QueryDev& Q, const ModelDev* hm) {
  const size_t per_group = (size_t)querys_group_doubles(hm->n, LD, hm->disc_stride, hm->nblk, G) * 8;
  const int gpc = groups_per_cta(per_group, G);
  const size_t smem = per_group * gpc;
  if (smem > ctx->smem_optin) { ctx->err = "query: shared memory need exceeds the device limit"; return SMOLGP_EUNSUPPORTED; }
  const int64_t groups = Q.batch * Q.Mq;
  SG_CUDA(ctx, cudaFuncSetAttribute(k_query_sqrt<G, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  sg_launch_begin(ctx, KID_QUERY);
  k_query_sqrt<G, LD><<<(unsigned)((groups + gpc - 1) / gpc), gpc * G, smem, ctx->stream>>>(Q);
  sg_launch_end(ctx);
  SG_CUDA(ctx, cudaGetLastError());
  return SMOLGP_OK;
}


int sg_launch_sqrt_chunk(smolgp_ctx* ctx, const ScanDev& P, const ModelDev* hm, int G, bool fold) {
  int rc = SMOLGP_EUNSUPPORTED;
#define SG_CALL_SQ(g_, ld_) rc = launch_sqrt<g_, ld_>(ctx, P, hm, fold)
  SG_DISPATCH_GL(G, chunk_ld(hm->n), SG_CALL_SQ);
#undef SG_CALL_SQ
  return rc;
}

int sg_launch_sqrt_query(smolgp_ctx* ctx, const QueryDev& Q, const ModelDev* hm, int G) {
  int rc = SMOLGP_EUNSUPPORTED;
#define SG_CALL_QS(g_, ld_) rc = launch_query_sqrt<g_, ld_>(ctx, Q, hm)
  SG_DISPATCH_GL(G, chunk_ld(hm->n), SG_CALL_QS);
#undef SG_CALL_QS
  return rc;
}
