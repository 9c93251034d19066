// jit.h -- run-time specialised chunk kernels (jit.cu)
#pragma once
#include "common.h"

struct Tab;
struct SgJitKernels {
  cudaLibrary_t lib;
  cudaKernel_t fold0, down0, query, foldD, downD;
};
const SgJitKernels* sg_jit_get(smolgp_ctx* ctx, const Tab& T, int G, int LD);
bool sg_jit_hot(smolgp_ctx* ctx, const Tab& T, int G, int LD, bool count);
void sg_jit_destroy(smolgp_ctx* ctx);
const char* sg_jit_log(smolgp_ctx* ctx);
