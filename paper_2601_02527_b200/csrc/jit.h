// jit.h -- run-time specialised chunk kernels (jit.cu)
#pragma once
#include "common.h"

struct Tab;
// what a specialised module is compiled for, beyond the model's structure
struct SgJitCfg {
  int G, LD;        // lanes per chunk and row stride of the shared-memory kernels (k_query; k_fold0 / k_down0 when !reg)
  int reg;          // 1: k_fold0 / k_down0 are the register-resident kernels of chunk_reg.cuh
  int rG, rCPL;     // k_down0 (register): lanes per chunk, columns per lane
  int fG, fCPL;     // k_fold0 (register)
  int dot2;         // bit 0: class-A products of the dense levels compensated, bit 1: class-B (dense_kernels.cuh)
  int rMinB, fMinB; // __launch_bounds__ min CTAs per SM of the two register kernels (caps their registers)
};
struct SgJitKernels {
  cudaLibrary_t lib;
  cudaKernel_t fold0, down0, query, foldD, downD, adjD;
  SgJitCfg cfg;
  int regs_fold0, regs_down0; // registers per thread of the compiled chunk kernels
  int prebuilt;               // 1: the module is the ahead-of-time copy linked into the library (no NVRTC involved)
};
const SgJitKernels* sg_jit_get(smolgp_ctx* ctx, const Tab& T, const SgJitCfg& cfg);
bool sg_jit_prebuilt(smolgp_ctx* ctx, const Tab& T, const SgJitCfg& cfg);
bool sg_jit_hot(smolgp_ctx* ctx, const Tab& T, const SgJitCfg& cfg, bool count);
void sg_jit_destroy(smolgp_ctx* ctx);
const char* sg_jit_log(smolgp_ctx* ctx);
