// jit.cu -- run-time specialisation of the scan kernels (k_fold0, k_down0, k_query, k_foldD, k_downD) for one model
// STRUCTURE: state dimension, block dimensions and offsets, number of instruments and which
// (instrument, block) couplings are non-zero become compile-time constants, so the loops over blocks and
// instruments unroll, the family switch disappears and all shared-memory addresses are immediates.
// Hyper-parameter VALUES (couplings c_qb, tau, sigma) stay run-time kernel parameters: one compilation
// serves every likelihood evaluation of an optimisation over the same kernel structure.
//
// The source is the very text of the statically compiled kernels (csrc/jit_src.inc, written by
// _build.py from dev_consts.h + grp_dev.cuh + chunk_dev.cuh + chunk_kernels.cuh + chunk_reg.cuh + dense_kernels.cuh), compiled with NVRTC
// for sm_100a and loaded through the runtime's library API.  NVRTC is opened with dlopen: when it is
// not there, or a compilation fails, the generic kernels run instead (same arithmetic, same results).
#include <dlfcn.h>
#include <nvrtc.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "chunk_dev.cuh"
#include "jit.h"

static const char* const JIT_SRC =
#include "jit_src.inc"
    ;

// ahead-of-time copies of the specialised module for the structures of the shipped workloads (_build.py: PREBUILT):
// binary blobs linked into this library, looked up by the same structure key as the run-time cache
struct SgPrebuilt { const char* key; const unsigned char* begin; const unsigned char* end; };
#define SG_INCBIN(sym, file)                                                                                              \
  asm(".section .rodata\n.balign 16\n.global " #sym "\n" #sym ":\n.incbin \"" file "\"\n.global " #sym "_end\n" #sym "_end:\n.byte 0\n.previous\n"); \
  extern "C" const unsigned char sym[];                                                                                   \
  extern "C" const unsigned char sym##_end[];
#include "prebuilt.inc"

struct NvrtcApi {
  void* h = nullptr;
  nvrtcResult (*create)(nvrtcProgram*, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
  nvrtcResult (*compile)(nvrtcProgram, int, const char* const*) = nullptr;
  nvrtcResult (*cubin_size)(nvrtcProgram, size_t*) = nullptr;
  nvrtcResult (*cubin)(nvrtcProgram, char*) = nullptr;
  nvrtcResult (*log_size)(nvrtcProgram, size_t*) = nullptr;
  nvrtcResult (*log)(nvrtcProgram, char*) = nullptr;
  nvrtcResult (*destroy)(nvrtcProgram*) = nullptr;
  bool ok = false;
};

struct JitEntry {
  std::string key;
  SgJitKernels k;
  bool good;
};

struct JitState {
  NvrtcApi api;
  bool tried_open = false;
  std::vector<JitEntry> cache;
  std::vector<std::pair<std::string, int64_t>> calls; // calls seen per structure (tiered compilation)
  std::string log;
};

static bool open_nvrtc(NvrtcApi& a) {
  const char* names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12"};
  for (const char* nm : names) { a.h = dlopen(nm, RTLD_NOW | RTLD_LOCAL); if (a.h) break; }
  if (!a.h) return false;
#define SG_SYM(field, name) *(void**)(&a.field) = dlsym(a.h, name); if (!a.field) return false
  SG_SYM(create, "nvrtcCreateProgram");
  SG_SYM(compile, "nvrtcCompileProgram");
  SG_SYM(cubin_size, "nvrtcGetCUBINSize");
  SG_SYM(cubin, "nvrtcGetCUBIN");
  SG_SYM(log_size, "nvrtcGetProgramLogSize");
  SG_SYM(log, "nvrtcGetProgramLog");
  SG_SYM(destroy, "nvrtcDestroyProgram");
#undef SG_SYM
  a.ok = true;
  return true;
}

static std::string structure_key(const Tab& T, const SgJitCfg& c) {
  char buf[128];
  snprintf(buf, sizeof buf, "%d,%d,%d,%d,%d,%d,%d,%d,%d,%d,%d,%d,%d,%d,%d|", T.n, T.d, T.ninst, T.nblk, T.stride, c.G, c.LD, c.reg, c.rG, c.rCPL, c.fG, c.fCPL,
           c.rMinB, c.fMinB, c.dot2);
  std::string k = buf;
  for (int b = 0; b < T.nblk; ++b) { snprintf(buf, sizeof buf, "%d.%d.%d;", T.bdim[b], T.boff[b], T.roff[b]); k += buf; }
  k += "|";
  for (int i = 0; i < T.ninst * T.nblk; ++i) k += (T.cz[i] != 0.0) ? '1' : '0';
  return k;
}

static void int_table(std::string& s, const char* name, int cnt, const int* v) {
  char buf[64];
  s += "__device__ constexpr int ";
  s += name;
  s += "(int i) { constexpr int v[] = {";
  for (int i = 0; i < cnt; ++i) { snprintf(buf, sizeof buf, "%d,", v[i]); s += buf; }
  s += "0}; return v[i]; }\n";
}

static std::string prelude(const Tab& T, const SgJitCfg& c) {
  const int G = c.G, LD = c.LD;
  std::string s = "#define SG_JIT 1\n"
                  "typedef long long int64_t;\ntypedef unsigned long long uint64_t;\n"
                  "typedef int int32_t;\ntypedef unsigned int uint32_t;\n";
  char buf[128];
  snprintf(buf, sizeof buf, "#define JT_N %d\n#define JT_D %d\n#define JT_NI %d\n#define JT_NB %d\n#define JT_STRIDE %d\n", T.n, T.d,
           T.ninst, T.nblk, T.stride);
  s += buf;
  snprintf(buf, sizeof buf, "#define JT_G %d\n#define JT_LD %d\n", G, LD);
  s += buf;
  snprintf(buf, sizeof buf, "#define JT_REG %d\n#define JT_RG %d\n#define JT_RCPL %d\n#define JT_FG %d\n#define JT_FCPL %d\n", c.reg, c.rG, c.rCPL, c.fG, c.fCPL);
  s += buf;
  snprintf(buf, sizeof buf, "#define JT_RTHREADS 32\n#define JT_FTHREADS 32\n#define JT_RMINB %d\n#define JT_FMINB %d\n#define JT_DOT2 %d\n", c.rMinB, c.fMinB, c.dot2);
  s += buf;
  int v[SG_MAXINST * SG_MAXBLK];
  for (int b = 0; b < T.nblk; ++b) v[b] = T.bdim[b];
  int_table(s, "jt_bdim", T.nblk, v);
  for (int b = 0; b < T.nblk; ++b) v[b] = T.boff[b];
  int_table(s, "jt_boff", T.nblk, v);
  for (int b = 0; b < T.nblk; ++b) v[b] = T.roff[b];
  int_table(s, "jt_roff", T.nblk, v);
  for (int j = 0; j < T.d; ++j) v[j] = T.blk_of[j];
  int_table(s, "jt_blkof", T.d, v);
  for (int i = 0; i < T.ninst * T.nblk; ++i) v[i] = (T.cz[i] != 0.0) ? 1 : 0;
  int_table(s, "jt_czmask", T.ninst * T.nblk, v);
  return s;
}

static JitState* state_of(smolgp_ctx* ctx) {
  if (!ctx->jit) ctx->jit = new JitState();
  return (JitState*)ctx->jit;
}

// Tiered compilation: counts the calls made with this structure (when `count`) and says whether it is
// "hot": already compiled, or seen SG_JIT_HOT_CALLS times -- a hyper-parameter optimisation over a small
// series then gets the specialised kernels after a few dozen evaluations, a one-off call never pays for them.
#define SG_JIT_HOT_CALLS 32
bool sg_jit_hot(smolgp_ctx* ctx, const Tab& T, const SgJitCfg& cfg, bool count) {
  JitState* st = state_of(ctx);
  const std::string key = structure_key(T, cfg);
  for (auto& e : st->cache)
    if (e.key == key) return e.good;
  for (auto& c : st->calls)
    if (c.first == key) { if (count) ++c.second; return c.second >= SG_JIT_HOT_CALLS; }
  st->calls.emplace_back(key, count ? 1 : 0);
  return false;
}

void sg_jit_destroy(smolgp_ctx* ctx) {
  JitState* st = (JitState*)ctx->jit;
  if (!st) return;
  for (auto& e : st->cache)
    if (e.good) cudaLibraryUnload(e.k.lib);
  if (st->api.h) dlclose(st->api.h);
  delete st;
  ctx->jit = nullptr;
}

const char* sg_jit_log(smolgp_ctx* ctx) { return ctx->jit ? ((JitState*)ctx->jit)->log.c_str() : ""; }

static bool load_module(JitState* st, JitEntry& ent, const void* cubin, const SgJitCfg& cfg) {
  cudaError_t e = cudaLibraryLoadData(&ent.k.lib, cubin, nullptr, nullptr, 0, nullptr, nullptr, 0);
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.fold0, ent.k.lib, "jit_fold0");
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.down0, ent.k.lib, "jit_down0");
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.query, ent.k.lib, "jit_query");
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.foldD, ent.k.lib, "jit_foldD");
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.downD, ent.k.lib, "jit_downD");
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&ent.k.adjD, ent.k.lib, "jit_adjD");
  if (e != cudaSuccess) { st->log = std::string("loading the specialised kernels: ") + cudaGetErrorString(e); cudaGetLastError(); return false; }
  cudaFuncAttributes fa;
  ent.k.regs_fold0 = (cudaFuncGetAttributes(&fa, (const void*)ent.k.fold0) == cudaSuccess) ? fa.numRegs : 255;
  ent.k.regs_down0 = (cudaFuncGetAttributes(&fa, (const void*)ent.k.down0) == cudaSuccess) ? fa.numRegs : 255;
  cudaGetLastError();
  ent.k.cfg = cfg;
  return true;
}

static const SgPrebuilt* find_prebuilt(const std::string& key) {
  if (getenv("SMOLGP_NO_PREBUILT") || getenv("SMOLGP_JIT_DEFS") || getenv("SMOLGP_JIT_DUMP")) return nullptr; // debugging aids: force the NVRTC path
  for (const SgPrebuilt& p : SG_PREBUILT)
    if (key == p.key) return &p;
  return nullptr;
}

// is there an ahead-of-time module for this structure?  (then it is used from the first call)
bool sg_jit_prebuilt(smolgp_ctx*, const Tab& T, const SgJitCfg& cfg) { return find_prebuilt(structure_key(T, cfg)) != nullptr; }

// returns the specialised kernels for (T's structure, G, LD), compiling them on first use; nullptr when
// run-time compilation is unavailable or failed (the reason is kept in sg_jit_log)
const SgJitKernels* sg_jit_get(smolgp_ctx* ctx, const Tab& T, const SgJitCfg& cfg) {
  JitState* st = state_of(ctx);
  const std::string key = structure_key(T, cfg);
  for (auto& e : st->cache)
    if (e.key == key) return e.good ? &e.k : nullptr;
  JitEntry ent;
  ent.key = key;
  ent.good = false;
  memset(&ent.k, 0, sizeof ent.k);
  ent.k.prebuilt = 0;
  if (const SgPrebuilt* pb = find_prebuilt(key)) {
    ent.good = load_module(st, ent, pb->begin, cfg);
    ent.k.prebuilt = ent.good ? 1 : 0;
  }
  if (!ent.good) {
    if (!st->tried_open) { st->tried_open = true; if (!open_nvrtc(st->api)) st->log = "NVRTC not available (dlopen libnvrtc.so.12 failed)"; }
    if (st->api.ok) {
      std::string src = prelude(T, cfg);
      if (const char* defs = getenv("SMOLGP_JIT_DEFS")) { src += defs; src += "\n"; } // debugging aid: extra #defines for the specialised build
      src += JIT_SRC;
      if (const char* dump = getenv("SMOLGP_JIT_DUMP")) { // debugging aid: the exact text handed to NVRTC
        if (FILE* f = fopen(dump, "w")) { fwrite(src.data(), 1, src.size(), f); fclose(f); }
      }
      nvrtcProgram prog = nullptr;
      const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo"};
      nvrtcResult r = st->api.create(&prog, src.c_str(), "smolgp_chunk_jit.cu", 0, nullptr, nullptr);
      if (r == NVRTC_SUCCESS) r = st->api.compile(prog, 3, opts);
      if (r != NVRTC_SUCCESS) {
        size_t ls = 0;
        if (prog && st->api.log_size(prog, &ls) == NVRTC_SUCCESS && ls > 1) { st->log.resize(ls); st->api.log(prog, &st->log[0]); }
        else st->log = "nvrtc: compilation failed";
      } else {
        size_t cs = 0;
        st->api.cubin_size(prog, &cs);
        std::vector<char> cubin(cs);
        st->api.cubin(prog, cubin.data());
        if (const char* dump = getenv("SMOLGP_JIT_DUMP")) { // debugging aid: the cubin beside the source (nvdisasm -g maps SASS to lines)
          if (FILE* f = fopen((std::string(dump) + ".cubin").c_str(), "wb")) { fwrite(cubin.data(), 1, cubin.size(), f); fclose(f); }
        }
        ent.good = load_module(st, ent, cubin.data(), cfg);
      }
      if (prog) st->api.destroy(&prog);
    }
  }
  st->cache.push_back(ent);
  return st->cache.back().good ? &st->cache.back().k : nullptr;
}
