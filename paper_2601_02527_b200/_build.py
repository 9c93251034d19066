"""Builds libsmolgp_b200.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libsmolgp_b200.so")
PROBE_SO = os.path.join(HERE, "libsmolgp_probe.so")  # bench.py's FP64 throughput probe (not part of the product library)
SOURCES = ["api.cu", "model.cu", "events.cu", "disc.cu", "scan.cu", "jit.cu"]
JIT_PARTS = ["dev_consts.h", "grp_dev.cuh", "chunk_dev.cuh", "chunk_kernels.cuh", "chunk_reg.cuh", "dense_kernels.cuh"]  # run-time specialised source, in order
DEPS = SOURCES + ["common.h", "dev_consts.h", "grp_dev.cuh", "chunk_dev.cuh", "chunk_kernels.cuh", "chunk_reg.cuh", "dense_kernels.cuh", "jit.h", "scan_host.cu", os.path.join("..", "..", "include", "smolgp.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _stale():
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def _write_jit_source():
    """csrc/jit_src.inc: the chunk kernels' source as one C++ raw string (local includes stripped),
    compiled at run time by jit.cu with the model's tables as constants."""
    text = []
    for f in JIT_PARTS:
        for line in open(os.path.join(CSRC, f)):
            st = line.strip()
            if st.startswith('#include "') or st == "#pragma once":
                continue
            text.append(line)
    body = "".join(text)
    assert ')SGJIT"' not in body
    out = os.path.join(CSRC, "jit_src.inc")
    new = 'R"SGJIT(' + body + ')SGJIT"\n'
    if not os.path.exists(out) or open(out).read() != new:
        open(out, "w").write(new)


def build(force=False, verbose=False):
    """Compile if missing or stale; returns the path of the shared library."""
    if not force and not _stale():
        return SO
    _write_jit_source()
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, "-c", os.path.join(CSRC, s), "-o", o]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
        objs.append(o)
    for s, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError("nvcc failed on %s:\n%s" % (s, out.decode()))
        if verbose:
            print(out.decode())
    subprocess.check_call([nvcc, "-shared", "-o", SO, *objs, "-lcudart", "-ldl"])
    return SO


def build_probe(force=False):
    """bench.py's measurement tool: a register-only FP64 FMA loop, its own shared object"""
    src = os.path.join(CSRC, "probe_fp64.cu")
    if force or not os.path.exists(PROBE_SO) or os.path.getmtime(PROBE_SO) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.check_call([nvcc, *NVCC_FLAGS, "-shared", src, "-o", PROBE_SO, "-lcudart"])
    return PROBE_SO


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
