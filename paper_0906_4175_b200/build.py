"""Build step of the CUDA library: `python -m paper_0906_4175_b200.build` -> paper_0906_4175_b200/libgwmf.so.

nvcc cross-compiles for sm_100a without a GPU.  The .so is built in-tree (git-ignored) so that it
travels with the repository snapshot to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgwmf.so")
SOURCES = ["api.cu", "segment.cu", "pass1.cu", "pass2.cu", "bandpower.cu", "triggers.cu", "static_scratch.cu"]
HEADERS = ["gwmf_internal.cuh", "fft_reg.cuh", os.path.join("..", "..", "include", "gwmf.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    hdr_time = _newest([os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)])
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s).replace(".cu", ".o"))
        objs.append(o)
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_time):
            log = open(o + ".log", "w")
            procs.append((s, log, subprocess.Popen(["nvcc", *NVCC_FLAGS, "-c", s, "-o", o], stdout=log, stderr=log)))
    failed = False
    for s, log, pr in procs:
        rc = pr.wait()
        log.close()
        if rc != 0 or verbose:
            sys.stderr.write(open(log.name).read())
        failed |= rc != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if procs or not os.path.exists(LIB) or os.path.getmtime(LIB) < _newest(deps):
        subprocess.run(["nvcc", "-shared", "-o", LIB, *objs], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
