"""Builds libmcqed.so (hand-written CUDA for sm_100a + host C++) in-tree with nvcc.

Usage: python -m paper_1905_08007_b200.build [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmcqed.so")
SOURCES = ["mcqed_api.cu"]
DEPS = SOURCES + ["mcqed_kernels.cuh", "dd_arith.cuh", "device_layout.h", "host_model.hpp", "coef_gen.hpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-pthread", "-shared", "-Xptxas", "-v"]


def build(force=False, verbose=False):
    deps = [os.path.join(CSRC, f) for f in DEPS] + [os.path.join(HERE, "..", "include", "mcqed.h")]
    newest = max(os.path.getmtime(f) for f in deps)
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, "build.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError("nvcc failed")
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
