"""Builds libmcqed.so in-tree: hand-written CUDA for sm_100a (nvcc) + host C++ (g++), linked by nvcc.

Usage: python -m paper_1905_08007_b200.build [--force] [-v]
Objects are rebuilt only when the content hash of their sources changes (snapshots lose mtimes).
"""
import concurrent.futures
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmcqed.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
DEFS = os.environ.get("MCQED_DEFS", "").split()    # tuning builds: -D macros seen by BOTH compilers, e.g. MCQED_DEFS="-DMQ_WL=2 -DMQ_TPB_F64=128" (diagram.hpp, device_layout.h)
NVCC_FLAGS = ARCH + ["-lineinfo", "-O3", "-std=c++17", "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC,-ffp-contract=off,-pthread", "-Xptxas", "-v"] + DEFS + os.environ.get("MCQED_NVCC_EXTRA", "").split()   # e.g. MCQED_NVCC_EXTRA=-DMQ_DUAL=0 for a tuning build
GXX_FLAGS = ["-O2", "-std=c++17", "-fPIC", "-ffp-contract=off", "-pthread", "-I/usr/local/cuda/include"] + DEFS
COMMON = ["device_layout.h", "host_model.hpp", "diagram.hpp", os.path.join("..", "..", "include", "mcqed.h")]
KERN = COMMON + ["mcqed_kernels.cuh", "dd_arith.cuh", "pt2_arith.cuh", "kern_common.cuh"]
UNITS = {  # object -> (compiler, source, dependencies)
    "host_prepare.o": ("g++", "host_prepare.cpp", COMMON + ["coef_gen.hpp"]),
    "mcqed_api.o": ("g++", "mcqed_api.cpp", COMMON),
    "kern_f64.o": ("nvcc", "kern_f64.cu", KERN),
    "kern_dd.o": ("nvcc", "kern_dd.cu", KERN),
    "kern_qd.o": ("nvcc", "kern_qd.cu", KERN + ["qd_arith.cuh"]),
    "kern_iv.o": ("nvcc", "kern_iv.cu", KERN + ["iv_arith.cuh"]),
    "prep_kernel.o": ("nvcc", "prep_kernel.cu", ["device_layout.h"]),
}


def _digest(files, flags):
    h = hashlib.sha256(" ".join(flags).encode())
    for f in files:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _compile(obj, force):
    comp, src, deps = UNITS[obj]
    flags = NVCC_FLAGS if comp == "nvcc" else GXX_FLAGS
    out, stamp = os.path.join(OBJ, obj), os.path.join(OBJ, obj + ".stamp")
    digest = _digest([src] + deps, flags)
    if not force and os.path.exists(out) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return False, ""
    cmd = ([NVCC] + flags if comp == "nvcc" else ["g++"] + flags) + ["-c", os.path.join(CSRC, src), "-o", out]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = " ".join(cmd) + "\n" + res.stdout + res.stderr
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError("compile failed: " + src)
    with open(stamp, "w") as fh:
        fh.write(digest)
    return True, log


def build(force=False, verbose=False):
    os.makedirs(OBJ, exist_ok=True)
    with concurrent.futures.ThreadPoolExecutor(max_workers=4) as ex:
        results = list(ex.map(lambda o: _compile(o, force), UNITS))
    changed = any(r[0] for r in results)
    log = "".join(r[1] for r in results)
    if log:
        with open(os.path.join(OBJ, "build.log"), "w") as fh:
            fh.write(log)
    if changed or not os.path.exists(LIB):
        cmd = [NVCC] + ARCH + ["-shared", "-o", LIB] + [os.path.join(OBJ, o) for o in UNITS] + ["-Xcompiler", "-pthread"]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("link failed")
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
