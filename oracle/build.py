"""oracle/build.py — builds liboracle.so (TEST INFRASTRUCTURE; plain C, gcc).

-ffp-contract=off: the sampler's bit-exactness contract (S2-S4) forbids FMA contraction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
LIB_A = os.path.join(HERE, "liboracle_a.so")
# two independent libraries: the table-driven oracle ("Oracle-B") and the per-point definition ("Oracle-A", qed_oracle_a.c),
# which includes none of Oracle-B's headers
TARGETS = {LIB: (["qed_oracle.c"], ["qed_combi.h", "qed_piece.h", "qed_sampler.h", "qed_tables.h", "qed_eval_impl.h"]),
           LIB_A: (["qed_oracle_a.c"], [])}


def _build_one(lib, src, deps, force):
    import hashlib
    h = hashlib.sha256()
    for f in src + deps:
        with open(os.path.join(HERE, f), "rb") as fh:
            h.update(fh.read())
    digest, stamp = h.hexdigest(), lib + ".stamp"
    if not force and os.path.exists(lib) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return lib      # content hash, not mtime: snapshots lose mtimes
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wno-unused-function", "-o", lib] + [os.path.join(HERE, f) for f in src] + ["-lm"]
    subprocess.check_call(cmd)
    with open(stamp, "w") as fh:
        fh.write(digest)
    return lib


def build(force=False):
    for lib, (src, deps) in TARGETS.items():
        _build_one(lib, src, deps, force)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
