"""oracle/build.py — builds liboracle.so (TEST INFRASTRUCTURE; plain C, gcc).

-ffp-contract=off: the sampler's bit-exactness contract (S2-S4) forbids FMA contraction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SRC = ["qed_oracle.c"]
DEPS = SRC + ["qed_combi.h", "qed_piece.h", "qed_sampler.h", "qed_tables.h", "qed_eval_impl.h"]


def build(force=False):
    import hashlib
    h = hashlib.sha256()
    for f in DEPS:
        with open(os.path.join(HERE, f), "rb") as fh:
            h.update(fh.read())
    digest, stamp = h.hexdigest(), LIB + ".stamp"
    if not force and os.path.exists(LIB) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return LIB      # content hash, not mtime: snapshots lose mtimes
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wno-unused-function", "-o", LIB] + [os.path.join(HERE, f) for f in SRC] + ["-lm"]
    subprocess.check_call(cmd)
    with open(stamp, "w") as fh:
        fh.write(digest)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
