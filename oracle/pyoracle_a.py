"""oracle/pyoracle_a.py — ctypes access to liboracle_a.so ("Oracle-A", qed_oracle_a.c).  TEST INFRASTRUCTURE.

Oracle-A evaluates the subtracted integrand per point straight from its definition (explicit 4x4 matrices, explicit
Wick pairings, explicit traces; no tables). It shares no code with the table-driven oracle (pyoracle.py / liboracle.so)
nor with the CUDA path; only tests/ may import this module.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


class GraphA(C.Structure):
    _fields_ = [("loops", C.c_int32), ("ext_pos", C.c_int32), ("chord_a", C.c_int32 * 5), ("chord_b", C.c_int32 * 5)]


def make_graph(loops, ext_pos, chords):
    g = GraphA()
    g.loops, g.ext_pos = loops, ext_pos
    for i, (a, b) in enumerate(chords):
        g.chord_a[i], g.chord_b[i] = a, b
    return g


_lib = None


def lib():
    global _lib
    if _lib is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        mod.build()
        _lib = C.CDLL(mod.LIB_A)
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def terms(loops, ext_pos, chords):
    """(subgraphs [(lo, hi, type)], terms [(forest bitmask, gprime or -1, sign)]) in canonical order"""
    g = make_graph(loops, ext_pos, chords)
    ns = C.c_int32()
    lo, hi, ty = (np.zeros(32, np.int32) for _ in range(3))
    f, gp, sg = np.zeros(1024, np.uint32), np.zeros(1024, np.int32), np.zeros(1024, np.int32)
    n = lib().oracle_a_terms(C.byref(g), C.byref(ns), _p(lo, C.c_int32), _p(hi, C.c_int32), _p(ty, C.c_int32), _p(f, C.c_uint32), _p(gp, C.c_int32), _p(sg, C.c_int32))
    if n < 0:
        raise ValueError("invalid graph")
    return [(int(lo[i]), int(hi[i]), int(ty[i])) for i in range(ns.value)], [(int(f[i]), int(gp[i]), int(sg[i])) for i in range(n)]


def eval_z(loops, ext_pos, chords, z, want_terms=False):
    """f(z) at the rows of z (n x 3L, by line index); with want_terms also the n x nterm signed term values"""
    g = make_graph(loops, ext_pos, chords)
    z = np.ascontiguousarray(z, np.float64).reshape(-1, 3 * loops)
    n = len(z)
    nt = len(terms(loops, ext_pos, chords)[1])
    f, tt = np.zeros(n), np.zeros((n, nt))
    rc = lib().oracle_a_eval(C.byref(g), C.c_uint64(n), _p(z, C.c_double), _p(f, C.c_double), _p(tt, C.c_double))
    if rc != 0:
        raise ValueError("oracle_a_eval: %d" % rc)
    return (f, tt) if want_terms else f


def set_variant(v):
    """0 = the definition; 1 / 2 = deliberately wrong operator assignments (negative controls of the infrared pin)"""
    lib().oracle_a_set_variant(int(v))
