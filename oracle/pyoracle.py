"""oracle/pyoracle.py — ctypes access to liboracle.so.  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module (the product path in paper_1905_08007_b200/ never does).
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
NGRADE = 6
MAXCHILD = 5


class OracleGraph(C.Structure):
    _fields_ = [("loops", C.c_int32), ("ext_pos", C.c_int32), ("chord_a", C.c_int32 * 5), ("chord_b", C.c_int32 * 5)]

    @classmethod
    def make(cls, loops, ext_pos, chords):
        g = cls()
        g.loops, g.ext_pos = loops, ext_pos
        for i, (a, b) in enumerate(chords):
            g.chord_a[i], g.chord_b[i] = a, b
        return g

    def chords(self):
        return [(self.chord_a[i], self.chord_b[i]) for i in range(self.loops)]

    def key(self):
        return (self.loops, self.ext_pos, tuple(self.chords()))


_lib = None


def lib():
    global _lib
    if _lib is None:
        import importlib.util
        spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(HERE, "build.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        _lib = C.CDLL(mod.build())
        _lib.oracle_u01.restype = C.c_double
        _lib.oracle_u01.argtypes = [C.c_uint32, C.c_uint32]
        _lib.oracle_sample_uniform.restype = C.c_double
        _lib.oracle_sample_uniform.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_int]
        for f in ("oracle_det_pow",):
            getattr(_lib, f).restype = C.c_double
            getattr(_lib, f).argtypes = [C.c_double, C.c_double]
        for f in ("oracle_det_log2", "oracle_det_exp2"):
            getattr(_lib, f).restype = C.c_double
            getattr(_lib, f).argtypes = [C.c_double]
        _lib.oracle_sample_uniform_mrg.restype = C.c_double
        _lib.oracle_sample_uniform_mrg.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_int]
        _lib.oracle_mrg32k3a.restype = None
        _lib.oracle_mrg32k3a.argtypes = [C.POINTER(C.c_uint64), C.c_uint64, C.c_int, C.POINTER(C.c_uint64)]
        _lib.oracle_mrg_matpow.restype = None
        _lib.oracle_mrg_matpow.argtypes = [C.c_int, C.c_int, C.c_uint64, C.POINTER(C.c_uint64)]
        _lib.oracle_set_generator.argtypes = [C.c_void_p, C.c_int]
        _lib.oracle_set_mixture.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double]
        _lib.oracle_prepare_diagram.argtypes = [C.POINTER(OracleGraph), C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.POINTER(C.c_void_p)]
        _lib.oracle_free_diagram.argtypes = [C.c_void_p]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def graph_count(L):
    return lib().oracle_graph_count(L)


def graph_get(L, idx):
    g = OracleGraph()
    if lib().oracle_graph_get(L, idx, C.byref(g)) != 0:
        raise IndexError(idx)
    return g


def all_graphs(L):
    n = graph_count(L)
    arr = (OracleGraph * n)()
    if lib().oracle_graph_list(L, arr) != n:
        raise RuntimeError("oracle_graph_list")
    out = []
    for i in range(n):
        g = OracleGraph()
        C.memmove(C.byref(g), C.byref(arr[i]), C.sizeof(OracleGraph))
        out.append(g)
    return out


def graph_class(g):
    k, m, n = C.c_int(), C.c_int(), C.c_int()
    if lib().oracle_graph_class(C.byref(g), C.byref(k), C.byref(m), C.byref(n)) != 0:
        raise ValueError("invalid graph")
    return (k.value, m.value, n.value)


def graph_mirror(g):
    out = OracleGraph()
    if lib().oracle_graph_mirror(C.byref(g), C.byref(out)) != 0:
        raise ValueError("invalid graph")
    return out


def graph_id(g):
    return lib().oracle_graph_id(C.byref(g))


def graph_validate(g):
    return lib().oracle_graph_validate(C.byref(g))


def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().oracle_philox(c, k, o)
    return list(o)


def mrg32k3a(state6, skip, nout):
    """raw MRG32k3a outputs w_n (L'Ecuyer 1999) after skipping `skip` outputs from the six-word state"""
    st = np.asarray(state6, dtype=np.uint64).copy()
    out = np.zeros(nout, dtype=np.uint64)
    lib().oracle_mrg32k3a(_p(st, C.c_uint64), C.c_uint64(skip), nout, _p(out, C.c_uint64))
    return out


def mrg_matpow(comp, e, mult=1):
    """A_comp^(mult * 2^e) mod m_comp, 3x3"""
    out = np.zeros(9, dtype=np.uint64)
    lib().oracle_mrg_matpow(comp, e, C.c_uint64(mult), _p(out, C.c_uint64))
    return out.reshape(3, 3)


def sample_uniform_mrg(idx, diag, seed, r):
    return lib().oracle_sample_uniform_mrg(C.c_uint64(idx), C.c_uint32(diag), C.c_uint64(seed), r)


class Diagram:
    """One prepared diagram (combinatorics + sampler tables [+ integrand tables])."""

    def __init__(self, g, deg_floor=None, deg_cap=1e30, level=1, prune=1, deg_floor_ir=None):
        """Deg of Eq.(1): defaults (deg_floor, deg_floor_ir) = (1.0, 0.5) (S5); a deg_floor given alone also is the value
        on the soft-photon sets (the one-floor reading of round 1)"""
        self.g = g
        self.h = C.c_void_p()
        if deg_floor is None:
            deg_floor, deg_floor_ir = 1.0, (0.5 if deg_floor_ir is None else deg_floor_ir)
        elif deg_floor_ir is None:
            deg_floor_ir = deg_floor
        rc = lib().oracle_prepare_diagram(C.byref(g), deg_floor, deg_cap, deg_floor_ir, level, prune, C.byref(self.h))
        if rc != 0:
            raise ValueError("oracle_prepare_diagram failed: %d" % rc)
        info = (C.c_int64 * 8)()
        lib().oracle_diagram_info(self.h, info)
        (self.id, self.M, self.nsub, self.nforest, self.nterm, self.ngeom, self.nnode, self.n_monomials) = list(info)

    def __del__(self):
        if getattr(self, "h", None):
            lib().oracle_free_diagram(self.h)
            self.h = None

    def subgraphs(self):
        lo, hi, ty = (np.zeros(32, np.int32) for _ in range(3))
        n = lib().oracle_get_subgraphs(self.h, _p(lo, C.c_int32), _p(hi, C.c_int32), _p(ty, C.c_int32))
        return [(int(lo[i]), int(hi[i]), int(ty[i])) for i in range(n)]

    def forests(self):
        f = np.zeros(512, np.uint32)
        n = lib().oracle_get_forests(self.h, _p(f, C.c_uint32))
        return [int(x) for x in f[:n]]

    def terms(self):
        f, gp, sg = np.zeros(512, np.uint32), np.zeros(512, np.int32), np.zeros(512, np.int32)
        n = lib().oracle_get_terms(self.h, _p(f, C.c_uint32), _p(gp, C.c_int32), _p(sg, C.c_int32))
        return [(int(f[i]), int(gp[i]), int(sg[i])) for i in range(n)]

    def sampler_tables(self):
        n = 1 << self.M
        deg, Z, Cn = np.zeros(n), np.zeros(n), C.c_double()
        lib().oracle_get_sampler_tables(self.h, _p(deg, C.c_double), _p(Z, C.c_double), C.byref(Cn))
        return deg, Z, Cn.value

    def set_generator(self, kind):
        """0 = Philox4x32-10 (default), 1 = MRG32k3a (S1b)"""
        assert lib().oracle_set_generator(self.h, kind) == 0

    def set_mixture(self, alpha, deg_floor2, deg_floor_ir2=0.0, deg_cap2=1e30):
        """defensive mixture (S5b): probability alpha of drawing from a second Eq.(1) density with these Deg floors"""
        assert lib().oracle_set_mixture(self.h, alpha, deg_floor2, deg_cap2, deg_floor_ir2) == 0

    def sample(self, first, n, seed):
        z, p, order = np.zeros((n, self.M)), np.zeros(n), np.zeros((n, self.M), np.int32)
        lib().oracle_sample_points(self.h, C.c_uint64(first), C.c_uint64(n), C.c_uint64(seed), _p(z, C.c_double), _p(p, C.c_double), _p(order, C.c_int32))
        return z, p, order

    def density(self, z):
        z = np.ascontiguousarray(z, np.float64).reshape(-1, self.M)
        p = np.zeros(len(z))
        lib().oracle_density(self.h, C.c_uint64(len(z)), _p(z, C.c_double), _p(p, C.c_double))
        return p

    def eval_z(self, z, wide=False, want_terms=False):
        """returns dict with f64, abs64 (round-off scale), optionally fwide and terms"""
        z = np.ascontiguousarray(z, np.float64).reshape(-1, self.M)
        n = len(z)
        f64, a64 = np.zeros(n), np.zeros(n)
        fw = np.zeros(n) if wide else None
        tt = np.zeros((n, self.nterm)) if want_terms else None
        rc = lib().oracle_eval_z(self.h, C.c_uint64(n), _p(z, C.c_double), _p(f64, C.c_double), _p(fw, C.c_double), _p(a64, C.c_double), _p(tt, C.c_double))
        if rc != 0:
            raise RuntimeError("oracle_eval_z: %d" % rc)
        out = {"f64": f64, "abs64": a64}
        if wide:
            out["fwide"] = fw
        if want_terms:
            out["terms"] = tt
        return out

    def integrate(self, first, n, seed, mode=0):
        s1, s2, nf = C.c_double(), C.c_double(), C.c_uint64()
        rc = lib().oracle_integrate(self.h, C.c_uint64(first), C.c_uint64(n), C.c_uint64(seed), mode, C.byref(s1), C.byref(s2), C.byref(nf))
        if rc != 0:
            raise RuntimeError("oracle_integrate: %d" % rc)
        return s1.value, s2.value, nf.value

    def nodes(self):
        n = self.nnode
        sub, op, nch, ch = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros((n, MAXCHILD), np.int32)
        lib().oracle_get_nodes(self.h, _p(sub, C.c_int32), _p(op, C.c_int32), _p(nch, C.c_int32), _p(ch, C.c_int32))
        return [(int(sub[i]), int(op[i]), [int(c) for c in ch[i, :nch[i]]]) for i in range(n)]

    def term_roots(self):
        r = np.zeros(self.nterm, np.int32)
        lib().oracle_get_term_roots(self.h, _p(r, C.c_int32))
        return [int(x) for x in r]

    def node_value(self, node, z):
        z = np.ascontiguousarray(z, np.float64)
        out, UV = np.zeros(2 * NGRADE), np.zeros(2)
        rc = lib().oracle_node_value(self.h, node, _p(z, C.c_double), _p(out, C.c_double), _p(UV, C.c_double))
        if rc != 0:
            raise RuntimeError("oracle_node_value: %d" % rc)
        return out.reshape(2, NGRADE), UV[0], UV[1]


def num_threads():
    return lib().oracle_num_threads()


def estimate(s1, s2, n):
    """O7: mean and 1-sigma error of the mean from the Monte Carlo sums"""
    mean = s1 / n
    var = max(s2 / n - mean * mean, 0.0) / n
    return mean, var ** 0.5
