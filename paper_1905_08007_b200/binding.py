"""Thin Python binding of libmcqed.so (include/mcqed.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels. PyTorch is used by callers for device
memory and streams; this module only needs raw pointers (torch tensors, numpy arrays or ints).
There is no CPU fallback: device entry points raise McError(MC_ECUDA) without a usable CUDA device.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
MC_OK, MC_EINVAL, MC_ENOMEM, MC_ECUDA, MC_ELIMIT, MC_ETOOBIG = 0, -1, -2, -3, -4, -5
STATIC_MAX_SAMPLES = 65536            # MC_STATIC_MAX_SAMPLES of include/mcqed.h
FLAG_NO_DD, FLAG_NO_TABLES, FLAG_MRG32K3A = 1, 2, 4    # mc_options.flags
FLAG_NO_QD = 2                        # mc_batch_integrate flags bit 1

EXPORTS = [
    "mc_prepare_diagram", "mc_prepare_diagram_host", "mc_free_diagram", "mc_diagram_info", "mc_diagram_id",
    "mc_diagram_subgraphs", "mc_diagram_forests", "mc_diagram_terms", "mc_diagram_sampler_tables", "mc_diagram_blob", "mc_diagram_set_flags", "mc_diagram_set_precision",
    "mc_integrate", "mc_integrate_host", "mc_integrate_static", "mc_batch_create", "mc_batch_integrate", "mc_batch_integrate_host", "mc_batch_integrate_counts", "mc_allocate_samples", "mc_batch_free", "mc_eval_points", "mc_eval_z", "mc_eval_z_qd", "mc_eval_z_interval", "mc_kernel_launch_count", "mc_fp64_peak",
    "mc_strerror", "mc_version",
]


class McGraph(C.Structure):
    _fields_ = [("loops", C.c_int32), ("ext_pos", C.c_int32), ("chord_a", C.c_int32 * 5), ("chord_b", C.c_int32 * 5)]


class McForests(C.Structure):
    _fields_ = [("n_sub", C.c_int32), ("seg_lo", C.POINTER(C.c_int32)), ("seg_hi", C.POINTER(C.c_int32)),
                ("n_forest", C.c_int32), ("forest_mask", C.POINTER(C.c_uint32))]


class McOptions(C.Structure):
    _fields_ = [("deg_floor", C.c_double), ("deg_cap", C.c_double), ("cond_max", C.c_double), ("amin_min", C.c_double), ("flags", C.c_uint32),
                ("deg_floor_ir", C.c_double), ("mix_alpha", C.c_double), ("deg_floor2", C.c_double), ("deg_floor_ir2", C.c_double)]


class McError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s: %s (%d)" % (where, lib().mc_strerror(code).decode(), code))


_lib = None


def library_path():
    return os.path.join(HERE, "libmcqed.so")


def lib():
    """loads libmcqed.so; fails loudly if it has not been built (python -m paper_1905_08007_b200.build)"""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError("libmcqed.so is missing: build it with `python -m paper_1905_08007_b200.build` (there is no fallback)")
        L = C.CDLL(path)
        vp, u64, i32p, dp = C.c_void_p, C.c_uint64, C.POINTER(C.c_int32), C.POINTER(C.c_double)
        L.mc_prepare_diagram.argtypes = [C.POINTER(McGraph), C.POINTER(McForests), C.POINTER(McOptions), C.POINTER(vp)]
        L.mc_prepare_diagram_host.argtypes = L.mc_prepare_diagram.argtypes
        L.mc_free_diagram.argtypes = [vp]
        L.mc_free_diagram.restype = None
        L.mc_diagram_info.argtypes = [vp, i32p, i32p, i32p, i32p, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        L.mc_diagram_id.argtypes = [vp, i32p]
        L.mc_diagram_subgraphs.argtypes = [vp, i32p, i32p, i32p, C.c_int32]
        L.mc_diagram_forests.argtypes = [vp, C.POINTER(C.c_uint32), C.c_int32]
        L.mc_diagram_terms.argtypes = [vp, C.POINTER(C.c_uint32), i32p, i32p, C.c_int32]
        L.mc_diagram_sampler_tables.argtypes = [vp, dp, dp, dp]
        L.mc_diagram_blob.argtypes = [vp, C.POINTER(C.c_uint64), C.c_int64]
        L.mc_diagram_blob.restype = C.c_int64
        L.mc_diagram_set_flags.argtypes = [vp, C.c_uint32]
        L.mc_diagram_set_precision.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_double]
        L.mc_integrate.argtypes = [vp, u64, u64, u64, vp, vp, vp, vp, vp]
        L.mc_integrate_static.argtypes = [vp, u64, u64, u64, vp, vp, vp, vp, vp]
        L.mc_integrate_host.argtypes = [vp, u64, u64, u64, vp, dp, dp, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]
        L.mc_batch_create.argtypes = [C.POINTER(vp), C.c_int32, u64, C.POINTER(vp)]
        L.mc_batch_integrate.argtypes = [vp, u64, u64, u64, C.c_uint32, vp, vp, vp, vp, vp]
        L.mc_batch_integrate_host.argtypes = [vp, u64, u64, u64, C.c_uint32, vp, vp, vp, vp, vp]
        L.mc_batch_integrate_counts.argtypes = [vp, vp, vp, u64, C.c_uint32, vp, vp, vp, vp, vp]
        L.mc_allocate_samples.argtypes = [dp, dp, C.c_int32, C.c_double, u64, C.POINTER(C.c_uint64)]
        L.mc_batch_free.argtypes = [vp]
        L.mc_batch_free.restype = None
        L.mc_eval_points.argtypes = [vp, u64, u64, u64, vp, vp, vp, vp, vp, vp, vp, vp]
        L.mc_eval_z.argtypes = [vp, u64, vp, vp, vp, vp, vp, vp]
        L.mc_eval_z_qd.argtypes = [vp, u64, vp, vp, vp]
        L.mc_eval_z_interval.argtypes = [vp, u64, vp, vp, vp, vp]
        L.mc_kernel_launch_count.restype = C.c_ulonglong
        L.mc_fp64_peak.argtypes = [C.c_int, vp, dp, dp]
        L.mc_strerror.restype = C.c_char_p
        L.mc_strerror.argtypes = [C.c_int]
        L.mc_version.restype = C.c_char_p
        _lib = L
    return _lib


def _ptr(x):
    """raw address of a torch tensor / numpy array / int / None"""
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        return C.c_void_p(x.data_ptr())
    if isinstance(x, np.ndarray):
        return C.c_void_p(x.ctypes.data)
    return C.c_void_p(int(x))


def _check(rc, where):
    if rc != MC_OK:
        raise McError(rc, where)


def make_graph(loops, ext_pos, chords):
    g = McGraph()
    g.loops, g.ext_pos = loops, ext_pos
    for i, (a, b) in enumerate(chords):
        g.chord_a[i], g.chord_b[i] = a, b
    return g


class Diagram:
    """RAII handle around mc_diagram*"""

    def __init__(self, loops, ext_pos, chords, deg_floor=None, deg_cap=1e30, cond_max=2.8e4, amin_min=1e-2, flags=0, host_only=False, forests=None, deg_floor_ir=None,
                 mix_alpha=0.0, deg_floor2=0.0, deg_floor_ir2=0.0):
        """Deg of Eq.(1): defaults (deg_floor, deg_floor_ir) = (1.0, 0.5) (mc_options); a deg_floor given alone also is the value on
        the soft-photon sets. mix_alpha > 0: defensive mixture with a second Eq.(1) density of floors (deg_floor2, deg_floor_ir2)"""
        self.loops, self.M = loops, 3 * loops
        g = make_graph(loops, ext_pos, chords)
        if deg_floor is None:
            deg_floor, deg_floor_ir = 1.0, (0.5 if deg_floor_ir is None else deg_floor_ir)
        elif deg_floor_ir is None:
            deg_floor_ir = deg_floor
        opt = McOptions(deg_floor, deg_cap, cond_max, amin_min, flags, deg_floor_ir, mix_alpha, deg_floor2, deg_floor_ir2)
        self.h = C.c_void_p()
        fo = None
        if forests is not None:
            subs, masks = forests
            lo = (C.c_int32 * len(subs))(*[s[0] for s in subs])
            hi = (C.c_int32 * len(subs))(*[s[1] for s in subs])
            mk = (C.c_uint32 * len(masks))(*masks)
            fo = C.byref(McForests(len(subs), lo, hi, len(masks), mk))
        fn = lib().mc_prepare_diagram_host if host_only else lib().mc_prepare_diagram
        _check(fn(C.byref(g), fo, C.byref(opt), C.byref(self.h)), "mc_prepare_diagram")

    def close(self):
        if getattr(self, "h", None):
            lib().mc_free_diagram(self.h)
            self.h = None

    __del__ = close

    def info(self):
        k, m, n, nt = (C.c_int32() for _ in range(4))
        fl, tb = C.c_int64(), C.c_int64()
        _check(lib().mc_diagram_info(self.h, C.byref(k), C.byref(m), C.byref(n), C.byref(nt), C.byref(fl), C.byref(tb)), "mc_diagram_info")
        return {"class": (k.value, m.value, n.value), "n_terms": nt.value, "flop_per_sample": fl.value, "table_bytes": tb.value}

    def id(self):
        v = C.c_int32()
        _check(lib().mc_diagram_id(self.h, C.byref(v)), "mc_diagram_id")
        return v.value

    def subgraphs(self):
        lo, hi, ty = ((C.c_int32 * 64)() for _ in range(3))
        n = lib().mc_diagram_subgraphs(self.h, lo, hi, ty, 64)
        return [(lo[i], hi[i], ty[i]) for i in range(n)]

    def forests(self):
        m = (C.c_uint32 * 1024)()
        n = lib().mc_diagram_forests(self.h, m, 1024)
        return [m[i] for i in range(n)]

    def terms(self):
        f, gp, sg = (C.c_uint32 * 1024)(), (C.c_int32 * 1024)(), (C.c_int32 * 1024)()
        n = lib().mc_diagram_terms(self.h, f, gp, sg, 1024)
        return [(f[i], gp[i], sg[i]) for i in range(n)]

    def sampler_tables(self):
        n = 1 << self.M
        deg, Z, Cn = np.zeros(n), np.zeros(n), C.c_double()
        dp = C.POINTER(C.c_double)
        _check(lib().mc_diagram_sampler_tables(self.h, deg.ctypes.data_as(dp), Z.ctypes.data_as(dp), C.byref(Cn)), "mc_diagram_sampler_tables")
        return deg, Z, Cn.value

    def set_flags(self, flags):
        _check(lib().mc_diagram_set_flags(self.h, flags), "mc_diagram_set_flags")

    def set_precision(self, cond_max=2.8e4, amin_min=1e-2, dd_cond_max=1e26, w_abs_tol=1e-10):
        _check(lib().mc_diagram_set_precision(self.h, cond_max, amin_min, dd_cond_max, w_abs_tol), "mc_diagram_set_precision")

    def blob(self):
        n = lib().mc_diagram_blob(self.h, None, 0)
        out = np.zeros(n, np.uint64)
        lib().mc_diagram_blob(self.h, out.ctypes.data_as(C.POINTER(C.c_uint64)), n)
        return out

    # ---- device entry points: argument marshalling only ----
    def integrate(self, first_sample, n_samples, seed, stream, out_sum, out_sumsq, out_n_flagged, out_n_dropped):
        """mc_integrate: out_* are device tensors/pointers (accumulated into); asynchronous on `stream` (int handle)"""
        _check(lib().mc_integrate(self.h, first_sample, n_samples, seed, _ptr(stream), _ptr(out_sum), _ptr(out_sumsq),
                                  _ptr(out_n_flagged), _ptr(out_n_dropped)), "mc_integrate")

    def integrate_static(self, first_sample, n_samples, seed, stream, out_sum, out_sumsq, out_n_flagged, out_n_dropped):
        """mc_integrate_static: binary64 tier, scratch in the library's static device array (no allocation); n_samples <= STATIC_MAX_SAMPLES"""
        _check(lib().mc_integrate_static(self.h, first_sample, n_samples, seed, _ptr(stream), _ptr(out_sum), _ptr(out_sumsq),
                                         _ptr(out_n_flagged), _ptr(out_n_dropped)), "mc_integrate_static")

    def integrate_host(self, first_sample, n_samples, seed, stream=None):
        s, s2, nf, nd = C.c_double(), C.c_double(), C.c_ulonglong(), C.c_ulonglong()
        _check(lib().mc_integrate_host(self.h, first_sample, n_samples, seed, _ptr(stream), C.byref(s), C.byref(s2), C.byref(nf), C.byref(nd)), "mc_integrate_host")
        return s.value, s2.value, nf.value, nd.value

    def eval_points(self, first_sample, n, seed, stream=None, z=None, order=None, p=None, f=None, f64=None, cond=None, flag=None):
        _check(lib().mc_eval_points(self.h, first_sample, n, seed, _ptr(stream), _ptr(z), _ptr(order), _ptr(p), _ptr(f), _ptr(f64),
                                    _ptr(cond), _ptr(flag)), "mc_eval_points")

    def eval_z_qd(self, n, z_in, stream, fqd):
        _check(lib().mc_eval_z_qd(self.h, n, _ptr(z_in), _ptr(stream), _ptr(fqd)), "mc_eval_z_qd")

    def eval_z_interval(self, n, z_in, stream, lo, hi):
        _check(lib().mc_eval_z_interval(self.h, n, _ptr(z_in), _ptr(stream), _ptr(lo), _ptr(hi)), "mc_eval_z_interval")

    def eval_z(self, n, z_in, stream=None, f64=None, fdd=None, cond=None, aux=None):
        _check(lib().mc_eval_z(self.h, n, _ptr(z_in), _ptr(stream), _ptr(f64), _ptr(fdd), _ptr(cond), _ptr(aux)), "mc_eval_z")


class Batch:
    """RAII handle around mc_batch*: a set of device-prepared Diagrams integrated by one launch per precision tier"""

    def __init__(self, diagrams, max_samples_per_call):
        self.diagrams = list(diagrams)                   # keeps the handles alive
        arr = (C.c_void_p * len(self.diagrams))(*[d.h.value for d in self.diagrams])
        self.h = C.c_void_p()
        _check(lib().mc_batch_create(arr, len(self.diagrams), max_samples_per_call, C.byref(self.h)), "mc_batch_create")

    def close(self):
        if getattr(self, "h", None):
            lib().mc_batch_free(self.h)
            self.h = None

    __del__ = close

    def integrate(self, first_sample, n_samples, seed, stream, out_sum, out_sumsq, out_n_flagged, out_n_dropped, flags=0):
        """mc_batch_integrate: out_* are device tensors/pointers of len(diagrams) elements (accumulated into)"""
        _check(lib().mc_batch_integrate(self.h, first_sample, n_samples, seed, flags, _ptr(stream), _ptr(out_sum), _ptr(out_sumsq),
                                        _ptr(out_n_flagged), _ptr(out_n_dropped)), "mc_batch_integrate")

    def integrate_counts(self, first_samples, n_samples, seed, stream, out_sum, out_sumsq, out_n_flagged, out_n_dropped, flags=0):
        """mc_batch_integrate_counts: per-diagram sample ranges (host sequences of len(diagrams) integers)"""
        f = np.ascontiguousarray(first_samples, np.uint64)
        n = np.ascontiguousarray(n_samples, np.uint64)
        assert len(f) == len(n) == len(self.diagrams)
        _check(lib().mc_batch_integrate_counts(self.h, _ptr(f), _ptr(n), seed, flags, _ptr(stream), _ptr(out_sum), _ptr(out_sumsq),
                                               _ptr(out_n_flagged), _ptr(out_n_dropped)), "mc_batch_integrate_counts")

    def integrate_host(self, first_sample, n_samples, seed, stream=None, flags=0):
        n = len(self.diagrams)
        s, s2, nf, nd = np.zeros(n), np.zeros(n), np.zeros(n, np.uint64), np.zeros(n, np.uint64)
        _check(lib().mc_batch_integrate_host(self.h, first_sample, n_samples, seed, flags, _ptr(stream), _ptr(s), _ptr(s2), _ptr(nf), _ptr(nd)),
               "mc_batch_integrate_host")
        return s, s2, nf, nd


def allocate_samples(sigma, cost, budget, n_min=1):
    """mc_allocate_samples: n_j ~ sigma_j / sqrt(cost_j) with sum n_j cost_j = budget"""
    sg, cs = np.ascontiguousarray(sigma, np.float64), np.ascontiguousarray(cost, np.float64)
    out = np.zeros(len(sg), np.uint64)
    dp = C.POINTER(C.c_double)
    _check(lib().mc_allocate_samples(sg.ctypes.data_as(dp), cs.ctypes.data_as(dp), len(sg), float(budget), int(n_min), out.ctypes.data_as(C.POINTER(C.c_uint64))), "mc_allocate_samples")
    return out


def kernel_launch_count():
    return int(lib().mc_kernel_launch_count())


def fp64_peak(iters=4096, stream=None):
    fl, ms = C.c_double(), C.c_double()
    _check(lib().mc_fp64_peak(iters, _ptr(stream), C.byref(fl), C.byref(ms)), "mc_fp64_peak")
    return fl.value, ms.value


def version():
    return lib().mc_version().decode()
