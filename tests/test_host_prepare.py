"""CPU tests of the product's host logic (no GPU): the C-ABI library loads and exports what
include/mcqed.h declares, rejects bad input, and its host preparation (combinatorics, Deg/Z tables,
numerator tables read through tests/blob_interp.py) agrees with the oracle."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from blob_interp import Blob

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def mc():
    from paper_1905_08007_b200 import build, binding
    build.build()
    return binding


def _has_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_library_exports_every_declared_symbol(mc):
    hdr = open(os.path.join(ROOT, "include", "mcqed.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(mc_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(mc.EXPORTS)
    lib = mc.lib()
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.mc_version()
    assert lib.mc_strerror(mc.MC_ECUDA).decode().startswith("CUDA")


def test_invalid_graphs_rejected(mc):
    for (L, e, ch) in [(1, 0, [(1, 2)]), (2, 2, [(0, 1), (3, 4)]), (2, 2, [(0, 1), (1, 4)]), (2, 2, [(0, 2), (1, 4)]), (6, 1, [(0, 2)]), (0, 0, [])]:
        with pytest.raises(mc.McError) as ei:
            mc.Diagram(L, e, ch, host_only=True)
        assert ei.value.code == mc.MC_EINVAL
    with pytest.raises(mc.McError):
        mc.Diagram(1, 1, [(0, 2)], deg_floor=-1.0, host_only=True)
    # user forests that disagree with the enumeration
    with pytest.raises(mc.McError):
        mc.Diagram(2, 2, [(0, 4), (1, 3)], host_only=True, forests=([(1, 2)], [0, 1]))
    d = mc.Diagram(2, 2, [(0, 4), (1, 3)], host_only=True, forests=([(1, 3)], [0, 1]))
    assert d.subgraphs() == [(1, 3, 1)]


def test_no_cpu_fallback(mc):
    d = mc.Diagram(1, 1, [(0, 2)], host_only=True)
    with pytest.raises(mc.McError) as ei:      # a host-only handle never computes
        d.integrate_host(0, 10, 1)
    assert ei.value.code == mc.MC_EINVAL
    with pytest.raises(mc.McError) as ei:      # neither does a batch built on one (no device: MC_ECUDA before the handles are looked at)
        mc.Batch([d], 1024)
    assert ei.value.code in (mc.MC_EINVAL, mc.MC_ECUDA)
    with pytest.raises(mc.McError) as ei:      # precision thresholds are validated on the host
        d.set_precision(cond_max=-1.0)
    assert ei.value.code == mc.MC_EINVAL
    d.set_precision(cond_max=1e4, amin_min=1e-2, dd_cond_max=1e26, w_abs_tol=0.0)
    if not _has_cuda():
        with pytest.raises(mc.McError) as ei:
            mc.Diagram(1, 1, [(0, 2)])
        assert ei.value.code == mc.MC_ECUDA
        with pytest.raises(mc.McError) as ei:
            mc.fp64_peak(16)
        assert ei.value.code == mc.MC_ECUDA


def _pairs(po, L, idxs):
    for i in idxs:
        g = po.graph_get(L, i)
        yield i, g


@pytest.mark.parametrize("L,idxs", [(1, [0]), (2, range(6)), (3, range(50)), (4, range(0, 518, 29)), (5, [0, 1234, 2345, 3333, 4444, 6353])])
def test_combinatorics_and_sampler_tables_equal_oracle(po, mc, L, idxs):
    """graph/forest indexing and the Eq.(1) tables must be bit-exact (north_star)"""
    for i, g in _pairs(po, L, idxs):
        o = po.Diagram(g, level=0)
        d = mc.Diagram(L, g.ext_pos, g.chords(), host_only=True, flags=mc.FLAG_NO_TABLES)
        assert d.id() == i == o.id
        assert d.info()["class"] == po.graph_class(g)
        assert d.subgraphs() == o.subgraphs()
        assert d.forests() == o.forests()
        assert d.terms() == o.terms()
        deg, Z, Cn = d.sampler_tables()
        odeg, oZ, oC = o.sampler_tables()
        assert np.array_equal(deg, odeg) and np.array_equal(Z, oZ) and Cn == oC
        d.close()


def test_sampler_tables_other_options(po, mc):
    g = po.graph_get(3, 7)
    o = po.Diagram(g, deg_floor=0.75, deg_cap=1.25, level=0)
    d = mc.Diagram(3, g.ext_pos, g.chords(), deg_floor=0.75, deg_cap=1.25, host_only=True, flags=mc.FLAG_NO_TABLES)
    assert np.array_equal(d.sampler_tables()[1], o.sampler_tables()[1])


@pytest.mark.parametrize("L,idxs,npts", [(1, [0], 20), (2, range(6), 8), (3, [0, 7, 8, 29, 47], 2)])
def test_numerator_tables_against_oracle(po, mc, L, idxs, npts):
    """the device tables, interpreted in Python, reproduce the oracle's integrand and every term"""
    rng = np.random.default_rng(L)
    for i, g in _pairs(po, L, idxs):
        o = po.Diagram(g)
        d = mc.Diagram(L, g.ext_pos, g.chords(), host_only=True)
        b = Blob(d.blob())
        assert int(b.h["diag_id"]) == i and int(b.h["nterm"]) == o.nterm
        z = rng.dirichlet([1.0] * (3 * L), npts)
        ref = o.eval_z(z, wide=True, want_terms=True)
        for k in range(npts):
            f, terms = b.integrand(z[k])
            scale = np.max(np.abs(ref["terms"][k]))
            assert abs(f - ref["fwide"][k]) <= 1e-10 * scale, (i, k, f, ref["fwide"][k])
            assert np.allclose(terms, ref["terms"][k], rtol=1e-9, atol=1e-10 * scale)
        d.close()


def test_info_counts(po, mc):
    g = po.graph_get(3, 29)
    d = mc.Diagram(3, g.ext_pos, g.chords(), host_only=True)
    info = d.info()
    assert info["n_terms"] == po.Diagram(g, level=0).nterm == 8
    assert info["flop_per_sample"] > 0 and info["table_bytes"] == 8 * len(d.blob())


@pytest.mark.parametrize("L,idx,npts", [(2, 1, 6), (2, 3, 6), (3, 7, 3), (3, 18, 2)])
def test_oracle_wide_value_equals_exact_rational_value(po, mc, L, idx, npts):
    """exact pin: Fraction arithmetic on the product's tables at points drawn from Eq.(1) (deep corners,
    condition numbers up to 1e9) reproduces the oracle's binary128 value to the last binary64 digit"""
    from fractions import Fraction as Fr
    from exact_interp import ExactBlob
    g = po.graph_get(L, idx)
    o = po.Diagram(g)
    d = mc.Diagram(L, g.ext_pos, g.chords(), host_only=True)
    b = ExactBlob(d.blob())
    z, _, _ = o.sample(0, npts, 5)
    ref = o.eval_z(z, wide=True)
    for k in range(npts):
        fe = float(b.integrand([Fr(float(v)) for v in z[k]]))
        assert abs(ref["fwide"][k] - fe) <= 2e-16 * abs(fe), (k, fe, ref["fwide"][k])


def test_mrg32k3a_power_table_in_blob_equals_oracle(po, mc):
    """mc_options.flags bit 2 (S1b): the blob carries A^(2^k) mod m, k < 64, of both companion matrices;
    every entry against the oracle's own matrix power (pinned to the published A^(2^76) in test_oracle_rng.py). Without the flag
    the blob has no such section."""
    import blob_interp
    d = mc.Diagram(2, 2, [(0, 4), (1, 3)], host_only=True, flags=mc.FLAG_MRG32K3A | mc.FLAG_NO_TABLES)
    words = d.blob()
    h = np.frombuffer(words.tobytes(), blob_interp.HDR, 1)[0]
    assert h["rng"] == 1 and 0 < h["off_mrg"] and h["off_mrg"] + 576 <= h["off_stream"] and h["total_words"] == len(words)
    tab = np.frombuffer(words.tobytes(), "<u4", 2 * 64 * 9, int(h["off_mrg"]) * 8).reshape(2, 64, 3, 3)
    for comp in (0, 1):
        for k in range(64):
            assert np.array_equal(tab[comp, k].astype(np.uint64), po.mrg_matpow(comp, k)), (comp, k)
    d.close()
    d = mc.Diagram(2, 2, [(0, 4), (1, 3)], host_only=True, flags=mc.FLAG_NO_TABLES)
    h = np.frombuffer(d.blob().tobytes(), blob_interp.HDR, 1)[0]
    assert h["rng"] == 0 and h["off_mrg"] == 0
    d.close()


def test_mixture_tables_in_blob_equal_oracle(po, mc):
    """mc_options.mix_alpha > 0 (S5b): the blob carries the second channel's Z, 1/Deg, C and Deg of both channels; against the
    oracle's tables built with the same floors. Off by default: no such sections."""
    import blob_interp
    g = po.graph_get(3, 17)
    d = mc.Diagram(3, g.ext_pos, g.chords(), host_only=True, flags=mc.FLAG_NO_TABLES, mix_alpha=0.25, deg_floor2=0.6, deg_floor_ir2=0.4)
    w = d.blob()
    h = np.frombuffer(w.tobytes(), blob_interp.HDR, 1)[0]
    n = 1 << 9
    o1, o2 = po.Diagram(g, level=0), po.Diagram(g, level=0, deg_floor=0.6, deg_floor_ir=0.4)
    deg1, Z1, C1 = o1.sampler_tables()
    deg2, Z2, C2 = o2.sampler_tables()
    sec = lambda off: w[int(off):int(off) + n].view(np.float64)
    assert h["mix_alpha"] == 0.25 and h["C2"] == C2 and h["C"] == C1
    assert np.array_equal(sec(h["off_Z"]), Z1) and np.array_equal(sec(h["off_Z2"]), Z2)
    assert np.array_equal(sec(h["off_deg1"]), deg1) and np.array_equal(sec(h["off_deg2"]), deg2)
    inv2 = sec(h["off_invdeg2"])
    assert np.array_equal(inv2[1:n - 1], 1.0 / deg2[1:n - 1])
    d.close()
    d = mc.Diagram(3, g.ext_pos, g.chords(), host_only=True, flags=mc.FLAG_NO_TABLES)
    h = np.frombuffer(d.blob().tobytes(), blob_interp.HDR, 1)[0]
    assert h["mix_alpha"] == 0.0 and h["off_Z2"] == 0 and h["off_deg1"] == 0
    d.close()
    with pytest.raises(mc.McError):
        mc.Diagram(3, g.ext_pos, g.chords(), host_only=True, flags=mc.FLAG_NO_TABLES, mix_alpha=1.0, deg_floor2=0.6)
    with pytest.raises(mc.McError):
        mc.Diagram(3, g.ext_pos, g.chords(), host_only=True, flags=mc.FLAG_NO_TABLES, mix_alpha=0.2, deg_floor2=0.0)
