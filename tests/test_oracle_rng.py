"""Pins of the oracle's random stream and deterministic pow (not GPU)."""
import math

import numpy as np

from conftest import read_golden


def test_philox_known_answers(po):
    for row in read_golden("philox4x32_10_kat.txt"):
        v = [int(x, 16) for x in row]
        assert po.philox(v[0:4], v[4:6]) == v[6:10]


def test_uniform_construction(po):
    lib = po.lib()
    assert lib.oracle_u01(0, 0) == 0.5 * 2.0 ** -52
    assert lib.oracle_u01(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 0.5 * 2.0 ** -52
    assert lib.oracle_u01(0x80000000, 0) == 0.5 + 0.5 * 2.0 ** -52
    # stream layout: uniform r comes from Philox block r//2 of ctr=(idx_lo, idx_hi, block, diagram)
    idx, diag, seed = (5 << 32) | 77, 9, (3 << 32) | 11
    for r in range(6):
        w = po.philox([77, 5, r // 2, 9], [11, 3])
        x, y = (w[2], w[3]) if r & 1 else (w[0], w[1])
        assert lib.oracle_sample_uniform(idx, diag, seed, r) == ((x >> 6) * 2.0 ** 26 + (y >> 6) + 0.5) * 2.0 ** -52


def test_uniform_moments(po):
    lib = po.lib()
    u = np.array([lib.oracle_sample_uniform(i, 0, 123, 0) for i in range(20000)])
    assert abs(u.mean() - 0.5) < 4 / math.sqrt(12 * len(u))
    assert abs((u ** 2).mean() - 1 / 3) < 0.01
    assert u.min() > 0 and u.max() < 1


def test_det_pow_accuracy_and_monotonicity(po):
    lib = po.lib()
    rng = np.random.default_rng(1)
    worst = 0.0
    for u, d in zip(rng.random(4000), rng.choice([0.5, 0.75, 1.0, 1.5, 2.0, 2.5, 3.0], 4000)):
        got, want = lib.oracle_det_pow(u, 1.0 / d), u ** (1.0 / d)
        worst = max(worst, abs(got - want) / want)
    assert worst < 5e-15
    # extreme uniforms the stream can produce
    for u in (0.5 * 2.0 ** -52, 1 - 0.5 * 2.0 ** -52, 2.0 ** -30):
        for d in (0.5, 1.0, 3.0):
            got, want = lib.oracle_det_pow(u, 1.0 / d), u ** (1.0 / d)
            assert abs(got - want) <= 5e-15 * want
    assert abs(lib.oracle_det_log2(0.7) - math.log2(0.7)) < 1e-15
    assert abs(lib.oracle_det_exp2(-3.3) - 2 ** -3.3) < 1e-15 * 2 ** -3.3
    us = np.sort(rng.random(2000))
    t = [lib.oracle_det_pow(x, 2.0) for x in us]
    assert all(b >= a for a, b in zip(t, t[1:]))


# ---------------------------------------------------------------- MRG32k3a (S1b)
M1, M2 = 4294967087, 4294944443


def test_mrg32k3a_jump_matrices_published_constants(po):
    """A^(2^76) and A^(2^127) of both components against the constants published with RngStreams (tests/golden/mrg32k3a_lecuyer.txt):
    pins multipliers, signs, lags and moduli of the two recurrences and the oracle's matrix power."""
    rows = read_golden("mrg32k3a_lecuyer.txt")
    assert len(rows) == 4
    for r in rows:
        comp, e, want = int(r[0]), int(r[1]), np.array([int(x) for x in r[2:]], dtype=np.uint64).reshape(3, 3)
        assert np.array_equal(po.mrg_matpow(comp, e), want), (comp, e)


def _py_mrg(state, n):
    """the two recurrences and the output w_n = (x1_n - x2_n) mod m1 with Python integers (no modular tricks)"""
    s1, s2, out = list(state[:3]), list(state[3:]), []
    for _ in range(n):
        x1 = (1403580 * s1[1] - 810728 * s1[0]) % M1
        x2 = (527612 * s2[2] - 1370589 * s2[0]) % M2
        s1, s2 = [s1[1], s1[2], x1], [s2[1], s2[2], x2]
        out.append((x1 - x2) % M1)
    return out


def test_mrg32k3a_stepping_equals_skipping(po):
    """n single steps (mrg_next: its own code) = one skip by the pinned matrix power, and both = the plain-integer recurrence;
    the composition law skip(a) o skip(b) = skip(a + b) far beyond what stepping can reach"""
    st = [12345] * 6
    ref = _py_mrg(st, 3000)
    assert [int(x) for x in po.mrg32k3a(st, 0, 3000)] == ref
    for n in (1, 2, 3, 63, 64, 1000, 2990):
        assert [int(x) for x in po.mrg32k3a(st, n, 8)] == ref[n:n + 8]
    st2 = [1, 2, 3, 4294944442, 7, 4294967086 % M2]
    assert [int(x) for x in po.mrg32k3a(st2, 500, 5)] == _py_mrg(st2, 505)[500:]
    for e, mult in ((40, 3), (62, 1), (63, 1)):                       # A^(mult 2^e) = (A^(2^(e-1)))^(2 mult)
        for comp in (0, 1):
            m = (M1, M2)[comp]
            h = po.mrg_matpow(comp, e - 1, mult).astype(object)
            assert np.array_equal((h.dot(h)) % m, po.mrg_matpow(comp, e, mult).astype(object))


def test_mrg32k3a_stream_layout(po):
    """DESIGN.md S1b: state (1 + seed_lo mod (m-1), 1 + seed_hi mod (m-1), 12345) per component; sample idx of diagram id owns
    outputs (id 2^38 + idx) 64 ...; uniform r = u01(w_2r, w_2r+1)"""
    lib = po.lib()
    seed = (12344 << 32) | 12344                                          # -> L'Ecuyer's reference state, all 12345
    ref = _py_mrg([12345] * 6, 64 * 4)
    for idx in (0, 1, 3):
        for r in (0, 1, 13, 27):
            a, b = ref[64 * idx + 2 * r], ref[64 * idx + 2 * r + 1]
            assert lib.oracle_sample_uniform_mrg(idx, 0, seed, r) == ((a >> 6) * 2.0 ** 26 + (b >> 6) + 0.5) * 2.0 ** -52
    seed = (0xFFFFFFFF << 32) | 0xFFFFFFF0
    st = [1 + 0xFFFFFFF0 % (M1 - 1), 1 + 0xFFFFFFFF % (M1 - 1), 12345, 1 + 0xFFFFFFF0 % (M2 - 1), 1 + 0xFFFFFFFF % (M2 - 1), 12345]
    idx, diag, r = (1 << 38) - 1, (1 << 20) - 1, 27                       # the last sample of the last diagram: position < 2^64
    w = po.mrg32k3a(st, ((diag << 38) + idx) * 64 + 2 * r, 2)
    assert lib.oracle_sample_uniform_mrg(idx, diag, seed, r) == ((int(w[0]) >> 6) * 2.0 ** 26 + (int(w[1]) >> 6) + 0.5) * 2.0 ** -52


def test_mrg32k3a_uniform_moments_and_sampler(po):
    lib = po.lib()
    u = np.array([lib.oracle_sample_uniform_mrg(i, 3, 123, 0) for i in range(20000)])
    assert abs(u.mean() - 0.5) < 4 / math.sqrt(12 * len(u)) and abs((u ** 2).mean() - 1 / 3) < 0.01 and u.min() > 0 and u.max() < 1
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 4 / math.sqrt(len(u))                 # neighbouring samples: 64 outputs apart
    # the sampler on this stream: same invariants as on Philox, other points
    d = po.Diagram(po.OracleGraph.make(2, 2, [(0, 4), (1, 3)]), level=0)
    zp, pp, _ = d.sample(0, 4000, 11)
    d.set_generator(1)
    z, p, order = d.sample(0, 4000, 11)
    assert not np.array_equal(z, zp)
    assert np.all(z > 0) and np.allclose(z.sum(1), 1.0, rtol=0, atol=1e-14) and np.allclose(d.density(z), p, rtol=1e-9)
    zs = np.take_along_axis(z, order.astype(np.int64), axis=1)
    assert np.all(np.diff(zs, axis=1) <= 0)
    a = np.array([1.0, 0.0, 2.0, 0.5, 0.0, 1.0])                         # Dirichlet closed form through the sampler (north_star pin)
    z, p, _ = d.sample(0, 100000, 17)
    w = np.prod(z ** a, axis=1) / p
    exact = math.exp(sum(math.lgamma(x + 1) for x in a) - math.lgamma(a.sum() + d.M))
    assert abs(w.mean() - exact) < 5 * w.std() / math.sqrt(len(w))
