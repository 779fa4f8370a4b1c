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
