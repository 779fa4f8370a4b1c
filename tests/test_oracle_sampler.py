"""Pins of the oracle's Hepp-sector sampler, Eq.(1) of the paper. Not GPU."""
import itertools
import math

import numpy as np
import pytest

G2 = [(2, 1, [(0, 3), (2, 4)]), (2, 1, [(0, 4), (2, 3)]), (2, 2, [(0, 3), (1, 4)]), (2, 2, [(0, 4), (1, 3)])]


def _diag(po, L, e, chords, **kw):
    return po.Diagram(po.OracleGraph.make(L, e, chords), level=0, **kw)


def test_points_on_simplex_and_in_their_sector(po):
    d = _diag(po, 2, 2, [(0, 4), (1, 3)])
    z, p, order = d.sample(0, 5000, 11)
    assert np.all(z > 0) and np.allclose(z.sum(1), 1.0, rtol=0, atol=1e-14)
    zs = np.take_along_axis(z, order.astype(np.int64), axis=1)
    assert np.all(np.diff(zs, axis=1) <= 0)          # z_{j_1} >= ... >= z_{j_M}
    assert np.all(np.sort(order, axis=1) == np.arange(d.M))
    assert np.all(p > 0) and np.all(np.isfinite(p))


def test_density_of_drawn_point_equals_eq1_recomputed_from_z(po):
    """p returned by the draw (C * prod u / prod z) against Eq.(1) evaluated from z alone (sort, tail sets)"""
    for (L, e, ch) in G2 + [(3, 1, [(0, 6), (2, 3), (4, 5)])]:
        d = _diag(po, L, e, ch)
        z, p, _ = d.sample(100, 3000, 5)
        assert np.allclose(d.density(z), p, rtol=1e-9)


def test_sector_masses_sum_to_one_bruteforce(po):
    """1/C = sum over all M! orderings of prod_l 1/Deg(tail set): brute force against the subset DP"""
    d = _diag(po, 2, 1, [(0, 4), (2, 3)])
    deg, Z, Cn = d.sampler_tables()
    M = d.M
    tot = 0.0
    for perm in itertools.permutations(range(M)):
        w = 1.0
        for l in range(1, M):
            mask = sum(1 << x for x in perm[l:])
            w /= deg[mask]
        tot += w
    assert abs(tot * Cn - 1.0) < 1e-12
    assert np.all(deg[1:(1 << M) - 1] > 0)             # "positive numbers"


def test_sector_frequencies_chi2(po):
    d = _diag(po, 1, 1, [(0, 2)])
    deg, Z, Cn = d.sampler_tables()
    n = 60000
    _, _, order = d.sample(0, n, 3)
    counts = {}
    for o in map(tuple, order):
        counts[o] = counts.get(o, 0) + 1
    chi2 = 0.0
    for perm in itertools.permutations(range(3)):
        w = Cn
        for l in range(1, 3):
            w /= deg[sum(1 << x for x in perm[l:])]
        chi2 += (counts.get(perm, 0) - n * w) ** 2 / (n * w)
    assert chi2 < 25.0                                  # 5 dof, p ~ 1e-4


def test_ratio_variables_are_power_law(po):
    """t_l^Deg must be uniform (independent power-law ratios): KS test on the first ratio"""
    d = _diag(po, 2, 2, [(0, 3), (1, 4)])
    deg, _, _ = d.sampler_tables()
    z, _, order = d.sample(0, 20000, 9)
    zs = np.take_along_axis(z, order.astype(np.int64), axis=1)
    full = (1 << d.M) - 1
    masks = full & ~(1 << order[:, 0].astype(np.int64))
    u = (zs[:, 1] / zs[:, 0]) ** deg[masks]
    u.sort()
    ks = np.max(np.abs(u - (np.arange(len(u)) + 0.5) / len(u)))
    assert ks < 1.95 / math.sqrt(len(u))


@pytest.mark.parametrize("graph", G2 + [(1, 1, [(0, 2)])])
def test_dirichlet_closed_form_through_sampler(po, graph):
    """E_p[ prod z^a / p ] = prod Gamma(a_i+1)/Gamma(sum a + M)  (north_star pin)"""
    d = _diag(po, *graph)
    z, p, _ = d.sample(0, 200000, 17)
    rng = np.random.default_rng(4)
    for a in ([0.0] * d.M, list(rng.integers(0, 3, d.M).astype(float)), list(rng.random(d.M) * 1.5)):
        w = np.prod(z ** np.array(a), axis=1) / p
        exact = math.exp(sum(math.lgamma(x + 1) for x in a) - math.lgamma(sum(a) + d.M))
        err = w.std() / math.sqrt(len(w))
        assert abs(w.mean() - exact) < 5 * err, (a, w.mean(), exact, err)
        assert err < 0.05 * exact


def test_flat_sampled_integral_of_density_is_one(po):
    """int p = 1 with points drawn uniformly on the simplex (independent of the sampler's own draw)"""
    d = _diag(po, 1, 1, [(0, 2)], deg_floor=0.75)      # flat sampling of p has finite variance only for Deg > 1/2 on every set
    rng = np.random.default_rng(2)
    z = rng.dirichlet([1.0] * 3, 400000)
    w = d.density(z) / math.gamma(3)                   # flat density on the simplex is (M-1)!
    # heavy-tailed (p ~ 1/z^(1-Deg)): loose tolerance
    assert abs(w.mean() - 1.0) < 0.05


def test_deg_values(po):
    """Deg = -omega on I-closures, floored (S5): spot values on the 1-loop graph"""
    d = _diag(po, 1, 1, [(0, 2)], deg_floor=0.5)
    deg, _, _ = d.sampler_tables()
    # lines: e0=bit0, e1=bit1, photon=bit2.  {e0}: |s|-|e|/2 = 0.5 ; {photon}: 1 ; {e0,e1}: I-closure is the full set -> floor
    assert deg[0b001] == 0.5 and deg[0b010] == 0.5 and deg[0b100] == 1.0
    assert deg[0b011] == 0.5
    assert deg[0b101] == 1.5 and deg[0b110] == 1.5
    d2 = _diag(po, 1, 1, [(0, 2)], deg_floor=0.75, deg_cap=1.25)
    deg2, _, _ = d2.sampler_tables()
    assert deg2[0b001] == 0.75 and deg2[0b101] == 1.25
    # 2-loop corner graph: {e0,e1,photon0} is a tree in G but closes a loop in G/G_s (the counter-term) -> floor
    d3 = _diag(po, 2, 1, [(0, 3), (2, 4)], deg_floor=0.5)
    deg3, _, _ = d3.sampler_tables()
    assert deg3[0b010011] == 0.5


def test_defensive_mixture_of_two_eq1_densities(po):
    """DESIGN.md S5b: with probability alpha a point comes from a second Eq.(1) density and every weight is
    divided by the mixture. Pins: the density returned with the point equals (1 - alpha) p1(z) + alpha p2(z) recomputed from z alone
    (two separate table sets, sort + tail sets); the share of points that differ from the single-channel draw is alpha; the
    Dirichlet closed form still comes out (unbiased); alpha = 0 restores the single-channel stream bit for bit."""
    g = po.OracleGraph.make(3, 1, [(0, 6), (2, 3), (4, 5)])
    d = po.Diagram(g, level=0)
    d1 = po.Diagram(g, level=0)
    d2 = po.Diagram(g, level=0, deg_floor=0.5, deg_floor_ir=0.35)
    z0, p0, o0 = d.sample(0, 20000, 11)
    alpha = 0.3
    d.set_mixture(alpha, 0.5, 0.35)
    z, p, order = d.sample(0, 20000, 11)
    want = (1 - alpha) * d1.density(z) + alpha * d2.density(z)
    assert np.allclose(p, want, rtol=1e-9) and np.allclose(d.density(z), want, rtol=1e-12)
    moved = ~np.all(z == z0, axis=1)
    assert abs(moved.mean() - alpha) < 4 * math.sqrt(alpha * (1 - alpha) / len(z))
    assert np.array_equal(p[~moved] > p0[~moved] * (1 - alpha) * 0.999999, np.ones((~moved).sum(), bool))   # p >= (1 - alpha) p1 on the unmoved points
    zs = np.take_along_axis(z, order.astype(np.int64), axis=1)
    assert np.all(np.diff(zs, axis=1) <= 0) and np.allclose(z.sum(1), 1.0, rtol=0, atol=1e-14)
    zz, pp, _ = d.sample(0, 200000, 17)
    a = np.array([1.0, 0.0, 2.0, 0.5, 0.0, 1.0, 0.0, 0.25, 1.0])
    w = np.prod(zz ** a, axis=1) / pp
    exact = math.exp(sum(math.lgamma(x + 1) for x in a) - math.lgamma(a.sum() + d.M))
    assert abs(w.mean() - exact) < 5 * w.std() / math.sqrt(len(w))
    d.set_generator(1)                                                       # the channel uniform on the MRG32k3a stream: outputs 4(M-1), 4(M-1)+1
    zm, pm, _ = d.sample(0, 20000, 11)
    assert np.allclose(pm, (1 - alpha) * d1.density(zm) + alpha * d2.density(zm), rtol=1e-9)
    d.set_generator(0)
    d.set_mixture(0.0, 1.0)
    z1, p1, o1 = d.sample(0, 20000, 11)
    assert np.array_equal(z1, z0) and np.array_equal(p1, p0) and np.array_equal(o1, o0)
