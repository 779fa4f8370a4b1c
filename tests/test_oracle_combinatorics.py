"""Pins of the oracle's combinatorics against what the paper prints (not GPU)."""
from collections import Counter

import pytest

from conftest import read_golden


def test_graph_counts(po):
    # valid 1PI vertex graphs without lepton loops; L=5 mirror-identified count is PAPER.md:91
    assert [po.graph_count(L) for L in (1, 2, 3, 4)] == [1, 6, 50, 518]


def _mirror_classes(po, L):
    graphs = po.all_graphs(L)
    keys = {g.key(): i for i, g in enumerate(graphs)}
    seen, reps = set(), []
    n_sym = 0
    for g in graphs:
        if g.key() in seen:
            continue
        m = po.graph_mirror(g)
        assert m.key() in keys, "mirror image must be a valid graph of the same order"
        seen.add(g.key()); seen.add(m.key())
        n_sym += m.key() == g.key()
        reps.append(g)
    return graphs, reps, n_sym


def test_five_loop_counts_and_table1_classes(po):
    graphs, reps, n_sym = _mirror_classes(po, 5)
    assert len(graphs) == 6354
    want_total = int([r for r in read_golden("paper_values.txt") if r[0] == "n_integrands_5loop"][0][1])
    assert len(reps) == want_total == 3213
    got = Counter(po.graph_class(g) for g in reps)
    want = {(int(k), int(m), int(n)): int(c) for k, m, n, c in read_golden("paper_table1_ndiag.txt")}
    assert dict(got) == want
    # a graph and its mirror image are in the same class (m>=n by definition)
    for g in graphs[::97]:
        assert po.graph_class(g) == po.graph_class(po.graph_mirror(g))


def test_canonical_ids_are_positions_in_enumeration(po):
    for L in (1, 2, 3):
        for i, g in enumerate(po.all_graphs(L)):
            assert po.graph_id(g) == i
    g = po.graph_get(5, 4321)
    assert po.graph_id(g) == 4321


def test_invalid_graphs_rejected(po):
    G = po.OracleGraph.make
    assert po.graph_validate(G(1, 1, [(0, 2)])) == 0
    assert po.graph_validate(G(1, 0, [(1, 2)])) != 0      # external-leg correction: line 0 uncovered
    assert po.graph_validate(G(2, 2, [(0, 1), (3, 4)])) != 0  # not 1PI
    assert po.graph_validate(G(2, 2, [(0, 1), (1, 4)])) != 0  # not a matching
    assert po.graph_validate(G(2, 2, [(0, 2), (1, 4)])) != 0  # chord ends on the external vertex


def test_two_loop_subgraphs_and_terms(po):
    """worked 2-loop instances of the forest-like formula (O1)"""
    G = po.OracleGraph.make
    lad = po.Diagram(G(2, 2, [(0, 4), (1, 3)]), level=0)
    assert lad.subgraphs() == [(1, 3, 1)]
    # A_G ; -A_G U_Gc ; -(L_G-U_G) A_Gc
    assert lad.terms() == [(0, -1, 1), (1, -1, -1), (1, 0, -1)]
    crossed = po.Diagram(G(2, 2, [(0, 3), (1, 4)]), level=0)
    assert crossed.subgraphs() == [] and crossed.terms() == [(0, -1, 1)]
    corner = po.Diagram(G(2, 1, [(0, 3), (2, 4)]), level=0)
    assert corner.subgraphs() == [(2, 4, 1)]                # vertex subgraph not containing e -> U only
    assert corner.terms() == [(0, -1, 1), (1, -1, -1)]
    se = po.Diagram(G(2, 1, [(0, 4), (2, 3)]), level=0)
    assert se.subgraphs() == [(2, 3, 0)] and se.terms() == [(0, -1, 1), (1, -1, -1)]


def test_forest_statistics(po):
    """max #subgraphs, #forests, #terms per graph and total #terms (DESIGN.md table; self-consistency)"""
    stats = {}
    for L in (1, 2, 3, 4):
        ds = [po.Diagram(g, level=0) for g in po.all_graphs(L)]
        stats[L] = (max(d.nsub for d in ds), max(d.nforest for d in ds), max(d.nterm for d in ds), sum(d.nterm for d in ds))
    assert stats[1] == (0, 1, 1, 1)
    assert stats[2] == (1, 2, 3, 12)
    assert stats[3] == (3, 6, 8, 181)
    assert stats[4] == (5, 16, 20, 3096)
    for d in ds[::37]:
        subs = d.subgraphs()
        for f in d.forests():
            members = [subs[i] for i in range(len(subs)) if f >> i & 1]
            for x in members:
                for y in members:
                    nested = (x[0] <= y[0] and y[1] <= x[1]) or (y[0] <= x[0] and x[1] <= y[1])
                    disjoint = x[1] < y[0] or y[1] < x[0]
                    assert nested or disjoint
