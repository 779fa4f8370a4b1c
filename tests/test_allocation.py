"""Sample allocation across the graphs of a set.
CPU: the allocation rule against its closed form. GPU: per-diagram sample ranges of mc_batch_integrate_counts against
the per-diagram entry point on the same ranges."""
import math

import numpy as np
import pytest


def test_allocation_rule_closed_form():
    """minimise sum sigma_j^2 / n_j at fixed sum n_j cost_j: n_j = budget * sigma_j / (sqrt(cost_j) * sum_k sigma_k sqrt(cost_k))"""
    from paper_1905_08007_b200 import binding as mc
    sigma, cost, budget = np.array([1.0, 2.0, 0.5, 0.0]), np.array([1.0, 4.0, 9.0, 1.0]), 6.5e6
    n = mc.allocate_samples(sigma, cost, budget, n_min=10).astype(float)
    norm = (sigma * np.sqrt(cost)).sum()
    want = np.maximum(10, np.rint(budget * sigma / (np.sqrt(cost) * norm)))
    assert np.array_equal(n, want)
    assert abs((n[:3] * cost[:3]).sum() - budget) <= 3 * cost.max()                 # the budget is spent (up to rounding)
    # it beats the equal split of the same budget
    eq = budget / cost.sum()
    var_alloc = (sigma[:3] ** 2 / n[:3]).sum()
    var_equal = (sigma[:3] ** 2 / eq).sum()
    assert var_alloc < var_equal
    # Lagrange condition: sigma_j^2 / (n_j^2 cost_j) equal for all j with sigma_j > 0
    lam = sigma[:3] ** 2 / (n[:3] ** 2 * cost[:3])
    assert np.allclose(lam, lam[0], rtol=1e-5)
    with pytest.raises(mc.McError):
        mc.allocate_samples([1.0], [0.0], 10.0)


@pytest.mark.gpu
def test_batch_with_per_diagram_ranges_matches_per_diagram_calls():
    import torch
    from paper_1905_08007_b200 import binding as mc
    st = torch.cuda.current_stream().cuda_stream
    graphs = [(2, 2, [(0, 4), (1, 3)]), (3, 1, [(0, 6), (2, 4), (3, 5)]), (2, 1, [(0, 4), (2, 3)]), (3, 3, [(0, 6), (1, 5), (2, 4)])]
    ds = [mc.Diagram(*g) for g in graphs]
    cap = 4096
    b = mc.Batch(ds, cap)
    first = [5, 1000003, 77, 12]
    n = [3001, 0, 9999, 130]                       # one empty range, one longer than the capacity (three passes), ragged tails
    S = torch.zeros(2, 4, dtype=torch.float64, device="cuda")
    C = torch.zeros(2, 4, dtype=torch.int64, device="cuda")
    b.integrate_counts(first, n, 11, st, S[0], S[1], C[0], C[1])
    torch.cuda.synchronize()
    s, c = S.cpu().numpy(), C.cpu().numpy()
    for j, d in enumerate(ds):
        if n[j] == 0:
            assert s[0, j] == 0 and s[1, j] == 0 and c[0, j] == 0
            continue
        r1, r2, nf, nd = d.integrate_host(first[j], n[j], 11, st)
        assert abs(s[0, j] - r1) <= 1e-12 * math.sqrt(n[j] * r2) and abs(s[1, j] - r2) <= 1e-12 * r2, (j, s[:, j], r1, r2)
        assert c[0, j] == nf and c[1, j] == nd == 0
    # a uniform call afterwards is unaffected by the per-diagram arrays left on the device
    h = b.integrate_host(3, 500, 11, st)
    for j, d in enumerate(ds):
        r1, r2, _, _ = d.integrate_host(3, 500, 11, st)
        assert abs(h[0][j] - r1) <= 1e-12 * math.sqrt(500 * r2)


def test_campaign_mirror_identification_matches_table_1(po):
    """campaign.py runs ONE graph of every mirror pair and counts its estimate twice (PAPER.md:153 fn5): its host logic against the
    paper's N_diag per class (tests/golden/paper_table1_ndiag.txt), the total 3213 and the
    oracle's own mirror map; the multiplicities add up to all 6354 graphs. No GPU."""
    from conftest import read_golden
    from paper_1905_08007_b200 import campaign, workloads
    graphs = workloads.all_graphs(5)
    reps = campaign.representatives(graphs)
    assert len(graphs) == 6354 and len(reps) == 3213 and sum(m for _, _, m in reps) == 6354
    want = {(int(k), int(m), int(n)): int(c) for k, m, n, c in read_golden("paper_table1_ndiag.txt")}
    got = {}
    for _, g, _ in reps:
        got[workloads.graph_class(g)] = got.get(workloads.graph_class(g), 0) + 1
    assert got == want
    og = po.all_graphs(5)
    for i, g, m in reps[::97]:
        mk = po.graph_mirror(og[i]).key()
        assert campaign.mirror(g) == mk and (m == 1) == (mk == og[i].key())
    assert len(campaign.representatives(graphs)[::8]) == 402          # the --stride 8 sample of DESIGN.md section 7
