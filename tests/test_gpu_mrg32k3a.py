"""GPU parity of the second random stream, MRG32k3a (the generator of the paper's "Calc 1"; mc_options.flags bit 2;
DESIGN.md S1b). The CUDA path (stored matrix powers, folding reduction mod 2^32 - c, sequential
outputs) against the oracle (square-and-multiply at every call, plain %): coordinates, density and sector bit for bit, at the
start of the sequence, at large sample indices and diagram ids (positions up to 2^63), then the integral on both streams."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

CASES = [  # (L, e, chords, first sample)
    (1, 1, [(0, 2)], 0),
    (2, 2, [(0, 4), (1, 3)], 0),
    (2, 1, [(0, 3), (2, 4)], (1 << 38) - 700),                       # the last samples a diagram can own
    (3, 3, [(0, 6), (1, 5), (2, 4)], 123456789012),
    (5, 4, [(0, 10), (1, 9), (2, 8), (3, 7), (5, 6)], (1 << 37) + 5),  # a 5-loop graph (28 uniforms per point)
]


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")


@pytest.mark.parametrize("L,e,chords,first", CASES)
def test_points_bit_exact_on_the_mrg32k3a_stream(po, L, e, chords, first):
    _need_gpu()
    from paper_1905_08007_b200 import binding as mc
    n, seed = 600, (0x9E3779B9 << 32) | 0xFFFFFFF7
    o = po.Diagram(po.OracleGraph.make(L, e, chords), level=0)
    zp, _, _ = o.sample(first, n, seed)
    o.set_generator(1)
    zo, p_o, ord_o = o.sample(first, n, seed)
    d = mc.Diagram(L, e, chords, flags=mc.FLAG_MRG32K3A | mc.FLAG_NO_DD)
    M = 3 * L
    z = torch.zeros(n, M, dtype=torch.float64, device="cuda")
    order = torch.zeros(n, M, dtype=torch.int32, device="cuda")
    p = torch.zeros(n, dtype=torch.float64, device="cuda")
    d.eval_points(first, n, seed, torch.cuda.current_stream().cuda_stream, z=z, order=order, p=p)
    torch.cuda.synchronize()
    assert np.array_equal(z.cpu().numpy(), zo) and np.array_equal(p.cpu().numpy(), p_o) and np.array_equal(order.cpu().numpy(), ord_o)
    assert not np.array_equal(zo, zp)                                   # and it is not the Philox stream
    d.close()


def test_last_diagram_id_and_range_limits(po):
    """diagram id 6353 (the last 5-loop graph) at the last sample index: position (6353 2^38 + 2^38 - 1) 64 of the sequence;
    one sample further is refused (MC_EINVAL), on every entry point that draws points"""
    _need_gpu()
    from paper_1905_08007_b200 import binding as mc
    g = po.all_graphs(5)[-1]
    o = po.Diagram(g, level=0)
    o.set_generator(1)
    first, n, seed = (1 << 38) - 64, 64, 7
    zo, p_o, ord_o = o.sample(first, n, seed)
    d = mc.Diagram(5, g.ext_pos, g.chords(), flags=mc.FLAG_MRG32K3A | mc.FLAG_NO_DD)
    assert d.id() == 6353
    st = torch.cuda.current_stream().cuda_stream
    z = torch.zeros(n, 15, dtype=torch.float64, device="cuda")
    p = torch.zeros(n, dtype=torch.float64, device="cuda")
    d.eval_points(first, n, seed, st, z=z, p=p)
    torch.cuda.synchronize()
    assert np.array_equal(z.cpu().numpy(), zo) and np.array_equal(p.cpu().numpy(), p_o)
    acc = torch.zeros(2, dtype=torch.float64, device="cuda")
    cnt = torch.zeros(2, dtype=torch.int64, device="cuda")
    for call in (lambda: d.eval_points(first, n + 1, seed, st, z=None, p=p),
                 lambda: d.integrate(first + 1, n, seed, st, acc[0:1], acc[1:2], cnt[0:1], cnt[1:2]),
                 lambda: d.integrate_static(1 << 38, 1, seed, st, acc[0:1], acc[1:2], cnt[0:1], cnt[1:2]),
                 lambda: mc.Batch([d], 1024).integrate(first + 1, n, seed, st, acc[0:1], acc[1:2], cnt[0:1], cnt[1:2])):
        with pytest.raises(mc.McError) as ei:
            call()
        assert ei.value.code == mc.MC_EINVAL
    d.close()


def test_integrals_on_both_streams_agree(po):
    """the six 2-loop graph values on the MRG32k3a stream against the Philox stream (independent samples:
    within their errors), the single-diagram path against the batch path on the same MRG samples (equal sums), and a short
    range against the oracle's own integration on that stream (fixed point set: relative 1e-9)"""
    _need_gpu()
    from paper_1905_08007_b200 import binding as mc
    st = torch.cuda.current_stream().cuda_stream
    graphs = po.all_graphs(2)
    n, seed = 400000, 2024
    dm = [mc.Diagram(2, g.ext_pos, g.chords(), flags=mc.FLAG_MRG32K3A) for g in graphs]
    dp = [mc.Diagram(2, g.ext_pos, g.chords()) for g in graphs]
    bm = mc.Batch(dm, n)
    S = torch.zeros(2, len(graphs), dtype=torch.float64, device="cuda")
    Cn = torch.zeros(2, len(graphs), dtype=torch.int64, device="cuda")
    bm.integrate(0, n, seed, st, S[0], S[1], Cn[0], Cn[1])
    torch.cuda.synchronize()
    sm = S.cpu().numpy()
    assert Cn[1].sum().item() == 0
    tot_m = tot_p = var = 0.0
    for j, g in enumerate(graphs):
        s1, s2, _, nd = dm[j].integrate_host(0, n, seed)
        assert nd == 0 and abs(s1 - sm[0, j]) <= 1e-12 * abs(s1) + 1e-9 and abs(s2 - sm[1, j]) <= 1e-9 * s2
        q1, q2, _, _ = dp[j].integrate_host(0, n, seed)
        am, ap = s1 / n, q1 / n
        vm, vp = (s2 / n - am * am) / n, (q2 / n - ap * ap) / n
        assert abs(am - ap) <= 4.5 * np.sqrt(vm + vp), (g.key(), am, ap, np.sqrt(vm + vp))
        tot_m += am; tot_p += ap; var += vm + vp
    assert abs(tot_m - tot_p) <= 4.0 * np.sqrt(var)
    # oracle on the same stream, mode 2 (binary64 with binary128 where the oracle's truth flag is set)
    g = graphs[3]
    o = po.Diagram(g)
    o.set_generator(1)
    os1, os2, _ = o.integrate(1000, 20000, seed, mode=2)
    s1, s2, _, _ = dm[3].integrate_host(1000, 20000, seed)
    assert abs(s1 - os1) <= 1e-9 * abs(os1) and abs(s2 - os2) <= 1e-9 * os2
    for d in dm + dp:
        d.close()
