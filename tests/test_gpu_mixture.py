"""GPU parity of the defensive mixture of two Eq.(1) densities (mc_options.mix_alpha; S5b):
coordinates, mixture density and Hepp sector bit for bit against the oracle on both random streams, integrand values of the mixed
points against the oracle, and the integral with and without the mixture (any positive density is unbiased)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

MIX = dict(mix_alpha=0.35, deg_floor2=0.6, deg_floor_ir2=0.4)
CASES = [  # (L, e, chords, first sample, MRG32k3a?)
    (1, 1, [(0, 2)], 0, False),
    (2, 2, [(0, 4), (1, 3)], 0, False),
    (2, 1, [(0, 3), (2, 4)], 5_000_000_000, True),
    (3, 1, [(0, 6), (2, 3), (4, 5)], 77, False),
    (3, 3, [(0, 6), (1, 5), (2, 4)], 77, True),
    (5, 4, [(0, 10), (1, 9), (2, 8), (3, 7), (5, 6)], 1000, False),
    (5, 2, [(0, 4), (1, 10), (3, 7), (5, 6), (8, 9)], 1000, True),
]


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")


@pytest.mark.parametrize("L,e,chords,first,mrg", CASES)
def test_mixture_points_bit_exact(po, L, e, chords, first, mrg):
    _need_gpu()
    from paper_1905_08007_b200 import binding as mc
    n, seed = 800, (0x1234567 << 32) | 0x89ABCDE
    o = po.Diagram(po.OracleGraph.make(L, e, chords), level=0)
    z1, _, _ = o.sample(first, n, seed) if not mrg else (None, None, None)
    o.set_mixture(MIX["mix_alpha"], MIX["deg_floor2"], MIX["deg_floor_ir2"])
    if mrg:
        o.set_generator(1)
    zo, p_o, ord_o = o.sample(first, n, seed)
    d = mc.Diagram(L, e, chords, flags=(mc.FLAG_MRG32K3A if mrg else 0) | mc.FLAG_NO_DD, **MIX)
    M = 3 * L
    z = torch.zeros(n, M, dtype=torch.float64, device="cuda")
    order = torch.zeros(n, M, dtype=torch.int32, device="cuda")
    p = torch.zeros(n, dtype=torch.float64, device="cuda")
    d.eval_points(first, n, seed, torch.cuda.current_stream().cuda_stream, z=z, order=order, p=p)
    torch.cuda.synchronize()
    assert np.array_equal(z.cpu().numpy(), zo) and np.array_equal(p.cpu().numpy(), p_o) and np.array_equal(order.cpu().numpy(), ord_o)
    if z1 is not None and L > 1:
        moved = (~np.all(zo == z1, axis=1)).mean()                       # the second channel really is used, about alpha of the time
        assert 0.25 < moved < 0.45, moved
    d.close()


def test_mixture_integrals(po):
    """the six 2-loop graphs: estimate with the mixture against the estimate without (independent of the density, within errors);
    single-diagram path = batch path on the same samples; a short range against the oracle's own integration on the same mixed
    stream (fixed point set, relative 1e-9); a 3-loop graph: values of the mixed points against the oracle's binary128 values"""
    _need_gpu()
    from paper_1905_08007_b200 import binding as mc
    st = torch.cuda.current_stream().cuda_stream
    graphs = po.all_graphs(2)
    n, seed = 400000, 31
    dm = [mc.Diagram(2, g.ext_pos, g.chords(), **MIX) for g in graphs]
    dp = [mc.Diagram(2, g.ext_pos, g.chords()) for g in graphs]
    S = torch.zeros(2, len(graphs), dtype=torch.float64, device="cuda")
    Cn = torch.zeros(2, len(graphs), dtype=torch.int64, device="cuda")
    mc.Batch(dm, n).integrate(0, n, seed, st, S[0], S[1], Cn[0], Cn[1])
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
    assert abs(tot_m + 0.344166) <= 4.0 * np.sqrt(sum((sm[1, j] / n - (sm[0, j] / n) ** 2) / n for j in range(len(graphs))))   # north_star's 2-loop value
    o = po.Diagram(graphs[3])
    o.set_mixture(MIX["mix_alpha"], MIX["deg_floor2"], MIX["deg_floor_ir2"])
    os1, os2, _ = o.integrate(1000, 20000, seed, mode=2)
    s1, s2, _, _ = dm[3].integrate_host(1000, 20000, seed)
    assert abs(s1 - os1) <= 1e-9 * abs(os1) and abs(s2 - os2) <= 1e-9 * os2
    for d in dm + dp:
        d.close()
    # 3 loops: per-point values at the mixed points
    g3 = po.OracleGraph.make(3, 2, [(0, 6), (1, 3), (4, 5)])
    o3 = po.Diagram(g3)
    o3.set_mixture(MIX["mix_alpha"], MIX["deg_floor2"], MIX["deg_floor_ir2"])
    zo, p_o, _ = o3.sample(0, 512, 9)
    fw = o3.eval_z(zo, wide=True)["fwide"]
    d3 = mc.Diagram(3, 2, [(0, 6), (1, 3), (4, 5)], **MIX)
    f = torch.zeros(512, dtype=torch.float64, device="cuda")
    p = torch.zeros(512, dtype=torch.float64, device="cuda")
    flag = torch.zeros(512, dtype=torch.uint8, device="cuda")
    d3.eval_points(0, 512, 9, st, p=p, f=f, flag=flag)
    torch.cuda.synchronize()
    f, flag = f.cpu().numpy(), flag.cpu().numpy()
    assert np.array_equal(p.cpu().numpy(), p_o)
    rel = np.abs(f - fw) <= 1e-10 * np.abs(fw)
    absw = np.abs(f - fw) <= 1e-10 * p_o
    assert np.all(rel[flag == 0]) and np.all(absw[flag == 2]) and np.all((rel | absw)[flag == 1])
    d3.close()
