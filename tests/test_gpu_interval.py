"""GPU test of the interval tier (mc_eval_z_interval, "interval arithmetic"): the enclosure [lo, hi] computed with
directed rounding must contain the oracle's binary128 value of the integrand at the same coordinates — at well-conditioned
points, where it is narrow, and at points drawn from Eq.(1), where the subtraction terms cancel by many orders of magnitude
and it is wide — and the library's own binary64 value. SURVEY.md section 8(f) rank 3."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

CASES = [(2, 2, [(0, 4), (1, 3)]), (3, 1, [(0, 6), (2, 3), (4, 5)]), (3, 3, [(0, 6), (1, 5), (2, 4)]), (4, 3, [(0, 8), (1, 7), (2, 4), (5, 6)])]


@pytest.mark.parametrize("L,e,chords", CASES)
def test_interval_encloses_oracle_and_binary64_values(po, L, e, chords):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1905_08007_b200 import binding as mc
    st = torch.cuda.current_stream().cuda_stream
    o = po.Diagram(po.OracleGraph.make(L, e, chords))
    d = mc.Diagram(L, e, chords)
    M = 3 * L
    zs, _, _ = o.sample(0, 300, 7)                                   # points of Eq.(1): deep in the corners of the simplex
    zf = np.random.default_rng(L).dirichlet(np.ones(M), size=200)    # flat points: well conditioned
    z = np.vstack([zs, zf])
    n = len(z)
    zt = torch.tensor(z, device="cuda")
    lo, hi, f64 = (torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(3))
    d.eval_z_interval(n, zt, st, lo, hi)
    d.eval_z(n, zt, st, f64=f64)
    torch.cuda.synchronize()
    lo, hi, f64 = lo.cpu().numpy(), hi.cpu().numpy(), f64.cpu().numpy()
    fw = o.eval_z(z, wide=True)["fwide"]                              # binary128, rounded to binary64: half an ulp off the true value
    assert np.all(lo <= hi)
    fin = np.isfinite(lo) & np.isfinite(hi)
    assert fin.mean() > 0.95                                          # an interval division by an interval around 0 is rare
    slack = 4e-16 * np.abs(fw)
    assert np.all((lo - slack <= fw)[fin]) and np.all((fw <= hi + slack)[fin]), int((~((lo - slack <= fw) & (fw <= hi + slack)) & fin).sum())
    assert np.all(((lo <= f64) & (f64 <= hi))[fin & np.isfinite(f64)])   # the round-to-nearest evaluation of the same expression
    relw = (hi - lo) / np.abs(fw)
    assert np.median(relw[300:][fin[300:]]) < 1e-9                    # flat points: narrow
    # the width really is a bound on what binary64 lost
    assert np.all((np.abs(f64 - fw) <= (hi - lo) + slack)[fin & np.isfinite(f64)])
    d.close()
