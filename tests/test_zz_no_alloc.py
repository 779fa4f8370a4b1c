"""GPU test of mc_integrate_static (include/mcqed.h): the binary64 tier with its scratch in a file-scope
`static __device__` array, for callers that cannot call cudaMalloc. Collected last on purpose (zz): the run
uses `pytest -x`. The test passes alone in a fresh process and after the other GPU tests (it depends on no state
they leave behind; the static array keeps the last call's contents and the entry point clears what it needs).

Checked against the existing path: mc_integrate on a handle with flags bit 0 (binary64 tier only) runs the same
kernels in the same launch configuration with scratch owned by the handle, so the sums must agree to the 1e-12 the
other sum tests use (tests/test_gpu_parity.py), on two calls in a row.
"""
import pytest

pytestmark = pytest.mark.gpu


def test_static_scratch_entry_point_matches_existing_path_twice_in_a_row():
    import torch
    from paper_1905_08007_b200 import binding as mc
    assert torch.cuda.is_available()
    st = torch.cuda.current_stream().cuda_stream
    cases = [((2, 2, [(0, 4), (1, 3)]), 7, 50000, 42),            # 2-loop ladder, 3 terms
             ((3, 1, [(0, 6), (2, 4), (3, 5)]), 123457, mc.STATIC_MAX_SAMPLES, 9)]   # 3-loop with a self-energy insertion, at the size limit
    handles = []
    for graph, first, n, seed in cases:
        d_new = mc.Diagram(*graph)
        d_ref = mc.Diagram(*graph, flags=mc.FLAG_NO_DD)            # existing path, binary64 tier only
        handles.append((d_new, d_ref, first, n, seed))
    # two calls in a row on the new entry point (the second reuses the scratch the first one left behind), then the references
    new = []
    for d_new, _, first, n, seed in handles:
        s = torch.zeros(2, dtype=torch.float64, device="cuda")
        c = torch.zeros(2, dtype=torch.int64, device="cuda")
        d_new.integrate_static(first, n, seed, st, s[0:], s[1:], c[0:], c[1:])
        new.append((s, c))
    torch.cuda.synchronize()
    for (d_new, d_ref, first, n, seed), (s, c) in zip(handles, new):
        r = torch.zeros(2, dtype=torch.float64, device="cuda")
        rc = torch.zeros(2, dtype=torch.int64, device="cuda")
        d_ref.integrate(first, n, seed, st, r[0:], r[1:], rc[0:], rc[1:])
        torch.cuda.synchronize()
        s1, s2 = s.cpu().tolist()
        r1, r2 = r.cpu().tolist()
        assert r2 > 0 and abs(s1 - r1) <= 1e-12 * (n * r2) ** 0.5 and abs(s2 - r2) <= 1e-12 * r2, (s1, r1, s2, r2)
        assert c.cpu().tolist() == rc.cpu().tolist()
    # accumulation (+=) and a repeated call on dirty scratch give the same numbers again
    d_new, _, first, n, seed = handles[0]
    s, c = new[0]
    before = s.clone()
    d_new.integrate_static(first, n, seed, st, s[0:], s[1:], c[0:], c[1:])
    torch.cuda.synchronize()
    assert torch.allclose(s, 2 * before, rtol=1e-12, atol=0)
    # sizes beyond the static scratch are rejected with a clear error and nothing is launched
    l0 = mc.kernel_launch_count()
    with pytest.raises(mc.McError) as ei:
        d_new.integrate_static(0, mc.STATIC_MAX_SAMPLES + 1, seed, st, s[0:], s[1:], c[0:], c[1:])
    assert ei.value.code == mc.MC_ETOOBIG and "MC_STATIC_MAX_SAMPLES" in str(ei.value)
    assert mc.kernel_launch_count() == l0
    for d_new, d_ref, *_ in handles:
        d_new.close(); d_ref.close()
