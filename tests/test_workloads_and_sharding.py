"""CPU tests of the seeded workload generator (BASELINE.json configs) and of the multi-GPU host logic:
the path shards by disjoint sample-index ranges (replicas, no data-path collective)."""
import os
import subprocess
import sys
from collections import Counter

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_config_sets(po):
    from paper_1905_08007_b200 import workloads as w
    assert [len(w.all_graphs(L)) for L in (1, 2, 3, 4)] == [1, 6, 50, 518]
    assert w.philox4x32_10((0, 0, 0, 0), (0, 0)) == (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)
    assert len(w.config_graphs(0)) == 1 and len(w.config_graphs(1)) == 6 and len(w.config_graphs(2)) == 50
    c3, c4 = w.config_graphs(3), w.config_graphs(4)
    assert len(c3) == 128 and len({i for i, _ in c3}) == 128
    assert len(c4) == 256 and len({i for i, _ in c4}) == 256
    assert len(Counter(w.graph_class(g) for _, g in c4)) == 9          # spread over the paper's nine classes
    assert w.config_graphs(4) == c4                                    # seeded: reproducible
    # canonical indices and classes agree with the oracle's own enumeration
    for i, g in c4[::25] + c3[::17]:
        og = po.graph_get(g[0], i)
        assert og.key() == (g[0], g[1], g[2]) and po.graph_class(og) == w.graph_class(g)


WORKER = r"""
import os, sys, torch, torch.distributed as dist
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
first = rank * (1 << 44)                       # bench.py: disjoint sample-index ranges per rank
t = torch.tensor([float(first), 10.0 + rank], dtype=torch.float64)
gathered = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
dist.all_gather(gathered, t)
firsts = [int(g[0].item()) for g in gathered]
assert len(set(firsts)) == world and all(abs(a - b) >= (1 << 44) for a in firsts for b in firsts if a != b)
ms = torch.tensor([10.0 + rank], dtype=torch.float64)
dist.all_reduce(ms, op=dist.ReduceOp.MAX)      # bench.py: time = max over ranks
assert ms.item() == 10.0 + world - 1
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_two_rank_sharding_logic_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = 29500 + (os.getpid() % 2000)
    res = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                          "--master-port", str(port), str(script)], capture_output=True, text=True, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    assert res.stdout.count("ok") == 2
