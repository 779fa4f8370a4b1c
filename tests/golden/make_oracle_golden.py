"""tests/golden/make_oracle_golden.py — writes the stored oracle results under tests/golden/.

Calls ONLY oracle/ (never the CUDA path).  Usage:  python tests/golden/make_oracle_golden.py two_loop [n_per_graph]
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import pyoracle as po  # noqa: E402


def two_loop(n):
    lines = ["# Oracle Monte Carlo of the six 2-loop graphs (BASELINE.json configs[1]), binary64 integrand values,",
             "# seed 2, first_sample 0, %d points per graph, Deg floor 0.5, no cap.  Written by make_oracle_golden.py (oracle only)." % n,
             "# The sum is pinned by north_star: -0.344166.",
             "# e chords k m n n_points mean sigma"]
    for g in po.all_graphs(2):
        d = po.Diagram(g, deg_floor=0.5)
        s1, s2, _ = d.integrate(0, n, 2, 0)
        m, e = po.estimate(s1, s2, n)
        k = po.graph_class(g)
        lines.append("%d %s %d %d %d %d %.9f %.9f" % (g.ext_pos, "".join("%d%d" % c for c in g.chords()), k[0], k[1], k[2], n, m, e))
        print(lines[-1], flush=True)
    with open(os.path.join(HERE, "oracle_two_loop_mc.txt"), "w") as fh:
        fh.write("\n".join(lines) + "\n")


if __name__ == "__main__":
    if sys.argv[1] == "two_loop":
        two_loop(int(float(sys.argv[2])) if len(sys.argv) > 2 else 20000000)
