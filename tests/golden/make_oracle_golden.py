"""tests/golden/make_oracle_golden.py — writes the stored oracle results under tests/golden/.

Calls ONLY oracle/ (never the CUDA path).  Usage:  python tests/golden/make_oracle_golden.py two_loop|three_loop [n_per_graph]
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
from oracle import pyoracle as po  # noqa: E402


def _mc_all(L, n, seed, deg_floor, path, head, mode=2):
    """Monte Carlo of ALL graphs of loop order L with the oracle alone. mode 2: binary64 value unless the truth flag
    |f64 - fwide| > 1e-10 |fwide| is set, then the binary128 value (O8); mode 0: binary64 values. Sums kept exactly (hex)"""
    lines = head + ["# e chords k m n n_points mean sigma S1(hex) S2(hex) n_truth_flagged"]
    for g in po.all_graphs(L):
        d = po.Diagram(g, deg_floor=deg_floor)
        s1, s2, nf = d.integrate(0, n, seed, mode)
        m, e = po.estimate(s1, s2, n)
        k = po.graph_class(g)
        lines.append("%d %s %d %d %d %d %.9f %.9f %s %s %d" % (g.ext_pos, "".join("%d%d" % c for c in g.chords()), k[0], k[1], k[2], n, m, e, float(s1).hex(), float(s2).hex(), nf))
        print(lines[-1], flush=True)
        with open(path + ".partial", "w") as fh:           # rewritten after every graph: a long run can be watched
            fh.write("\n".join(lines) + "\n")
    os.replace(path + ".partial", path)


def two_loop(n):
    _mc_all(2, n, 2, 0.5, os.path.join(HERE, "oracle_two_loop_mc.txt"),
            ["# Oracle Monte Carlo of the six 2-loop graphs (BASELINE.json configs[1]), seed 2, first_sample 0, %d points per graph," % n,
             "# Deg floor 0.5, no cap, oracle mode 2 (binary128 value where binary64 loses more than 1e-10).  Written by make_oracle_golden.py (oracle only).",
             "# The sum of the six means is pinned by north_star: -0.344166."])


def three_loop(n):
    _mc_all(3, n, 3, 0.75, os.path.join(HERE, "oracle_three_loop_mc.txt"),
            ["# Oracle Monte Carlo of all 50 3-loop graphs (BASELINE.json configs[2]), seed 3, first_sample 0, %d points per graph," % n,
             "# Deg floor 0.75 on all clamped sets, no cap, oracle mode 0 (binary64 values: on graphs 0, 20, 45 the binary128 re-evaluation of mode 2",
             "# moves the mean by 1e-13, far below the statistical error, and costs 8x the time).  Written by make_oracle_golden.py (oracle only).",
             "# Soft pin: the literature value of the 3-loop contribution of graphs without lepton loops, 0.904979 (SURVEY.md P9; not in PAPER.md)."], mode=0)


def high_loop(L, indices, n, seed, first):
    """per-point oracle values at L=4,5 (the oracle's table build takes minutes per graph at L=5):
    sample index range, seed and, per point, the binary128 value rounded to binary64 (hex) and the binary64 value"""
    lines = ["# Oracle per-point integrand values, loop order %d, points first_sample=%d..+%d of seed %d, default Deg (floor 1.0, 0.5 on the soft-photon sets: DESIGN.md S5)." % (L, first, n, seed),
             "# Written by make_oracle_golden.py (oracle only). Values of L>=4 graphs are 'parity unpinned' by the paper (DESIGN.md section 3).",
             "# graph_index point fwide(hex) f64(hex)"]
    for idx in indices:
        d = po.Diagram(po.graph_get(L, idx))
        z, p, _ = d.sample(first, n, seed)
        r = d.eval_z(z, wide=True)
        for k in range(n):
            lines.append("%d %d %s %s" % (idx, k, float(r["fwide"][k]).hex(), float(r["f64"][k]).hex()))
        print("graph", idx, "done", flush=True)
        del d
        with open(os.path.join(HERE, "oracle_points_L%d.txt.partial" % L), "w") as fh:
            fh.write("\n".join(lines) + "\n")
    os.replace(os.path.join(HERE, "oracle_points_L%d.txt.partial" % L), os.path.join(HERE, "oracle_points_L%d.txt" % L))


# 33 graphs of BASELINE.json configs[4] (canonical indices): the first graph of each of the nine classes of Table 1, the graph with
# the most formula terms (2821: 40 terms), the graphs with the most self-energy subgraphs (691, 705, 6351: four each), the rest
# spread evenly over the set; plus the three graphs of the round-1 file
L5_GRAPHS = [3, 49, 453, 691, 692, 705, 709, 1029, 1408, 1443, 1529, 1954, 2110, 2145, 2302, 2324, 2718, 2806, 2821, 2825, 2877, 3120,
             3304, 3625, 4026, 4651, 4984, 5454, 5512, 5660, 5957, 6290, 6351]

if __name__ == "__main__":
    if sys.argv[1] == "high_loop":
        high_loop(int(sys.argv[2]), L5_GRAPHS if sys.argv[3] == "default" else [int(x) for x in sys.argv[3].split(",")], int(sys.argv[4]), 5, 1000)
    if sys.argv[1] == "two_loop":
        two_loop(int(float(sys.argv[2])) if len(sys.argv) > 2 else 20000000)
    if sys.argv[1] == "three_loop":
        three_loop(int(float(sys.argv[2])) if len(sys.argv) > 2 else 4000000)
