"""Precision scan: how many points of a diagram lose precision in binary64, and how well the run-time
indicators of the binary64 kernel (cond = a/|f| with a the running bound on the sum of |monomial|; inner = min(|A_t|, g_t,
pivot ratio)) predict it. Used to choose mc_options.cond_max / amin_min / deg_floor (DESIGN.md sections 6, 7).
profiles/r1_precision_scan.md is the output of this tool on the final code of round 1.

  python -m paper_1905_08007_b200.precision_scan [--points N] [--loops L --index I ...] > profiles/<name>.md

Everything is computed by the library's own kernels (mc_eval_points, mc_eval_z): the double-double value is the
reference for the binary64 value of the same point.
"""
import argparse

import numpy as np
import torch

from . import binding as mc
from . import workloads

DEFAULT = [(2, 0), (2, 1), (2, 3), (3, 7), (3, 29), (3, 12), (4, 100), (4, 305), (5, 1000), (5, 3333)]


def scan(L, idx, n, floor, cap, seed=7):
    g = workloads.all_graphs(L)[idx]
    d = mc.Diagram(g[0], g[1], g[2], deg_floor=floor, deg_cap=cap)
    st = torch.cuda.current_stream().cuda_stream
    z = torch.zeros(n, 3 * L, dtype=torch.float64, device="cuda")
    p = torch.zeros(n, dtype=torch.float64, device="cuda")
    d.eval_points(0, n, seed, st, z, None, p, None, None, None, None)
    f64, fdd, cond = (torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(3))
    aux = torch.zeros(n, 2, dtype=torch.float64, device="cuda")
    d.eval_z(n, z, st, f64, fdd, cond, aux)
    torch.cuda.synchronize()
    rel = ((f64 - fdd).abs() / fdd.abs()).cpu().numpy()
    c, inner = cond.cpu().numpy(), aux.cpu().numpy().min(axis=1)
    w = (fdd / p).cpu().numpy()
    w = np.where(np.isfinite(w), w, 0.0)
    row = {"graph": "L=%d #%d" % (L, idx), "floor": floor, "cap": cap, "mean": w.mean(), "err": w.std() / np.sqrt(n),
           "rel_q": [np.quantile(rel, q) for q in (0.5, 0.9, 0.99)], "P_cond": [(c > t).mean() for t in (1e4, 1e6, 1e9, 1e12)]}
    for (t, tau) in ((3e4, 1e-2), (1e4, 1e-2), (1e5, 1e-2)):
        ok = (c <= t) & (inner >= tau)
        row["flag_%g_%g" % (t, tau)] = (1 - ok.mean(), rel[ok].max() if ok.any() else 0.0)
    d.close()
    return row


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--points", type=int, default=100000)
    a = ap.parse_args()
    print("| graph | floor | cap | estimate | rel.err of f64 (50/90/99 %) | P(cond > 1e4/1e6/1e9/1e12) | not accepted by the relative bound, max accepted err @ (3e4,1e-2) | @ (1e4,1e-2) | @ (1e5,1e-2) |")
    print("|---|---|---|---|---|---|---|---|---|")
    for (L, idx) in DEFAULT:
        for (floor, cap) in ((0.5, 1e30), (0.75, 1e30), (0.75, 1.0)):
            r = scan(L, idx, a.points if L < 5 else a.points // 4, floor, cap)
            fl = ["%.2f, %.0e" % r[k] for k in ("flag_30000_0.01", "flag_10000_0.01", "flag_100000_0.01")]
            print("| %s | %g | %s | %.4f ± %.4f | %s | %s | %s | %s | %s |" % (
                r["graph"], r["floor"], "-" if r["cap"] > 1e20 else "%g" % r["cap"], r["mean"], r["err"],
                " / ".join("%.0e" % x for x in r["rel_q"]), " / ".join("%.3f" % x for x in r["P_cond"]), fl[0], fl[1], fl[2]))


if __name__ == "__main__":
    main()
