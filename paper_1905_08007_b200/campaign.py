"""Table-1-style run over ALL graphs of a loop order with two-pass sample allocation.

The paper's deliverable is the sum over all 3213 mirror-identified 5-loop graphs without lepton loops, split
over the nine gauge-invariant classes (k,m,n) of Table 1 (columns: value, N_diag, sum |a_j|, max |a_j|). This script does
that run with the library: one representative of every mirror pair (PAPER.md:153 fn5; its estimate counts twice, a
mirror-symmetric graph once), a pilot pass of --pilot samples per graph, the allocation n_j ~ sigma_j / sqrt(cost_j) of the
remaining budget (mc_allocate_samples; the paper does not disclose its own allocation), the main pass, and the class table.
Graphs are prepared, integrated and released in chunks so that the tables of a chunk fit the device (6354 five-loop
graphs hold ~57 GB of tables). All arithmetic of the method runs in the CUDA kernels; this file only schedules calls.

    python -m paper_1905_08007_b200.campaign --loops 5 --pilot 4096 --mean-samples 16384 --chunk 384 --out profiles/r2_campaign_L5

The statistics are LOW by design (the paper used 1.9e14 samples): the table shows the bookkeeping (N_diag must
equal Table 1 after mirror identification) and the allocation gain, not a physics result.
"""
import argparse
import json
import math
import sys
import time

import numpy as np


def mirror(graph):
    L, e, chords = graph
    return (L, 2 * L - e, tuple(sorted((2 * L - b, 2 * L - a) for a, b in chords)))


def representatives(graphs):
    """one graph per mirror pair (the one that comes first in canonical order) with its multiplicity 1 or 2"""
    index = {g: i for i, g in enumerate(graphs)}
    out = []
    for i, g in enumerate(graphs):
        j = index[mirror(g)]
        if j >= i:
            out.append((i, g, 1 if j == i else 2))
    return out


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--loops", type=int, default=5)
    ap.add_argument("--pilot", type=int, default=4096, help="samples per graph in the pilot pass")
    ap.add_argument("--mean-samples", type=int, default=16384, help="mean samples per graph in the main pass (budget = this x cost)")
    ap.add_argument("--chunk", type=int, default=384, help="graphs prepared and integrated together")
    ap.add_argument("--max-graphs", type=int, default=0, help="only the first N representatives (0 = all; for a quick look)")
    ap.add_argument("--cap", type=int, default=0, help="samples per graph and pass held by the batch scratch (0 = max(pilot, 4 x mean-samples); longer ranges take several passes)")
    ap.add_argument("--stride", type=int, default=1, help="every K-th representative only (a sample spread over the whole set)")
    ap.add_argument("--seed", type=int, default=5)
    ap.add_argument("--deg-floor", type=float, default=None, help="Deg floor of the UV-type sets (DESIGN.md S5; default: the library's)")
    ap.add_argument("--deg-floor-ir", type=float, default=None, help="Deg of the soft-photon sets (default: the library's)")
    ap.add_argument("--mix", type=float, nargs=3, default=None, metavar=("ALPHA", "FLOOR2", "FLOOR_IR2"), help="defensive mixture: probability and Deg floors of the second channel (DESIGN.md S5b)")
    ap.add_argument("--mrg32k3a", action="store_true", help="second random stream (mc_options.flags bit 2)")
    ap.add_argument("--out", default="")
    a = ap.parse_args(argv)
    import torch
    from . import binding as mc
    from . import workloads
    assert torch.cuda.is_available(), "campaign needs a CUDA device (no CPU fallback)"
    st = torch.cuda.current_stream().cuda_stream
    graphs = workloads.all_graphs(a.loops)
    reps = representatives(graphs)[::max(1, a.stride)]
    if a.max_graphs:
        reps = reps[:a.max_graphs]
    G = len(reps)
    mean, err, n_used, cost, flagged = np.zeros(G), np.zeros(G), np.zeros(G), np.zeros(G), np.zeros(G)
    sig1 = np.zeros(G)
    t_prep = t_run = 0.0
    cap = a.cap if a.cap > 0 else max(a.pilot, 4 * a.mean_samples)
    # per chunk: prepare once, pilot pass, allocation of the chunk's share of the budget (mean_samples x the chunk's cost: the
    # split between chunks stays equal-cost so that every chunk is prepared only once; inside a chunk of a few hundred graphs
    # the per-sample sigmas already span orders of magnitude), main pass on the sample indices after the pilot's
    chunks = [list(range(c, min(G, c + a.chunk))) for c in range(0, G, a.chunk)]
    n_main = np.zeros(G, np.int64)
    for ids in chunks:
        t0 = time.perf_counter()
        ds = [mc.Diagram(*reps[i][1], deg_floor=a.deg_floor, deg_floor_ir=a.deg_floor_ir, flags=mc.FLAG_MRG32K3A if a.mrg32k3a else 0,
                         **({} if a.mix is None else {"mix_alpha": a.mix[0], "deg_floor2": a.mix[1], "deg_floor_ir2": a.mix[2]})) for i in ids]
        t_prep += time.perf_counter() - t0
        for k, i in enumerate(ids):
            cost[i] = ds[k].info()["flop_per_sample"]
        b = mc.Batch(ds, cap)
        S = torch.zeros(2, len(ids), dtype=torch.float64, device="cuda")
        C = torch.zeros(2, len(ids), dtype=torch.int64, device="cuda")
        torch.cuda.synchronize(); t0 = time.perf_counter()
        b.integrate(0, a.pilot, a.seed, st, S[0], S[1], C[0], C[1])
        torch.cuda.synchronize(); t_run += time.perf_counter() - t0
        s = S.cpu().numpy()
        m1 = s[0] / a.pilot
        sig1[ids] = np.sqrt(np.maximum(s[1] / a.pilot - m1 * m1, 0.0))
        budget = float(a.mean_samples) * cost[ids].sum()
        nm = mc.allocate_samples(np.maximum(sig1[ids], 1e-300), cost[ids], budget, n_min=0).astype(np.int64)
        n_main[ids] = np.minimum(nm, 64 * a.mean_samples)        # a pilot sigma is noisy: bound the share of one graph
        torch.cuda.synchronize(); t0 = time.perf_counter()
        b.integrate_counts([a.pilot] * len(ids), n_main[ids], a.seed, st, S[0], S[1], C[0], C[1])
        torch.cuda.synchronize(); t_run += time.perf_counter() - t0
        s, c = S.cpu().numpy(), C.cpu().numpy()
        n = a.pilot + n_main[ids]
        mean[ids] = s[0] / n
        err[ids] = np.sqrt(np.maximum(s[1] / n - (s[0] / n) ** 2, 0.0) / n)
        n_used[ids] = n; flagged[ids] = c[0]
        del b, ds
    # ---- Table 1 columns per class ----
    mult = np.array([r[2] for r in reps], float)
    classes = {}
    for i, (_, g, m) in enumerate(reps):
        e = classes.setdefault(workloads.graph_class(g), {"n_diag": 0, "value": 0.0, "var": 0.0, "sum_abs": 0.0, "max_abs": 0.0, "samples": 0})
        e["n_diag"] += 1; e["value"] += m * mean[i]; e["var"] += (m * err[i]) ** 2
        e["sum_abs"] += abs(m * mean[i]); e["max_abs"] = max(e["max_abs"], abs(m * mean[i])); e["samples"] += int(n_used[i])
    total, tvar = float((mult * mean).sum()), float(((mult * err) ** 2).sum())
    # what the same budget would have given with an equal split (from the measured per-sample sigmas of the whole run)
    sig_ps = err * np.sqrt(n_used)
    n_eq = (a.pilot + a.mean_samples) * np.ones(G) * cost.mean() / cost          # equal COST per graph
    var_equal = float(((mult * sig_ps) ** 2 / np.maximum(n_eq, 1)).sum())
    res = {"mix": a.mix, "deg_floor": a.deg_floor, "deg_floor_ir": a.deg_floor_ir, "generator": "mrg32k3a" if a.mrg32k3a else "philox4x32_10", "loops": a.loops, "n_graphs_all": len(graphs), "n_mirror_identified": G, "pilot": a.pilot, "mean_samples": a.mean_samples, "seed": a.seed,
           "samples_total": int(n_used.sum()), "prepare_s": t_prep, "run_s": t_run, "samples_per_s": float(n_used.sum()) / t_run,
           "total": total, "sigma": math.sqrt(tvar), "sigma2_time_s": tvar * t_run, "sigma_equal_cost_split_same_budget": math.sqrt(var_equal),
           "variance_gain_of_allocation": var_equal / tvar if tvar > 0 else None, "flagged_fraction": float(flagged.sum() / n_used.sum()),
           "classes": {"%d,%d,%d" % k: {**v, "sigma": math.sqrt(v.pop("var"))} for k, v in sorted(classes.items())}}
    lines = ["| class (k,m,n) | value | sigma | N_diag | sum abs a_j | max abs a_j | samples |", "|---|---|---|---|---|---|---|"]
    for k, v in res["classes"].items():
        lines.append("| (%s) | %+.3f | %.3f | %d | %.2f | %.2f | %d |" % (k, v["value"], v["sigma"], v["n_diag"], v["sum_abs"], v["max_abs"], v["samples"]))
    lines.append("| all | %+.3f | %.3f | %d | | | %d |" % (total, res["sigma"], G, res["samples_total"]))
    print("\n".join(lines))
    print(json.dumps({k: v for k, v in res.items() if k != "classes"}))
    if a.out:
        with open(a.out + ".json", "w") as fh:
            json.dump(res, fh, indent=1)
        with open(a.out + ".md", "w") as fh:
            fh.write("# Table-1-style run, %d loops, %d mirror-identified graphs (command: python -m paper_1905_08007_b200.campaign %s)\n\n" % (a.loops, G, " ".join(sys.argv[1:])))
            fh.write("\n".join(lines) + "\n\n" + json.dumps({k: v for k, v in res.items() if k != "classes"}, indent=1) + "\n")
    return res


if __name__ == "__main__":
    main()
