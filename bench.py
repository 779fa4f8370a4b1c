#!/usr/bin/env python
"""bench.py — throughput of the Monte Carlo hot path on BASELINE.json configs[4] (5-loop graphs).

Contract (driver): python bench.py --gpus N --steps K --warmup W [--impl reference]; under torchrun for N>1.
A "step" is one pass of the whole hot path (sampler, scalars, integrand with all subtraction terms, weight,
reduction, double-double re-evaluation of flagged points) over one batch of --batch sample points for EVERY
diagram of the workload. The workload is the 256 seeded 5-loop graphs of configs[4] (A12); the
path shards trivially (independent sample-index ranges), so N GPUs run N replicas on disjoint ranges with no
data-path collective: scaling is "weak".
"""
import argparse
import json
import math
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "5-loop integrand samples/s on 1 B200; % of FP64 peak; sigma^2*time"
UNIT = "samples/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (4 = the metric's workload)")
    ap.add_argument("--graphs", type=int, default=0, help="use only the first G graphs of the config (0 = all; for debugging)")
    ap.add_argument("--batch", type=int, default=37888, help="sample points per diagram per step")
    ap.add_argument("--ref-points", type=int, default=384, help="oracle sample points per graph and step, at most (reference arm / cpu_baseline)")
    ap.add_argument("--ref-seconds", type=float, default=150.0, help="reference arm: oracle work of the whole --steps/--warmup run, seconds (the points per step are cut to fit)")
    ap.add_argument("--cpu-seconds", type=float, default=25.0, help="cpu_baseline leg of the default run: oracle work of its one timed step, seconds")
    ap.add_argument("--ref-graphs", type=int, default=3, help="graphs of the workload the oracle is timed on, spread over the set")
    ap.add_argument("--no-second-policy", action="store_true", help="skip the timed step under the purely relative precision policy (w_abs_tol = 0)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--deg-floor", type=float, default=None, help="Deg floor of Eq.(1) (default: the library's, 1.0)")
    ap.add_argument("--mix", type=float, nargs=3, default=None, metavar=("ALPHA", "FLOOR2", "FLOOR_IR2"), help="defensive mixture of two Eq.(1) densities (DESIGN.md S5b; default: off)")
    ap.add_argument("--deg-floor-ir", type=float, default=None, help="Deg on the soft-photon sets (default: the library's, 0.5)")
    return ap.parse_args()


class ClockSampler:
    """samples nvidia-smi clocks and throttle reasons during the timed region: ONE looping nvidia-smi process (-lms 200, the
    profiling recipe's form), started and past its NVML set-up before the timed region begins and killed after it, so that
    no process start and no driver attach falls into the timed steps"""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.index, self.rows, self.proc, self.log = index, [], None, None

    def start(self):
        import tempfile
        try:
            self.log = tempfile.NamedTemporaryFile(prefix="mcqed_clocks_", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=self.log, stderr=subprocess.DEVNULL)
            t0 = time.perf_counter()
            while os.path.getsize(self.log.name) == 0 and time.perf_counter() - t0 < 5.0 and self.proc.poll() is None:
                time.sleep(0.05)                 # first row written = set-up done
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        if self.log is not None:
            self.log.close()
            with open(self.log.name) as fh:
                self.rows = [[x.strip() for x in ln.split(",")] for ln in fh if ln.count(",") >= 5]
            os.unlink(self.log.name)
        if len(self.rows) > 2:
            self.rows = self.rows[1:]            # the row written before the timed region began

    def summary(self):
        sm = sorted(int(r[0]) for r in self.rows if r[0].isdigit())
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mx = max((int(r[1]) for r in self.rows if r[1].isdigit()), default=0)
        return {"sm_mhz": sm[len(sm) // 2] if sm else 0, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def oracle_run(args, graphs, seed, steps, warmup, budget_s):
    """times the CPU oracle as it stands on a bounded sample of the workload: --ref-graphs graphs spread evenly over the set
    (the set is sorted by canonical index = by external-vertex position, so the sample spans the gauge classes), the same n
    points per graph and step for every graph. n is --ref-points, cut down so that the timed steps and the warm-up steps
    together take about budget_s seconds: the first warm-up pass of every graph (32 points) is timed for that estimate."""
    from oracle import pyoracle as po
    from paper_1905_08007_b200 import workloads
    G = len(graphs)
    pick = sorted(set(int(round(k * (G - 1) / max(1, args.ref_graphs - 1))) for k in range(args.ref_graphs))) if args.ref_graphs > 1 else [0]
    n0 = min(32, args.ref_points)
    prep = 0.0
    ds, spp, classes = [], 0.0, []
    for gi in pick:
        idx, g = graphs[gi]
        t0 = time.perf_counter()
        d = po.Diagram(po.OracleGraph.make(g[0], g[1], g[2]))
        prep += time.perf_counter() - t0
        t0 = time.perf_counter()
        d.integrate(0, n0, seed, 2)                       # warm-up pass 1 = the pilot
        spp += (time.perf_counter() - t0) / n0
        ds.append(d)
        classes.append("%d,%d,%d" % workloads.graph_class(g))
    passes = steps + max(0, warmup - 1)
    n = int(max(16, min(args.ref_points, budget_s / (passes * spp))))
    dt = var = 0.0
    for d in ds:
        for w in range(max(0, warmup - 1)):
            d.integrate(n0 + w * n, n, seed, 2)
        t0 = time.perf_counter()
        s1 = s2 = 0.0
        for k in range(steps):
            a, b, _ = d.integrate(n0 + (max(0, warmup - 1) + k) * n, n, seed, 2)
            s1 += a
            s2 += b
        dt += time.perf_counter() - t0
        mean, err = po.estimate(s1, s2, n * steps)
        var += err * err
    del ds
    tot = n * steps * len(pick)
    return {"value": tot / dt, "seconds": dt, "cores": po.num_threads(), "prepare_s": prep, "points": tot,
            "sample": "graphs #%s of the workload (classes %s), %d points per graph and step (sized for about %.0f s of oracle work), %d timed step(s) after %d warm-up pass(es), binary64 + __float128 re-evaluation" % (
                ",".join(str(x) for x in pick), " ".join(classes), n, budget_s, steps, max(1, warmup)),
            "sigma2_time": var * dt}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1905_08007_b200 import workloads
    graphs = workloads.config_graphs(args.config)
    seed = workloads.CONFIG_SEED[args.config]
    r = oracle_run(args, graphs, seed, max(1, args.steps), args.warmup, args.ref_seconds)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * r["seconds"] / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": "configs[%d] (bounded sample)" % args.config, "sample": r["sample"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1905_08007_b200 import binding as mc
    from paper_1905_08007_b200 import build, workloads
    build.build()
    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    graphs = workloads.config_graphs(args.config)
    if args.graphs:
        graphs = graphs[:args.graphs]
    seed = workloads.CONFIG_SEED[args.config]
    G, B = len(graphs), args.batch
    # ---- prepare (not timed as throughput; reported) ----
    t0 = time.perf_counter()
    mix = {} if args.mix is None else {"mix_alpha": args.mix[0], "deg_floor2": args.mix[1], "deg_floor_ir2": args.mix[2]}
    diagrams = [mc.Diagram(g[0], g[1], g[2], deg_floor=args.deg_floor, deg_floor_ir=args.deg_floor_ir, **mix) for _, g in graphs]
    prepare_s = time.perf_counter() - t0
    infos = [d.info() for d in diagrams]
    flop = [i["flop_per_sample"] for i in infos]
    stream = torch.cuda.current_stream().cuda_stream
    batch = mc.Batch(diagrams, B)                # one persistent launch per precision tier for the whole diagram set
    sums = torch.zeros(2, G, dtype=torch.float64, device="cuda")
    cnts = torch.zeros(2, G, dtype=torch.int64, device="cuda")
    state = {"first": rank * (1 << 44), "flags": 0}        # disjoint sample-index ranges per rank (weak scaling, no collective)

    def step():
        f = state["first"]
        batch.integrate(f, B, seed, stream, sums[0], sums[1], cnts[0], cnts[1], flags=state["flags"])
        state["first"] = f + B

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()

    def timed(nsteps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(nsteps):
            step()
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    for _ in range(args.warmup):
        step()
    sums.zero_(); cnts.zero_()
    clocks = ClockSampler(local)
    clocks.start()
    l0 = mc.kernel_launch_count()
    ms = timed(args.steps)
    launches = mc.kernel_launch_count() - l0
    clocks.stop()
    n_tot = args.steps * B
    s = sums.cpu().numpy(); c = cnts.cpu().numpy()
    value = world * G * n_tot / (ms * 1e-3)
    var_sum = 0.0
    for i in range(G):
        mean = s[0, i] / n_tot
        var_sum += max(s[1, i] / n_tot - mean * mean, 0.0) / n_tot
    flagged_frac = float(c[0].sum()) / (G * n_tot)
    # per gauge-invariant class (k,m,n) of PAPER.md:104, the columns of Table 1: sum a_j, its sigma, sum |a_j|, max |a_j|
    classes = {}
    for i, (_, g) in enumerate(graphs):
        mean = s[0, i] / n_tot
        var = max(s[1, i] / n_tot - mean * mean, 0.0) / n_tot
        e = classes.setdefault("%d,%d,%d" % workloads.graph_class(g), {"n_diag": 0, "sum": 0.0, "var": 0.0, "sum_abs": 0.0, "max_abs": 0.0})
        e["n_diag"] += 1; e["sum"] += mean; e["var"] += var; e["sum_abs"] += abs(mean); e["max_abs"] = max(e["max_abs"], abs(mean))
    for e in classes.values():
        e["sigma"] = math.sqrt(e.pop("var"))
    # ---- per-kernel times: the same steps with the higher tiers switched off (flags bit 0: binary64 kernel alone;
    #      bit 1: no quad-double pass); the double-double and quad-double kernels are timed as the differences ----
    keep = (sums.clone(), cnts.clone())           # the sums of the timed region: the legs below add to them and are undone (with bit 0 set
    state["flags"] = mc.FLAG_NO_DD                # the ill-conditioned points keep their binary64 values, which must not reach the tail diagnostic)
    step()
    nk = min(args.steps, 5)                      # the per-kernel legs time at most 5 steps and are scaled to args.steps
    sc = args.steps / nk
    ms_f64 = timed(nk) * sc
    state["flags"] = mc.FLAG_NO_QD
    step()
    cnts.zero_()
    ms_noqd = timed(nk) * sc
    n_qd = float(cnts[1].sum().item()) * sc           # with the quad-double pass skipped its points are counted as dropped
    sums.copy_(keep[0]); cnts.copy_(keep[1])
    state["flags"] = 0
    ms_dd = max(ms_noqd - ms_f64, 0.0)
    ms_qd = max(ms - ms_noqd, 0.0)
    peak_flops, _ = mc.fp64_peak(4096)
    flops_f64 = sum(flop) * n_tot                                    # every point goes through the binary64 kernel
    flops_dd = float(sum(fl * cc for fl, cc in zip(flop, c[0])))     # flagged points are re-evaluated (same algorithmic flop)
    ach_f64 = flops_f64 / (ms_f64 * 1e-3) if ms_f64 > 0 else 0.0
    ach_dd = flops_dd / (ms_dd * 1e-3) if ms_dd > 0 else 0.0
    dom = "k_batch_dd" if ms_dd > ms_f64 else "k_batch_f64"
    # DRAM traffic of the dominant kernel: not measurable without a profiler, so it is read from the ncu capture of this launch
    # configuration that profiles/r2_traffic.json records (written by hand from `ncu --set full`, command in profiles/r2_summary.md);
    # null when the run is another configuration or the file has no entry for the kernel
    traffic, traffic_note = None, "no ncu capture of this configuration under profiles/"
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.json")) as fh:
            tj = json.load(fh)
        ent = tj.get(dom)
        if ent and ent["graphs"] == G and ent["batch"] == B and ent["config"] == args.config:
            traffic, traffic_note = ent["dram_bytes_per_launch"], "from profile, not live: " + ent["source"]
    except (OSError, ValueError, KeyError):
        pass
    ach = ach_dd if dom == "k_batch_dd" else ach_f64
    roofline = {"bound": "alu", "kernel": dom, "achieved": ach / 1e12, "peak": peak_flops / 1e12, "unit": "TFLOP/s", "frac": ach / peak_flops,
                "traffic": traffic, "traffic_note": traffic_note,
                "peak_source": "FP64 FMA peak measured live by mc_fp64_peak (MEASURED_PEAKS.json has no FP64 entry)",
                "kernels": {"k_batch_f64": {"ms_per_step": ms_f64 / args.steps, "achieved_tflops": ach_f64 / 1e12, "frac": ach_f64 / peak_flops, "points_per_step": G * B},
                            "k_batch_dd": {"ms_per_step": ms_dd / args.steps, "achieved_tflops": ach_dd / 1e12, "frac": ach_dd / peak_flops,
                                           "points_per_step": float(c[0].sum()) / args.steps,
                                           "note": "double-double: one algorithmic flop costs 5-6 binary64 instructions (pair arithmetic), so frac is bounded by ~0.18"},
                            "k_batch_qd": {"ms_per_step": ms_qd / args.steps, "points_per_step": n_qd / args.steps}}}
    # ---- is the variance estimate itself trustworthy? sigma*sqrt(N) of the sum must not depend on N; a few more steps outside
    #      the timed region, with a snapshot after each (heavy-tailed weights show up as a growing sigma*sqrt(N)) ----
    keep2 = (sums.clone(), cnts.clone())
    trace = []
    for k in range(min(4, max(2, args.steps))):
        step()
        torch.cuda.synchronize()
        nn = n_tot + (k + 1) * B
        sk = sums.cpu().numpy()
        mk = sk[0] / nn
        trace.append(float(math.sqrt(float((np.maximum(sk[1] / nn - mk * mk, 0.0) / nn).sum()) * nn)))
    first_s = math.sqrt(var_sum * n_tot)
    tail = {"sigma_sqrtN_after_timed_steps": first_s, "sigma_sqrtN_with_more_steps": trace,
            "variance_unreliable": bool(max(trace + [first_s]) > 1.25 * min(trace + [first_s])),
            "note": "sigma*sqrt(N per graph) of the sum of estimates; it is constant in N when the variance estimate has converged"}
    sums.copy_(keep2[0]); cnts.copy_(keep2[1])
    # ---- the same step under the purely relative precision policy (w_abs_tol = 0: north_star's literal reading, a point is
    #      accepted in binary64 only if its relative round-off bound holds), one warm-up + one timed step ----
    second = None
    if not args.no_second_policy:
        for d in diagrams:
            d.set_precision(w_abs_tol=0.0)
        batch_rel = mc.Batch(diagrams, B)
        for d in diagrams:
            d.set_precision()                      # back to the defaults (the first batch copied its values at creation)
        s_rel = torch.zeros(2, G, dtype=torch.float64, device="cuda")
        c_rel = torch.zeros(2, G, dtype=torch.int64, device="cuda")
        f0 = state["first"]
        batch_rel.integrate(f0, B, seed, stream, s_rel[0], s_rel[1], c_rel[0], c_rel[1])
        s_rel.zero_(); c_rel.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier(); e0.record()
        batch_rel.integrate(f0 + B, B, seed, stream, s_rel[0], s_rel[1], c_rel[0], c_rel[1])
        e1.record(); barrier()
        ms_rel = e0.elapsed_time(e1)
        # the default policy on the same sample range, for a like-for-like difference of the sums
        s_def = torch.zeros(2, G, dtype=torch.float64, device="cuda")
        c_def = torch.zeros(2, G, dtype=torch.int64, device="cuda")
        batch.integrate(f0 + B, B, seed, stream, s_def[0], s_def[1], c_def[0], c_def[1])
        barrier()
        second = {"policy": "relative only (w_abs_tol = 0)", "value": world * G * B / (ms_rel * 1e-3), "unit": UNIT, "ms_per_step": ms_rel, "steps": 1,
                  "flagged_fraction": float(c_rel[0].sum().item()) / (G * B), "flagged_fraction_default_same_range": float(c_def[0].sum().item()) / (G * B),
                  "max_abs_difference_of_estimates": float(((s_rel[0] - s_def[0]).abs() / B).max().item()),
                  "sum_of_estimates": float((s_rel[0] / B).sum().item()), "sum_of_estimates_default_same_range": float((s_def[0] / B).sum().item())}
        del batch_rel
    # ---- end to end through the public host-pointer API (mc_batch_integrate_host: results copied back every call) ----
    barrier()
    t0 = time.perf_counter()
    f = state["first"]
    for _ in range(args.steps):
        batch.integrate_host(f, B, seed, stream)
        f += B
    barrier()
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e = {"value": world * G * n_tot / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 32 * G,
           "note": "inputs are (first_sample, n, seed) scalars: no host->device tensor; 4 results (32 B) per diagram come back per step"}
    # precision-policy mix on a sample (mc_eval_points flag_out: 0 accepted by the relative bound, 1 re-evaluated in
    # double-double, 2 precision loss detected but accepted by the absolute bound on the weight; O8)
    mix = [0, 0, 0]
    ns = 4096
    for d in diagrams[::max(1, G // 8)][:8]:
        fl = torch.zeros(ns, dtype=torch.uint8, device="cuda")
        d.eval_points(state["first"], ns, seed, stream, flag=fl)
        torch.cuda.synchronize()
        cts = torch.bincount(fl.long(), minlength=3).cpu().numpy()
        mix = [mix[i] + int(cts[i]) for i in range(3)]
    mixn = float(sum(mix))
    precision = {"cond_max": 2.8e4, "amin_min": 1e-2, "w_abs_tol": 1e-10, "dd_cond_max": 1e26,
                 "sample_mix": {"accepted_relative": mix[0] / mixn, "reevaluated_dd": mix[1] / mixn, "accepted_absolute": mix[2] / mixn, "points": int(mixn)}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[%d]: %d seeded 5-loop graphs without lepton loops, %d points per graph per step" % (args.config, G, B) if args.config == 4
                       else "configs[%d]: %d graphs, %d points per graph per step" % (args.config, G, B),
                       "n_graphs": G, "batch": B, "seed": seed, "second_policy": second,
                       "headline_policy": "relative OR absolute acceptance (w_abs_tol = 1e-10 on the weight f/p; DESIGN.md section 6)", "l2": "tables of 256 diagrams (%.0f MB) exceed the 126 MB L2; no per-sample input is read" % (sum(i["table_bytes"] for i in infos) / 1e6),
                       "prepare_s": prepare_s, "flagged_fraction": flagged_frac, "precision": precision, "dropped": int(c[1].sum()),
                       "sigma2_time_s": var_sum * ms * 1e-3, "sum_of_estimates": float((s[0] / n_tot).sum()), "sigma": math.sqrt(var_sum), "tail": tail,
                       "algorithmic_flop_per_sample_mean": sum(flop) / G, "classes": classes},
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        r = oracle_run(args, graphs, seed, 1, 1, args.cpu_seconds)
        line["cpu_baseline"] = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"],
                                "prepare_s": r["prepare_s"], "sigma2_time_s": r["sigma2_time"]}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse()
    sys.exit(run_reference(a) if a.impl == "reference" else run_ours(a))
