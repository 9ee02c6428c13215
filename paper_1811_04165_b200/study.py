"""The paper's GA experiments on this GPU: sweeps of the GA settings at a fixed evaluation budget,
the convergence statistic c_v, and the GA-versus-random histogram of best fitness values.

    python -m paper_1811_04165_b200.study [--budget 250] [--seeds 5] [--runs 30] [--out gpurun_out/study.json]

What follows the paper (PAPER.md, cited P:n):
  * baseline settings N_pop = 20, tournament pool = 20 % of N_pop, p_cross = 0.8, p_mut = 0.1 per kernel, offspring
    replace parents by "best half of each group";
  * one quantity varied at a time: mutation rate, crossover rate, population size, crossover operator (single
    point / coin toss), and pure random search (Fig. 3 a-d); every run gets the same budget of fitness
    evaluations (the paper gives every run the same wall time);
  * c_v = sigma / mu of every gene over the configurations a run ends with, averaged over the runs, GA against
    random search (Fig. 4);
  * histogram of the best fitness of >= 30 GA and >= 30 random runs (Fig. 5).
The paper's figures are images, so there is no curve to match: the numbers below are this GPU's, for these kernels.
The workload is a scaled-down subband plan (seconds per run); fitness = the library's CUDA-event harness.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import time
from typing import Dict, List, Sequence

GENES = ("threads_t", "threads_dm", "samples_per_thread", "dms_per_thread", "unroll", "staging", "vec_bytes")


def gene_cv(final_configs: Sequence[Sequence[Sequence[int]]], slots: Sequence[int]) -> Dict[str, Dict[str, float]]:
    """c_v = sigma / mu (population standard deviation over the mean) of every gene over a set of end
    configurations.  final_configs[i][s] = the 7 genes of pipeline slot s of configuration i.  Returns
    {slot: {gene: c_v}}; a gene whose mean is 0 (only `staging` can be: all "direct") has c_v 0 when it does not
    vary and inf otherwise (the paper leaves its binary localMem out for that reason)."""
    out: Dict[str, Dict[str, float]] = {}
    n = len(final_configs)
    for s in slots:
        row = {}
        for g, name in enumerate(GENES):
            vals = [float(c[s][g]) for c in final_configs]
            mu = sum(vals) / n
            var = sum((v - mu) ** 2 for v in vals) / n
            sd = math.sqrt(var)
            row[name] = (sd / mu) if mu > 0 else (0.0 if sd == 0 else float("inf"))
        out[str(s)] = row
    return out


def mean_cv(per_run: Sequence[Dict[str, Dict[str, float]]]) -> Dict[str, Dict[str, float]]:
    """Average of gene_cv results over runs ("We then average c_v over multiple algorithm runs"); infinite
    entries are left out of a gene's average."""
    acc: Dict[str, Dict[str, List[float]]] = {}
    for r in per_run:
        for s, row in r.items():
            for g, v in row.items():
                if math.isfinite(v):
                    acc.setdefault(s, {}).setdefault(g, []).append(v)
    return {s: {g: sum(v) / len(v) for g, v in row.items()} for s, row in acc.items()}


def histogram(values: Sequence[float], lo: float, hi: float, nbins: int) -> List[int]:
    """Counts of values in nbins equal bins over [lo, hi]; values outside are clamped into the end bins."""
    h = [0] * nbins
    for v in values:
        b = int((v - lo) / (hi - lo) * nbins) if hi > lo else 0
        h[min(max(b, 0), nbins - 1)] += 1
    return h


def curve_at(history: Sequence[float], marks: Sequence[int]) -> List[float]:
    """Best-so-far fitness after the given numbers of evaluations (the last value if the run was shorter)."""
    return [history[min(m, len(history)) - 1] if history else float("inf") for m in marks]


def small_config():
    """A scaled-down subband plan (the structure of BASELINE.json configs[2]) on which one tuning run takes seconds."""
    from synth import configs
    from synth.configs import SubbandPlan
    return configs.scaled(configs.apertif_direct(), name="study_subband", nchan=256, nsamp_out=8192, ndm=64,
                          widths=(1, 2, 4, 8, 16, 32, 64), n_pulses=2,
                          subband=SubbandPlan(n_subbands=8, n_coarse=8, coarse_first=0.0, coarse_step=8.0, n_fine=8,
                                              fine_step=0.25))


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--budget", type=int, default=250, help="fitness evaluations per run")
    ap.add_argument("--seeds", type=int, default=5, help="runs per sweep setting")
    ap.add_argument("--runs", type=int, default=30, help="GA and random runs of the c_v / histogram study")
    ap.add_argument("--out", default="gpurun_out/study.json")
    ap.add_argument("--parts", nargs="+", default=["sweeps", "cv"], choices=["sweeps", "cv"])
    args = ap.parse_args(argv)

    import torch
    import paper_1811_04165_b200 as ddp
    from synth import filterbank

    if not torch.cuda.is_available():
        raise SystemExit("study: no CUDA device -- the tuners' hardware harness has no CPU fallback")
    cfg = small_config()
    plan = ddp.plan_from_config(cfg)
    info = plan.query()
    buf = ddp.alloc_buffers(plan, "cuda:0")
    X, _ = filterbank.make_filterbank(cfg, int(info.nsamp_in_required), int(info.in_stride_min))
    buf["d_in"].copy_(torch.from_numpy(X))
    torch.cuda.synchronize()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda:0")
    io = ddp.make_tune_io(buf["d_in"], buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"], d_flush=flush,
                          reps=5, warmup=1, cutoff_factor=3.0)
    slots = [0, 1, 2, 3]
    kern = (ddp.K_SUB1, ddp.K_SUB2, ddp.K_INTEGRATE, ddp.K_SNR)
    defaults = [plan.get_kcfg(k) for k in kern]
    marks = [m for m in (20, 50, 100, 150, 200, 250, 400, 600, 1000) if m <= args.budget] or [args.budget]
    report = {"workload": cfg.name, "gpu": torch.cuda.get_device_name(0), "budget_evaluations": args.budget,
              "curve_marks": marks, "space": {ddp.KERNEL_NAMES[k]: len(plan.enumerate_kcfgs(k)) for k in kern},
              "baseline": {"population": 20, "tournament": 4, "p_cross": 0.8, "p_mut": 0.1, "mutation_kind": 1,
                           "crossover_kind": 0, "replacement": 1}}
    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)

    def store():
        with open(args.out + ".tmp", "w") as fh:
            json.dump(report, fh, indent=1)
        os.replace(args.out + ".tmp", args.out)

    def reset():
        for k, c in zip(kern, defaults):
            plan.set_kcfg(k, c)

    def ga(seed, **over):
        p = dict(report["baseline"])
        p.update(over)
        reset()
        return plan.tune_ga(io, seed=seed, population=p["population"], generations=1 << 20,
                            tournament=max(2, round(0.2 * p["population"])) if "tournament" not in over else p["tournament"],
                            p_cross=p["p_cross"], crossover_kind=p["crossover_kind"], p_mut=p["p_mut"],
                            mutation_kind=p["mutation_kind"], elitism=0, replacement=p["replacement"],
                            max_evals=args.budget, final_cap=p["population"])

    def rnd(seed, final_cap=20):
        reset()
        return plan.tune_random(io, seed=seed, max_evals=args.budget, final_cap=final_cap)

    ms, per = plan.time_pipeline(io, defaults)
    report["defaults_ms"] = ms
    t_start = time.time()
    if "sweeps" in args.parts:
        sweeps = {"p_mut": [("p_mut", v) for v in (0.01, 0.05, 0.1, 0.3, 1.0)],
                  "p_cross": [("p_cross", v) for v in (0.2, 0.5, 0.8, 1.0)],
                  "population": [("population", v) for v in (20, 30, 50, 64)],
                  "crossover_kind": [("crossover_kind", v) for v in (0, 1)],
                  "replacement": [("replacement", v) for v in (0, 1)]}
        report["sweeps"] = {}
        for name, settings in sweeps.items():
            for key, val in settings:
                runs = []
                for seed in range(1, args.seeds + 1):
                    over = {key: val}
                    if key == "replacement" and val == 0:
                        over["replacement"] = 0
                    r = ga(seed, **over)
                    runs.append({"seed": seed, "best_ms": r["best_ms"], "curve": curve_at(r["history"], marks),
                                 "evaluations": r["n_fitness_calls"]})
                best = sorted(x["best_ms"] for x in runs)
                report["sweeps"].setdefault(name, {})[str(val)] = {
                    "median_best_ms": best[len(best) // 2], "min_best_ms": best[0], "max_best_ms": best[-1],
                    "median_curve": [sorted(x["curve"][i] for x in runs)[len(runs) // 2] for i in range(len(marks))],
                    "runs": runs}
                store()
                print("sweep %s = %s: median best %.4f ms over %d seeds (%.0f s elapsed)" % (
                    name, val, best[len(best) // 2], len(runs), time.time() - t_start), flush=True)
        runs = []
        for seed in range(1, args.seeds + 1):
            r = rnd(seed)
            runs.append({"seed": seed, "best_ms": r["best_ms"], "curve": curve_at(r["history"], marks)})
        best = sorted(x["best_ms"] for x in runs)
        report["sweeps"]["random_search"] = {"median_best_ms": best[len(best) // 2], "min_best_ms": best[0],
                                             "max_best_ms": best[-1], "runs": runs}
        store()
    if "cv" in args.parts:
        cvs = {"ga": [], "random": []}
        bests = {"ga": [], "random": []}
        for seed in range(101, 101 + args.runs):
            for kind in ("ga", "random"):
                r = ga(seed) if kind == "ga" else rnd(seed)
                finals = [[list(c.astuple()) for c in joint] for joint, _ in r["final"]]
                if len(finals) >= 2:
                    cvs[kind].append(gene_cv(finals, slots))
                bests[kind].append(r["best_ms"])
            print("cv study: %d / %d runs (%.0f s elapsed)" % (seed - 100, args.runs, time.time() - t_start), flush=True)
            allv = bests["ga"] + bests["random"]
            lo, hi = min(allv), max(allv)
            report["cv"] = {"runs": len(bests["ga"]), "end_configurations_per_run": 20,
                            "ga": mean_cv(cvs["ga"]), "random": mean_cv(cvs["random"]),
                            "slot_names": {str(s): ddp.KERNEL_NAMES[k] for s, k in zip(slots, kern)}}
            report["histogram"] = {"lo_ms": lo, "hi_ms": hi, "bins": 12, "ga": histogram(bests["ga"], lo, hi, 12),
                                   "random": histogram(bests["random"], lo, hi, 12),
                                   "ga_best_ms": sorted(bests["ga"]), "random_best_ms": sorted(bests["random"])}
            store()
    report["wall_seconds"] = time.time() - t_start
    store()
    plan.destroy()
    return 0


if __name__ == "__main__":
    sys.exit(main())
