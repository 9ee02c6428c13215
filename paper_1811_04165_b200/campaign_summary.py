"""Condenses a campaign report (campaign.py) into the small committed summary that bench.py quotes.

    python -m paper_1811_04165_b200.campaign_summary gpurun_out/campaign_cfg2.json \
        paper_1811_04165_b200/campaign_b200.json

Pure bookkeeping on numbers the tuners measured on the GPU: per tuner and seed the re-timed pipeline
time of its best joint configuration (the campaign's interleaved `final` stage), the number of
fitness calls, compiles and wall seconds, and the best-so-far fitness at fixed numbers of
evaluations (P:225 / Fig. 3: best configuration time against evaluations).  BASELINE.json's target
is read off two ratios: GA time / brute-force time, and GA evaluations / brute-force evaluations.
"""
from __future__ import annotations

import json
import statistics
import sys

CHECKPOINTS = (64, 125, 250, 500, 1000, 2000, 3000)


def _curve(history):
    out = {str(n): history[n - 1] for n in CHECKPOINTS if n <= len(history)}
    out[str(len(history))] = history[-1]
    return out


def summarise(report: dict) -> dict:
    final = report.get("final", {})
    out = {"workload": report.get("workload"), "gpu": report.get("gpu"), "host_cores": report.get("host_cores"),
           "space": report.get("space"), "ga_params": report.get("ga_params"),
           "defaults_ms": final.get("defaults", {}).get("ms", report.get("defaults_ms", {}).get("total"))}
    for kind in ("ga", "random"):
        runs = {}
        for seed, rec in sorted(report.get(kind, {}).items(), key=lambda kv: int(kv[0])):
            f = final.get("%s_%s" % (kind, seed), {})
            runs[seed] = {"final_ms": f.get("ms"), "tuner_best_ms": rec["best_ms"], "per_slot_ms": f.get("per_slot"),
                          "cfg": rec["best"], "n_fitness_calls": rec["n_fitness_calls"],
                          "n_kernel_timings": rec["n_kernel_timings"], "n_compiles": rec["n_compiles"],
                          "wall_seconds": rec["wall_seconds"], "best_so_far_at": _curve(rec["history"])}
        if runs:
            fm = [r["final_ms"] for r in runs.values() if r["final_ms"] is not None]
            out[kind] = {"runs": runs,
                         "final_ms_median": statistics.median(fm) if fm else None,
                         "final_ms_min": min(fm) if fm else None, "final_ms_max": max(fm) if fm else None,
                         "n_fitness_calls_median": statistics.median(r["n_fitness_calls"] for r in runs.values()),
                         "wall_seconds_median": statistics.median(r["wall_seconds"] for r in runs.values())}
    bf = report.get("bf", {})
    if bf.get("winners"):
        out["bf"] = {"winners": bf["winners"], "final_ms": final.get("bf", {}).get("ms"),
                     "per_slot_ms": final.get("bf", {}).get("per_slot"),
                     "sum_isolated_min_ms": bf.get("sum_isolated_min_ms"),
                     "n_fitness_calls": bf.get("n_fitness_calls"),
                     "per_kernel": {k: {"n_fitness_calls": v["n_fitness_calls"], "n_compiles": v["n_compiles"],
                                        "wall_seconds": v["wall_seconds"], "kernel_min_ms": v["kernel_min_ms"]}
                                    for k, v in bf.get("per_slot", {}).items()},
                     "wall_seconds": sum(v["wall_seconds"] for v in bf.get("per_slot", {}).values())}
    if "ga" in out and out.get("bf", {}).get("final_ms") and out["ga"]["final_ms_median"]:
        b = out["bf"]
        out["ga_vs_bf"] = {"time_ratio_median": out["ga"]["final_ms_median"] / b["final_ms"],
                           "time_ratio_worst_seed": out["ga"]["final_ms_max"] / b["final_ms"],
                           "evaluation_ratio": out["ga"]["n_fitness_calls_median"] / b["n_fitness_calls"]
                           if b.get("n_fitness_calls") else None}
    if "ga" in out and "random" in out and out["random"]["final_ms_median"]:
        out["ga_vs_random_time_ratio_median"] = out["ga"]["final_ms_median"] / out["random"]["final_ms_median"]
    out["tuned"] = report.get("tuned")
    out["tuned_from"] = report.get("tuned_from")
    return out


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    if len(argv) != 2:
        raise SystemExit(__doc__)
    with open(argv[0]) as fh:
        report = json.load(fh)
    with open(argv[1], "w") as fh:
        json.dump(summarise(report), fh, indent=1)
        fh.write("\n")
    return 0


if __name__ == "__main__":
    sys.exit(main())
