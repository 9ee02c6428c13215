"""Host-only checks of campaign_summary.summarise(): pure bookkeeping on a hand-made campaign report."""
from __future__ import annotations

import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1811_04165_b200 import campaign_summary as cs  # noqa: E402


def _run(best_ms, calls, hist):
    return {"best": [[64, 1, 4, 1, 1, 0, 4]] * 4, "best_ms": best_ms, "kernel_ms": [0, 0, 0, 0], "n_fitness_calls": calls,
            "n_kernel_timings": calls * 20, "n_compiles": 7, "wall_seconds": 10.0, "history": hist,
            "sum_isolated_min_ms": 0.0}


def _report():
    h = [2.0] * 63 + [1.5] * 37 + [1.0] * 50  # best-so-far after each of 150 evaluations
    return {
        "workload": "w", "gpu": "g", "host_cores": 4, "space": {"sub1": 10, "sub2": 20},
        "ga_params": {"population": 8}, "defaults_ms": {"total": 3.0, "per_slot": [1, 1, 0.5, 0.5]},
        "ga": {"1": _run(1.0, 150, h), "2": _run(1.2, 150, h)},
        "random": {"1": _run(1.6, 150, h), "2": _run(1.8, 150, h)},
        "bf": {"winners": {"sub1": [1] * 7}, "n_fitness_calls": 3000, "sum_isolated_min_ms": 0.9,
               "per_slot": {"sub1": {"n_fitness_calls": 3000, "n_compiles": 1, "wall_seconds": 5.0, "kernel_min_ms": 0.9}}},
        "final": {"defaults": {"ms": 3.1}, "bf": {"ms": 1.0, "per_slot": [1, 0, 0, 0]},
                  "ga_1": {"ms": 1.04, "per_slot": []}, "ga_2": {"ms": 1.30, "per_slot": []},
                  "random_1": {"ms": 1.5, "per_slot": []}, "random_2": {"ms": 2.0, "per_slot": []}},
        "tuned": {"sub1": [1] * 7}, "tuned_from": "bf",
    }


def test_ratios_and_checkpoints():
    s = cs.summarise(_report())
    assert s["defaults_ms"] == 3.1                      # the re-timed figure wins over the first measurement
    assert s["bf"]["final_ms"] == 1.0 and s["bf"]["n_fitness_calls"] == 3000
    assert abs(s["ga"]["final_ms_median"] - 1.17) < 1e-12
    assert abs(s["ga_vs_bf"]["time_ratio_median"] - 1.17) < 1e-12
    assert abs(s["ga_vs_bf"]["time_ratio_worst_seed"] - 1.30) < 1e-12
    assert abs(s["ga_vs_bf"]["evaluation_ratio"] - 0.05) < 1e-12
    assert abs(s["ga_vs_random_time_ratio_median"] - 1.17 / 1.75) < 1e-12
    curve = s["ga"]["runs"]["1"]["best_so_far_at"]
    assert curve["64"] == 1.5 and curve["125"] == 1.0 and curve["150"] == 1.0 and "250" not in curve


def test_partial_report_has_no_invented_numbers():
    r = _report()
    del r["final"], r["bf"], r["random"]
    s = cs.summarise(r)
    assert s["ga"]["runs"]["1"]["final_ms"] is None and s["ga"]["final_ms_median"] is None
    assert "ga_vs_bf" not in s and "bf" not in s and "random" not in s
    assert s["defaults_ms"] == 3.0


def test_cli_round_trip(tmp_path):
    src, dst = tmp_path / "in.json", tmp_path / "out.json"
    src.write_text(json.dumps(_report()))
    assert cs.main([str(src), str(dst)]) == 0
    assert json.loads(dst.read_text())["tuned_from"] == "bf"


def test_committed_summary_is_what_bench_quotes():
    """bench.stored_campaign() quotes the committed campaign summary with its source and its L2 state (the
    round-1 campaign timed with a warm L2); the paper's own figures are labelled as context."""
    import bench
    assert "Titan X" in bench.PAPER_TUNING_CONTEXT["hardware"]
    st = bench.stored_campaign()
    if os.path.exists(bench.CAMPAIGN_JSON):
        assert "campaign_b200.json" in st["source"] and st["l2"]
        with open(bench.CAMPAIGN_JSON) as fh:
            c = json.load(fh)
        assert st["brute_force"]["final_ms"] == c["bf"]["final_ms"]
        assert st["ga_vs_bf"] == c["ga_vs_bf"]
    else:
        assert st is None


def test_bench_reference_arm_does_not_load_the_product_library():
    """The oracle arm takes its input geometry from the oracle's own delay tables."""
    import subprocess
    import sys
    code = ("import sys, bench; from synth import configs; c = configs.tiny(); "
            "print(bench.oracle_geometry(c)); "
            "assert not any(m.startswith('paper_1811_04165_b200') for m in sys.modules); "
            "assert 'libddp' not in open('/proc/self/maps').read()")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, "-c", code], cwd=root, capture_output=True, text=True)
    assert out.returncode == 0, out.stderr
    assert out.stdout.strip() == "(4440, 4480)"       # cfg0: 4096 + 344, rounded up with the 32-byte slack


def test_oracle_geometry_equals_the_plan_geometry_on_every_config():
    import bench
    import paper_1811_04165_b200 as ddp
    from synth import configs
    for mk in (configs.tiny, configs.apertif_direct, configs.apertif_subband):
        cfg = mk()
        plan = ddp.plan_from_config(cfg, cache_dir=None)
        i = plan.query()
        assert bench.oracle_geometry(cfg) == (int(i.nsamp_in_required), int(i.in_stride_min))
        plan.destroy()
