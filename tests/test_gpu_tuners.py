"""-m gpu: the tuners on the REAL fitness (CUDA-event timing harness), tiny budgets.

The fake-fitness tests (test_tuners.py) pin the tuners' logic; these check that the hardware harness
times real launches through the same C ABI, that its bookkeeping holds, and that a plan left at the
tuned configurations still reproduces the oracle bit for bit.
"""
from __future__ import annotations

import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)

import paper_1811_04165_b200 as ddp  # noqa: E402
from synth import configs  # noqa: E402
from synth.configs import SubbandPlan  # noqa: E402

pytestmark = pytest.mark.gpu

from gpu_common import GpuSearch, compare_all, oracle_subband  # noqa: E402


def _plan():
    cfg = configs.scaled(configs.apertif_direct(), name="tune_sb", nchan=128, nsamp_out=4200, ndm=16 * 8,
                         widths=(1, 2, 4, 8), n_pulses=2,
                         subband=SubbandPlan(n_subbands=8, n_coarse=16, coarse_first=0.0, coarse_step=8.0,
                                             n_fine=8, fine_step=0.25))
    g = GpuSearch(cfg)
    io = ddp.make_tune_io(g.buf["d_in"], g.buf["d_out"], g.buf["d_integ"], g.buf["d_snr"], g.buf["d_argmax"],
                          reps=3, warmup=1, cutoff_factor=3.0)
    return cfg, g, io


SLOT_KERNEL = (ddp.K_SUB1, ddp.K_SUB2, ddp.K_INTEGRATE, ddp.K_SNR)


def _check_result(g, res, max_calls):
    assert 0 < res["n_fitness_calls"] <= max_calls
    assert res["n_kernel_timings"] >= 4 * res["n_fitness_calls"]  # >= one timed pass of four kernels per call
    assert math.isfinite(res["best_ms"]) and res["best_ms"] > 0.0
    h = res["history"]
    assert len(h) == res["n_fitness_calls"]
    assert all(b <= a for a, b in zip(h, h[1:])) and h[-1] == res["best_ms"]  # best-so-far never rises
    for s, k in enumerate(SLOT_KERNEL):
        assert g.plan.check_kcfg(k, res["best"][s])
        assert g.plan.get_kcfg(k).astuple() == res["best"][s].astuple()     # best is left active in the plan
    assert all(t > 0.0 for t in res["kernel_ms"])
    assert abs(sum(res["kernel_ms"]) - res["best_ms"]) <= 0.25 * res["best_ms"]


def test_time_pipeline_on_hardware_is_positive_and_repeatable():
    cfg, g, io = _plan()
    c = [g.plan.get_kcfg(k) for k in SLOT_KERNEL]
    a, per_a = g.plan.time_pipeline(io, c)
    b, per_b = g.plan.time_pipeline(io, c)
    assert a > 0.0 and b > 0.0 and all(t > 0.0 for t in per_a)
    assert abs(a - b) <= 0.5 * min(a, b)          # medians of the same launches: same order of magnitude
    assert abs(sum(per_a) - a) <= 0.25 * a
    g.close()


def test_ga_random_bruteforce_on_hardware_then_parity():
    cfg, g, io = _plan()
    So, Yo = oracle_subband(cfg, g.X)
    ga = g.plan.tune_ga(io, seed=1, population=8, generations=2, elitism=2)
    _check_result(g, ga, 8 + 2 * 6)
    g.run_all()                                    # with the GA's best configurations active
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="after tune_ga")

    rnd = g.plan.tune_random(io, seed=1, max_evals=10)
    _check_result(g, rnd, 10)
    g.run_all()
    compare_all(g, Yo, what="after tune_random")

    bf = g.plan.tune_bruteforce(io, max_evals_per_kernel=6)
    assert bf["n_fitness_calls"] <= 4 * 6 and math.isfinite(bf["best_ms"]) and bf["best_ms"] > 0.0
    for s, k in enumerate(SLOT_KERNEL):
        assert g.plan.get_kcfg(k).astuple() == bf["best"][s].astuple()
    g.run_all()
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="after tune_bruteforce")
    g.close()
