"""The statistics of the paper's GA experiments (PAPER.md P:231 c_v, P:253 histogram) and the tuners' "end
configurations" output, on a fake fitness -- no GPU.  Closed forms pin the statistics; the tuner output is pinned
by what the algorithm fixes (GA: the last population, ranked, every member valid and its fitness the callback's;
random search: its last draws in order)."""
import math

import pytest

import paper_1811_04165_b200 as ddp
from paper_1811_04165_b200 import study
from test_tuners import Fake, GENES, sub_plan, valid_targets


def test_gene_cv_closed_forms():
    # two configurations, one slot: threads_t 16 and 48 -> mu 32, sigma 16 -> 0.5; a constant gene -> 0;
    # staging all zero -> 0; staging 0 and 2 -> mu 1, sigma 1 -> 1.0
    a = [[16, 4, 8, 2, 1, 0, 4]]
    b = [[48, 4, 8, 6, 1, 0, 4]]
    cv = study.gene_cv([a, b], slots=[0])["0"]
    assert cv["threads_t"] == pytest.approx(0.5)
    assert cv["threads_dm"] == 0.0 and cv["staging"] == 0.0
    assert cv["dms_per_thread"] == pytest.approx(2.0 / 4.0)
    b2 = [[48, 4, 8, 6, 1, 2, 4]]
    assert study.gene_cv([a, b2], slots=[0])["0"]["staging"] == pytest.approx(1.0)
    # three equal configurations: every c_v is 0
    assert all(v == 0.0 for v in study.gene_cv([a, a, a], slots=[0])["0"].values())
    # scale invariance (the reason the paper uses sigma / mu): doubling every value leaves c_v unchanged
    d = [[[2 * x for x in a[0]]], [[2 * x for x in b[0]]]]
    cv2 = study.gene_cv(d, slots=[0])["0"]
    assert cv2["threads_t"] == pytest.approx(cv["threads_t"])


def test_mean_cv_histogram_and_curve():
    r1 = {"0": {"threads_t": 0.2, "staging": float("inf")}}
    r2 = {"0": {"threads_t": 0.4, "staging": 1.0}}
    m = study.mean_cv([r1, r2])
    assert m["0"]["threads_t"] == pytest.approx(0.3) and m["0"]["staging"] == pytest.approx(1.0)
    assert study.histogram([0.0, 0.1, 0.5, 0.99, 1.0], 0.0, 1.0, 4) == [2, 0, 1, 2]
    assert study.histogram([3.0, 3.0], 3.0, 3.0, 3) == [2, 0, 0]
    assert study.curve_at([5.0, 4.0, 4.0, 2.0], [1, 3, 4, 10]) == [5.0, 4.0, 2.0, 2.0]


def test_ga_and_random_report_their_end_configurations():
    plan = sub_plan()
    fake = Fake(plan, valid_targets(plan))
    io = ddp.make_tune_io(fitness=fake)
    r = plan.tune_ga(io, seed=3, population=20, generations=1 << 20, tournament=4, p_cross=0.8, p_mut=0.1,
                     mutation_kind=1, elitism=0, replacement=1, max_evals=200, final_cap=20)
    fin = r["final"]
    assert len(fin) == 20
    fits = [f for _, f in fin]
    assert fits == sorted(fits) and fits[0] == pytest.approx(r["best_ms"])   # ranked, best first (P:201 keeps the fittest)
    for joint, f in fin:
        for s, k in fake.kernels.items():
            assert plan.check_kcfg(k, joint[s])
        genes = tuple(tuple(getattr(joint[s], n) for n in GENES) for s in range(4))
        assert genes in fake.calls                                            # every member was evaluated
        assert f == pytest.approx(1.0 + sum(fake.slot_cost(s, genes[s]) for s in fake.slots))
    # the GA converges: its end configurations vary less than random search's (Fig. 4)
    fake2 = Fake(plan, valid_targets(plan))
    rr = plan.tune_random(ddp.make_tune_io(fitness=fake2), seed=3, max_evals=200, final_cap=20)
    assert len(rr["final"]) == 20
    last20 = fake2.calls[-20:]
    got = [tuple(tuple(getattr(j[s], n) for n in GENES) for s in range(4)) for j, _ in rr["final"]]
    assert got == last20                                                       # the last draws, in order
    cv_ga = study.gene_cv([[list(c.astuple()) for c in j] for j, _ in fin], [0, 1, 2, 3])
    cv_rn = study.gene_cv([[list(c.astuple()) for c in j] for j, _ in rr["final"]], [0, 1, 2, 3])
    mean = lambda cv: sum(v for row in cv.values() for g, v in row.items() if math.isfinite(v)) / 28.0
    assert mean(cv_ga) < mean(cv_rn)
    # final_cap = 0: nothing recorded
    assert plan.tune_random(ddp.make_tune_io(fitness=Fake(plan, valid_targets(plan))), seed=1, max_evals=10)["final"] == []
    plan.destroy()
