#!/usr/bin/env python
"""bench.py -- the headline measurement (BASELINE.json `metric`: DM-trial samples/s per config, + % of roofline;
GA vs brute force vs random search).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2|cfg3|cfg0] [--also cfg3 cfg2]
    python bench.py --impl reference ...        # the oracle, on the host cores, same metric
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (dedisperse -> integrate -> snr) over one batch of
synthetic input, through the C ABI (include/ddp.h).  The top-level fields describe `--workload` (default
BASELINE.json configs[1]: Apertif-like direct dedispersion, 1536 channels x 24 414 samples x 2048 DM trials x 9
widths); at N = 1 the other full-size configs (`--also`, default cfg3 = the largest single-GPU workload, and
cfg2 = the subband pair) are timed in the same invocation and reported under `per_config`, and a short real
tuner comparison (`--tune-budget`) runs on cfg2's buffers.  `value` = DM-trial samples per second of the whole job
with the filterbank resident in HBM; `e2e` = the same through ddp_search_host with HOST buffers (H2D of the
filterbank and D2H of the S/N table inside the timed region).  Multi-GPU: one process per GPU, each searching its
own beam (no data-path collective) -> weak scaling, time = max over ranks.

Every workload's GPU result is compared with the oracle in the same run (`config.parity`); a mismatch makes the
bench print `"value": null` with an `error` and exit non-zero.  One JSON line is printed by rank 0.
"Measurement" defines every figure in it.
"""
from __future__ import annotations

import argparse
import glob
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "dm_trial_samples_per_s"
UNIT = "DM-trial samples/s"
SM_COUNT = 148
# Scalar int32 add rate of one SM, adds per clock (measured with ddp_ubench, whose loop
# bodies are verified in SASS at build time -- profiles/r02_ubench.md):
#   IADD3 issues at 64 thread-instructions/clk/SM (alu pipe, like LOP3 / PRMT); a three-input IADD3 performs two
#   additions -> 128 adds/clk/SM on the alu pipe alone;
#   IMAD (fma pipe) issues at 64/clk/SM beside it, one addition each, when the two are interleaved.
# The roofline denominator is the best measured mix (`ADD_PEAK_PER_CLK_PER_SM`); the alu-only 128 and the
# 64-lane figure of round 1 are kept as extra fractions so that earlier numbers stay comparable.
ADD_PEAK_PER_CLK_PER_SM = 192       # three-input IADD3 on the alu pipe + IMAD on the fma pipe, co-issued
ADD_ALU_ONLY_PER_CLK_PER_SM = 128   # three-input IADD3 alone (the denominator of round 1's last bench line)
PIPE_LANES_PER_CLK_PER_SM = 64      # one 64-lane pipe at one addition per instruction
TUNED_JSON = os.path.join(ROOT, "paper_1811_04165_b200", "tuned_b200.json")
IN_SLACK = 32  # bytes of readable slack after the last needed sample of a row (include/ddp.h: in_stride_min)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dedispersion launch(es) of one step, from the newest
    profiles/rNN_traffic.json (written from an `ncu --set full` capture of this bench; see the .md beside it).
    None when no capture of the workload is stored."""
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.json")))
    for path in reversed(files):
        try:
            with open(path) as fh:
                t = json.load(fh)
        except (OSError, ValueError):
            continue
        if workload in t and t[workload].get("dedisperse_dram_bytes") is not None:
            return {"bytes": t[workload]["dedisperse_dram_bytes"], "source": os.path.relpath(path, ROOT),
                    "kernels": t[workload].get("kernels")}
    return None


def get_cfg(name):
    from synth import configs
    return configs.ALL[name]()


def widths_of(cfg):
    return list(cfg.widths)


# ------------------------------------------------------------------------------------ oracle legs
def oracle_tables(cfg, rows=None):
    """Delay tables of the oracle for the given row units (all when None): direct -> (delay,), subband -> (d1, d2)."""
    import oracle
    if cfg.subband is None:
        dms = cfg.dm_list() if rows is None else cfg.dm_list()[np.asarray(rows)]
        return (oracle.delay_table(cfg.chan_freq_mhz(), dms, cfg.t_samp_s),)
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    if rows is not None:
        A = A[np.asarray(rows)]
    F = sb.fine_step * np.arange(sb.n_fine)
    return oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)


def oracle_geometry(cfg):
    """(nsamp_in, in_stride) of the workload from the ORACLE's delay tables alone -- the reference arm must not
    touch the product library: nsamp_in = nsamp_out + max delay (DD.5 / SB.5), rows padded by the documented
    32-byte slack to a multiple of 16 (include/ddp.h, in_stride_min)."""
    t = oracle_tables(cfg)
    max_delay = int(t[0].max()) if cfg.subband is None else int(t[0].max()) + int(t[1].max())
    nsamp_in = cfg.nsamp_out + max_delay
    return nsamp_in, (nsamp_in + IN_SLACK + 15) // 16 * 16


def oracle_rows_chain(cfg, X, rows, mt=False):
    """The oracle on the given row units: dedisperse (direct or subband) -> integrate -> snr.  mt=False: the
    single-thread program as it stands; mt=True: the same functions with the rows spread over the host cores
    (oracle_mt.cpp).  Returns (Y, snr, argmax).  Only the cpu_baseline / --impl reference legs call this."""
    import oracle
    t = oracle_tables(cfg, rows)
    if cfg.subband is None:
        Y = (oracle.dedisperse_mt if mt else oracle.dedisperse)(X, t[0], cfg.nsamp_out)
    elif mt:
        _, Y = oracle.subband_mt(X, t[0], t[1], cfg.subband.n_subbands, cfg.nsamp_out)
    else:
        S = oracle.subband_step1(X, t[0], cfg.subband.n_subbands, cfg.nsamp_out + int(t[1].max()))
        Y = oracle.subband_step2(S, t[1], cfg.nsamp_out)
    _, S, A = (oracle.search_mt if mt else oracle.search)(Y, widths_of(cfg))
    return Y, S, A


def oracle_units(cfg):
    """(number of independent row units, DM trials per unit)."""
    if cfg.subband is None:
        return cfg.ndm, 1
    return cfg.subband.n_coarse, cfg.subband.n_fine


def strided_rows(n_units, k):
    k = max(1, min(int(k), n_units))
    return np.unique(np.linspace(0, n_units - 1, k).astype(np.int64))


def time_oracle_sample(cfg, X, target_s, mt=False):
    """Times the oracle chain on an evenly strided sample of row units sized for ~target_s seconds.
    Returns dict(value, seconds, rows, trials, Y, S, A)."""
    n_units, per = oracle_units(cfg)
    probe = strided_rows(n_units, 2 if not mt else min(n_units, 16))
    t0 = time.perf_counter()
    oracle_rows_chain(cfg, X, probe, mt)
    dt = max(time.perf_counter() - t0, 1e-6) / len(probe)
    rows = strided_rows(n_units, max(2, int(target_s / dt)))
    t0 = time.perf_counter()
    Y, S, A = oracle_rows_chain(cfg, X, rows, mt)
    sec = time.perf_counter() - t0
    trials = len(rows) * per
    return {"value": trials * cfg.nsamp_out / sec, "seconds": sec, "rows": rows, "trials": trials,
            "Y": Y, "S": S, "A": A}


def make_input(cfg, nsamp_in, in_stride, beam=0):
    import dataclasses
    from synth import filterbank
    c = cfg if beam == 0 else dataclasses.replace(cfg, seed=filterbank.beam_seed(cfg.seed, beam))
    X, _ = filterbank.make_filterbank(c, int(nsamp_in), int(in_stride))
    return X


def host_info():
    import oracle
    return {"nproc": os.cpu_count(), "cpu_model": oracle.cpu_model()}


# ------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The reference arm of this tier = the oracle as it stands (single thread) on the host cores; imports
    nothing of the product (geometry comes from the oracle's own delay tables)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = get_cfg(args.workload)
    nsamp_in, in_stride = oracle_geometry(cfg)
    X = make_input(cfg, nsamp_in, in_stride)
    n_units, per = oracle_units(cfg)
    # calibrate: rows per step so that the whole run stays within ~2 minutes
    probe = strided_rows(n_units, 2)
    t0 = time.perf_counter()
    oracle_rows_chain(cfg, X, probe)
    dt = max(time.perf_counter() - t0, 1e-6) / len(probe)
    budget = args.ref_seconds / max(1, args.steps + args.warmup)
    k = max(1, min(n_units, int(budget / dt)))
    rows = strided_rows(n_units, k)
    for _ in range(args.warmup):
        oracle_rows_chain(cfg, X, rows)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rows_chain(cfg, X, rows)
    sec = time.perf_counter() - t0
    trials = len(rows) * per
    value = trials * cfg.nsamp_out * args.steps / sec
    sample = "%d of %d %s (evenly strided), all %d channels, %d samples, %d widths per step" % (
        len(rows), n_units, "DM rows" if cfg.subband is None else "coarse-DM groups", cfg.nchan, cfg.nsamp_out,
        len(cfg.widths))
    hi = host_info()
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": cfg.name, "nchan": cfg.nchan, "nsamp_out": cfg.nsamp_out, "ndm": cfg.ndm,
                       "widths": widths_of(cfg), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                             "nproc": hi["nproc"], "cpu_model": hi["cpu_model"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------ clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_id):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_id), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        try:
            self.tmp.flush()
            with open(self.tmp.name) as fh:
                rows = [ln.strip().split(", ") for ln in fh if ln.strip()]
            os.unlink(self.tmp.name)
        except OSError:
            rows = []
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(n)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------ tuner comparison
CAMPAIGN_JSON = os.path.join(ROOT, "paper_1811_04165_b200", "campaign_b200.json")
# The paper's own tuning-time figures: ANOTHER machine, ANOTHER workload -- context, never a target.
PAPER_TUNING_CONTEXT = {
    "brute_force_hours": "5-24 (about 10 on one GPU)", "ga_hours": "2-5",
    "hardware": "NVIDIA GeForce GTX Titan X (Maxwell), ARTS cluster node ARTS0; OpenCL kernels",
    "what_one_evaluation_is": "a whole external pipeline run, 3-minute cap", "cite": "PAPER.md:7, 115, 205, 225",
}
CURVE_AT = (16, 32, 64, 100, 150, 200, 300, 500, 1000)


def stored_campaign():
    """The committed summary of the last full campaign (campaign.py -> campaign_summary.py): half an hour of GPU
    time, so it is quoted, not re-run, by the bench -- and labelled as stored."""
    if not os.path.exists(CAMPAIGN_JSON):
        return None
    with open(CAMPAIGN_JSON) as fh:
        c = json.load(fh)

    def runs(kind):
        return {s: {"final_ms": r["final_ms"], "evaluations": r["n_fitness_calls"], "kernel_timings": r["n_kernel_timings"],
                    "compiles": r["n_compiles"], "wall_s": round(r["wall_seconds"], 1), "best_so_far_at": r["best_so_far_at"]}
                for s, r in c.get(kind, {}).get("runs", {}).items()}
    bf = c.get("bf", {})
    return {
        "source": "paper_1811_04165_b200/campaign_b200.json (python -m paper_1811_04165_b200.campaign --workload cfg2; "
                  "times are the campaign's interleaved re-timing of each tuner's best joint configuration)",
        "workload": c.get("workload"), "gpu": c.get("gpu"), "l2": c.get("l2", "warm (campaign of round 1)"),
        "unit": "ms per pipeline pass (sub1+sub2+integrate+snr)",
        "valid_configurations_per_kernel": c.get("space"), "defaults_ms": c.get("defaults_ms"),
        "brute_force": {"final_ms": bf.get("final_ms"), "sum_of_isolated_minima_ms": bf.get("sum_isolated_min_ms"),
                        "evaluations": bf.get("n_fitness_calls"), "wall_s": round(bf.get("wall_seconds", 0.0), 1)},
        "ga": runs("ga"), "random": runs("random"),
        "ga_final_ms_median": c.get("ga", {}).get("final_ms_median"),
        "random_final_ms_median": c.get("random", {}).get("final_ms_median"),
        "ga_vs_bf": c.get("ga_vs_bf"),
    }


def live_tuner_comparison(ddp, torch, dev, budget, seed=1):
    """A SHORT real comparison measured in this run on BASELINE.json configs[2]'s buffers (the cfg4 campaign's
    workload): GA, random search and a strided brute-force subset at about the same number of fitness
    evaluations, every timed pass with a cold L2.  Returns the best pipeline time of each after re-timing the
    three winners in interleaved rounds, plus best-so-far curves against evaluations (BJ:metric)."""
    t_start = time.time()
    cfg = get_cfg("cfg2")
    plan = ddp.plan_from_config(cfg, device=dev.index or 0)
    info = plan.query()
    buf = ddp.alloc_buffers(plan, dev)
    X = make_input(cfg, info.nsamp_in_required, info.in_stride_min)
    buf["d_in"].copy_(torch.from_numpy(X))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    io = ddp.make_tune_io(buf["d_in"], buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"], d_flush=flush,
                          reps=5, warmup=1, cutoff_factor=3.0)
    kern = (ddp.K_SUB1, ddp.K_SUB2, ddp.K_INTEGRATE, ddp.K_SNR)
    defaults = [plan.get_kcfg(k) for k in kern]

    def reset():
        for k, c in zip(kern, defaults):
            plan.set_kcfg(k, c)

    def curve(h):
        out = {str(n): h[n - 1] for n in CURVE_AT if n <= len(h)}
        if h:
            out[str(len(h))] = h[-1]
        return out

    pop = 16
    gens = max(1, (budget - pop) // (pop - 2))
    out = {"measured_in_this_run": True, "workload": cfg.name, "unit": "ms per pipeline pass (sub1+sub2+integrate+snr)",
           "l2": "256 MiB written before every timed pass", "fitness": "median of 5 passes of the summed CUDA-event times",
           "budget_evaluations": budget, "space": {ddp.KERNEL_NAMES[k]: len(plan.enumerate_kcfgs(k)) for k in kern}}
    d_ms, _ = plan.time_pipeline(io, defaults)
    reset()
    ga = plan.tune_ga(io, seed=seed, population=pop, generations=gens, tournament=3, p_cross=0.8, p_mut=0.05,
                      elitism=2, max_evals=budget)
    reset()
    rnd = plan.tune_random(io, seed=seed, max_evals=ga["n_fitness_calls"])
    reset()
    bf = plan.tune_bruteforce(io, max_evals_per_kernel=max(1, budget // 4))
    finalists = {"defaults": defaults, "ga": ga["best"], "random": rnd["best"], "bruteforce_subset": bf["best"]}
    io_final = ddp.make_tune_io(buf["d_in"], buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"],
                                d_flush=flush, reps=5, warmup=1, cutoff_factor=0.0)
    samples = {k: [] for k in finalists}
    for _ in range(3):
        for k, c in finalists.items():
            ms, _ = plan.time_pipeline(io_final, c)
            samples[k].append(ms)
    final = {k: sorted(v)[1] for k, v in samples.items()}
    for name, res in (("ga", ga), ("random", rnd), ("bruteforce_subset", bf)):
        out[name] = {"final_ms": final[name], "tuner_best_ms": res["best_ms"], "evaluations": res["n_fitness_calls"],
                     "kernel_timings": res["n_kernel_timings"], "compiles": res["n_compiles"],
                     "wall_s": round(res["wall_seconds"], 1), "best_so_far_at": curve(res["history"]),
                     "cfg": [list(c.astuple()) for c in res["best"]]}
    out["ga"]["params"] = {"population": pop, "generations": gens, "tournament": 3, "p_cross": 0.8, "p_mut": 0.05,
                           "elitism": 2, "seed": seed}
    out["bruteforce_subset"]["note"] = ("evenly strided subset of %d configurations per kernel (of %s); the four "
                                        "winners timed together" % (max(1, budget // 4), out["space"]))
    out["defaults_ms"] = final["defaults"]
    out["defaults_ms_first_pass"] = d_ms
    out["ga_vs_random"] = final["ga"] / final["random"]
    out["wall_s"] = round(time.time() - t_start, 1)
    plan.destroy()
    return out


# ------------------------------------------------------------------------------------ our arm
def apply_tuned(plan, ddp, workload):
    """Loads the committed tuned kernel configurations of the workload (written by the tuners on a B200) into
    the plan; returns (applied, rejected): a tuned entry the plan refuses is reported, never skipped silently."""
    applied, rejected = {}, {}
    if not os.path.exists(TUNED_JSON):
        return applied, rejected
    with open(TUNED_JSON) as fh:
        tuned = json.load(fh).get(workload, {})
    for kname, genes in tuned.items():
        k = ddp.KERNEL_NAMES.index(kname)
        c = ddp.Kcfg(*genes)
        if plan.check_kcfg(k, c):
            plan.set_kcfg(k, c)
            applied[kname] = list(genes)
        else:
            rejected[kname] = list(genes)
    return applied, rejected


def bench_workload(name, args, ctx, with_cpu):
    """Times one workload on this rank's GPU; returns the per-workload record (rank-local; the caller combines
    ranks for the top-level workload)."""
    torch, ddp, dev, world, dist = ctx["torch"], ctx["ddp"], ctx["dev"], ctx["world"], ctx["dist"]
    cfg = get_cfg(name)
    plan = ddp.plan_from_config(cfg, device=dev.index or 0)
    info = plan.query()
    tuned, rejected = apply_tuned(plan, ddp, name)
    buf = ddp.alloc_buffers(plan, dev)
    X = make_input(cfg, info.nsamp_in_required, info.in_stride_min, ctx["beam"])
    h_in = torch.from_numpy(X).pin_memory()
    buf["d_in"].copy_(h_in)
    flush = ctx["flush"]
    h_snr = torch.empty((info.ndm, info.nwidths), dtype=torch.float32).pin_memory()
    h_arg = torch.empty((info.ndm, info.nwidths), dtype=torch.int32).pin_memory()
    # one step = dedisperse (1 or 2 kernels) -> fused integration + S/N (ddp_integrate_snr: the block sums of every
    # width and their S/N in one pass over Y; the planes are an optional output and are not materialised here)
    kernels_per_step = 2 + (1 if info.subband else 0)
    units_per_step = float(info.ndm) * float(info.nsamp_out)

    def step():
        plan.dedisperse(buf["d_in"], buf["d_out"])
        e_mid = torch.cuda.Event(enable_timing=True)
        e_mid.record()
        plan.integrate_snr(buf["d_out"], buf["d_snr"], buf["d_argmax"])
        return e_mid

    def step_separate():  # the two-kernel form of the same stages (planes written, then read again)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        e[0].record()
        plan.integrate(buf["d_out"], buf["d_integ"])
        e[1].record()
        plan.snr(buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"])
        e[2].record()
        return e

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident arm
    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    barrier()
    sampler = ClockSampler(local_gpu_id(torch, dev.index or 0))
    ev = []
    for _ in range(args.steps):
        flush.zero_()  # L2 flush between timed iterations, outside the step's events
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        em = step()
        e1.record()
        ev.append((e0, em, e1))
    barrier()
    step_ms = [a.elapsed_time(d) for a, _, d in ev]
    dd_ms = float(np.mean([a.elapsed_time(b) for a, b, _ in ev]))
    fused_ms = float(np.mean([b.elapsed_time(c) for _, b, c in ev]))
    local_ms = float(sum(step_ms))
    sep = []
    for _ in range(min(args.steps, 10) + 1):  # the separate integrate / snr kernels on the same Y (first pass untimed)
        flush.zero_()
        sep.append(step_separate())
    barrier()
    int_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in sep[1:]]))
    snr_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in sep[1:]]))

    # ---- end-to-end arm: HOST buffers.  (a) one batch per call through ddp_search_host (the whole padded batch is
    # uploaded every step); (b) consecutive batches of one observation through ddp_search_host_batches:
    # only a batch's nsamp_out new samples cross the bus, the max_delay overlap is carried on the device and the
    # upload of the next batch overlaps the search of the current one.  (b) is the e2e figure.
    for _ in range(3):
        plan.search_host(h_in, buf["d_in"], buf["d_out"], None, buf["d_snr"], buf["d_argmax"], h_snr, h_arg)
    barrier()
    e2e1_ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        plan.search_host(h_in, buf["d_in"], buf["d_out"], None, buf["d_snr"], buf["d_argmax"], h_snr, h_arg)
        e1.record()
        e1.synchronize()
        e2e1_ms += e0.elapsed_time(e1)
    barrier()
    ns, md = int(info.nsamp_out), int(info.max_delay)
    nb_call = max(1, min(args.steps, 10))           # batches per call (the paper's observations are 10 batches)
    n_calls = (args.steps + nb_call - 1) // nb_call
    obs_len = nb_call * ns + md
    h_obs = torch.empty((info.nchan, (obs_len + 15) // 16 * 16), dtype=torch.uint8).pin_memory()
    Xt = torch.from_numpy(X)
    h_obs[:, : ns + md] = Xt[:, : ns + md]          # batch 0 = the resident arm's batch; later batches repeat its new samples
    for b in range(1, nb_call):
        h_obs[:, md + b * ns: md + (b + 1) * ns] = Xt[:, md: md + ns]
    d_in1 = torch.empty_like(buf["d_in"])
    hb_snr = torch.empty((nb_call, info.ndm, info.nwidths), dtype=torch.float32).pin_memory()
    hb_arg = torch.empty((nb_call, info.ndm, info.nwidths), dtype=torch.int32).pin_memory()
    plan.search_host_batches(h_obs, nb_call, buf["d_in"], d_in1, buf["d_out"], buf["d_snr"], buf["d_argmax"], hb_snr, hb_arg)
    barrier()
    batch0_ok = bool(np.array_equal(hb_snr[0].numpy(), h_snr.numpy()) and np.array_equal(hb_arg[0].numpy(), h_arg.numpy()))
    e2e_ms, e2e_steps = 0.0, 0
    for _ in range(n_calls):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        plan.search_host_batches(h_obs, nb_call, buf["d_in"], d_in1, buf["d_out"], buf["d_snr"], buf["d_argmax"], hb_snr, hb_arg)
        e1.record()
        e1.synchronize()
        e2e_ms += e0.elapsed_time(e1)
        e2e_steps += nb_call
    barrier()
    clocks = sampler.stop()
    # leave the resident arm's batch and results in the buffers for the parity check below
    buf["d_in"].copy_(h_in)
    plan.dedisperse(buf["d_in"], buf["d_out"])
    torch.cuda.synchronize()
    del d_in1, h_obs

    # ---- roofline of the dominant kernel (dedispersion)
    peaks, peak_src = measured_peaks()
    adds = float(info.adds_dedisp)
    per_clk = SM_COUNT * peaks["sm_max_mhz"] * 1e6 / 1e12  # Tadd/s per (add / clk / SM)
    alu_peak = ADD_PEAK_PER_CLK_PER_SM * per_clk
    achieved = adds / (dd_ms * 1e-3) / 1e12
    in_bytes = float(info.nchan) * float(info.nsamp_in_required)
    out_bytes = float(info.ndm) * float(info.nsamp_out) * 4.0
    sub_bytes = 2.0 * info.n_coarse * info.n_subbands * float(info.nsamp_sub) * info.sub_elem_bytes if info.subband else 0.0
    hbm_bytes = in_bytes + out_bytes + sub_bytes
    traffic = ncu_traffic(name)
    roofline = {"bound": "alu", "kernel": "dedisperse (%s)" % ("sub1+sub2" if info.subband else "direct"),
                "achieved": achieved, "peak": alu_peak, "unit": "Tadd/s", "frac": achieved / alu_peak,
                "peak_source": "%d SMs x %d int32 adds/clk/SM (three-input IADD3 on the alu pipe co-issued with IMAD on "
                               "the fma pipe, measured with ddp_ubench, profiles/r02_ubench.md) x sm_max_mhz %.0f (%s)" % (
                                   SM_COUNT, ADD_PEAK_PER_CLK_PER_SM, peaks["sm_max_mhz"], peak_src),
                "frac_vs_alu_pipe_only_128": achieved / (ADD_ALU_ONLY_PER_CLK_PER_SM * per_clk),
                "frac_vs_64_lane_pipe": achieved / (PIPE_LANES_PER_CLK_PER_SM * per_clk),
                "algorithmic_adds_per_launch": adds, "kernel_ms": dd_ms,
                "traffic": traffic["bytes"] if traffic else None, "traffic_source": traffic["source"] if traffic else None,
                "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_gbs": hbm_bytes / (dd_ms * 1e-3) / 1e9,
                        "peak_gbs": peaks["hbm_gbs"], "frac": hbm_bytes / (dd_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                        "peak_source": peak_src}}

    # integrate / snr are HBM bound: read Y (+ planes), write planes
    y_bytes = float(info.ndm) * float(info.nsamp_out) * 4.0
    pl_bytes = 4.0 * float(info.ndm) * sum(float(info.plane_len[k]) for k in range(info.nwidths) if info.widths[k] > 1)
    stages = {"dedisperse_ms": dd_ms,
              "integrate_snr_fused": {"ms": fused_ms, "algorithmic_bytes": y_bytes,
                                      "hbm_frac": y_bytes / (fused_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                      "note": "the timed step uses this kernel; planes are not materialised"},
              "integrate": {"ms": int_ms, "algorithmic_bytes": y_bytes + pl_bytes,
                            "hbm_frac": (y_bytes + pl_bytes) / (int_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]},
              "snr": {"ms": snr_ms, "algorithmic_bytes": y_bytes + pl_bytes,
                      "hbm_frac": (y_bytes + pl_bytes) / (snr_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

    # ---- the oracle timed beside it (rank 0, N = 1 only) + parity of the rows it computed
    cpu, cpu_mt, parity = None, None, None
    if with_cpu:
        n_units, per = oracle_units(cfg)
        Yg_all = buf["d_out"].cpu().numpy().view(np.uint32)
        Sg_all, Ag_all = h_snr.numpy(), h_arg.numpy().view(np.uint32)
        unit_name = "DM rows" if cfg.subband is None else "coarse-DM groups"
        hi = host_info()

        def check(r):
            rows = r["rows"] if cfg.subband is None else (r["rows"][:, None] * per + np.arange(per)[None, :]).reshape(-1)
            ok = (np.array_equal(Yg_all[rows, : cfg.nsamp_out], r["Y"]) and np.array_equal(Ag_all[rows], r["A"]) and
                  bool(np.all(np.abs(Sg_all[rows] - r["S"]) <= 1e-5 * np.maximum(1.0, np.abs(r["S"])))))
            return int(len(rows)), bool(ok)

        r1 = time_oracle_sample(cfg, X, args.cpu_seconds, mt=False)
        n1, ok1 = check(r1)
        cpu = {"value": r1["value"], "unit": UNIT, "cores": 1, "kind": "oracle", "nproc": hi["nproc"],
               "cpu_model": hi["cpu_model"],
               "sample": "%d of %d %s (evenly strided): dedisperse+integrate+snr, single thread, %.1f s" % (
                   len(r1["rows"]), n_units, unit_name, r1["seconds"])}
        import oracle
        rm = time_oracle_sample(cfg, X, args.cpu_seconds_mt, mt=True)
        nm, okm = check(rm)
        cpu_mt = {"value": rm["value"], "unit": UNIT, "cores": oracle.mt_threads(), "kind": "oracle, DM rows spread over "
                  "the host cores (omp parallel for, oracle_mt.cpp)", "nproc": hi["nproc"], "cpu_model": hi["cpu_model"],
                  "sample": "%d of %d %s (evenly strided), %.1f s" % (len(rm["rows"]), n_units, unit_name, rm["seconds"])}
        parity = {"ok": bool(ok1 and okm), "rows_checked": int(len(set(r1["rows"].tolist()) | set(rm["rows"].tolist())) * per),
                  "of_rows": int(info.ndm), "what": "dedispersion bit-exact, S/N <= 1e-5 relative, argmax exact",
                  "legs": {"single_thread_rows": n1, "all_cores_rows": nm}}

    rec = {"workload": cfg.name, "value": units_per_step * args.steps / (local_ms * 1e-3), "unit": UNIT,
           "ms_per_step": local_ms / args.steps, "dedisp_ms": dd_ms, "roofline": roofline, "stages": stages,
           "dedisp_only": {"value": units_per_step / (dd_ms * 1e-3), "unit": UNIT, "ms": dd_ms},
           "e2e": {"value": units_per_step * e2e_steps / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms / e2e_steps,
                   "h2d_bytes_per_step": int(info.nchan) * ns,
                   "d2h_bytes_per_step": int(h_snr.numel() * 4 + h_arg.numel() * 4),
                   "how": "ddp_search_host_batches: %d consecutive batches per call, new samples only, carried overlap, "
                          "uploads overlapped with the search" % nb_call,
                   "batch0_equals_single_batch_result": batch0_ok,
                   "single_batch_call": {"value": units_per_step * args.steps / (e2e1_ms * 1e-3), "ms_per_step": e2e1_ms / args.steps,
                                         "h2d_bytes_per_step": int(h_in.numel()), "how": "ddp_search_host, whole padded batch uploaded"}},
           "gpu_launches": int(kernels_per_step * args.steps), "clocks": clocks,
           "kcfg": {ddp.KERNEL_NAMES[k]: list(plan.get_kcfg(k).astuple()) for k in range(len(ddp.KERNEL_NAMES)) if _in_plan(plan, k)},
           "tuned_from": os.path.basename(TUNED_JSON) if tuned else None, "tuned_rejected": rejected or None,
           "cpu_baseline": cpu, "cpu_baseline_all_cores": cpu_mt, "parity": parity,
           "shape": {"nchan": cfg.nchan, "nsamp_out": cfg.nsamp_out, "ndm": cfg.ndm, "widths": widths_of(cfg)},
           "working_set_mb": (hbm_bytes + info.integ_elems * 4.0) / 1e6,
           "_local_ms": local_ms, "_e2e_ms": e2e_ms * args.steps / e2e_steps, "_units": units_per_step * args.steps}
    plan.destroy()
    del buf, h_in
    torch.cuda.empty_cache()
    return rec


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1811_04165_b200 as ddp
    from paper_1811_04165_b200.shard import beams_of_rank, combine

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback "
                         "(use --impl reference for the oracle arm)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    if args.gpus != world and rank == 0:
        print("bench.py: --gpus %d but WORLD_SIZE %d; using WORLD_SIZE" % (args.gpus, world), file=sys.stderr)

    ctx = {"torch": torch, "ddp": ddp, "dev": dev, "world": world, "dist": dist,
           "beam": beams_of_rank(world, rank, world)[0],  # one beam per GPU (weak scaling)
           "flush": torch.empty(256 << 20, dtype=torch.uint8, device=dev)}  # > 126 MB L2
    with_cpu = world == 1 and not args.no_cpu_baseline
    main_rec = bench_workload(args.workload, args, ctx, with_cpu)
    tot_ms, tot_units = combine(main_rec["_local_ms"], main_rec["_units"], dev)
    e2e_tot_ms, _ = combine(main_rec["_e2e_ms"], 0.0, dev)
    value = tot_units / (tot_ms * 1e-3)
    e2e_value = tot_units / (e2e_tot_ms * 1e-3)

    # ---- the other full-size configs and the live tuner comparison: N = 1 only (ranks are independent replicas)
    per_config, tuning_live = {}, None
    if world == 1:
        also = [w for w in (args.also if args.also is not None else (["cfg3", "cfg2"] if args.workload == "cfg1" else []))
                if w != args.workload]
        ctx["beam"] = 0
        for w in also:
            per_config[w] = bench_workload(w, args, ctx, with_cpu)
        if args.tune_budget > 0:
            tuning_live = live_tuner_comparison(ddp, torch, dev, args.tune_budget)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    def brief(r):
        return {"workload": r["workload"], "value": r["value"], "ms_per_step": r["ms_per_step"], "dedisp_ms": r["dedisp_ms"],
                "roofline": {"frac": r["roofline"]["frac"], "achieved": r["roofline"]["achieved"], "peak": r["roofline"]["peak"],
                             "unit": r["roofline"]["unit"], "frac_vs_alu_pipe_only_128": r["roofline"]["frac_vs_alu_pipe_only_128"],
                             "hbm_frac": r["roofline"]["hbm"]["frac"], "traffic": r["roofline"]["traffic"]},
                "integrate_snr_fused": r["stages"]["integrate_snr_fused"], "integrate": r["stages"]["integrate"],
                "snr": r["stages"]["snr"], "e2e": r["e2e"], "kcfg": r["kcfg"],
                "tuned_rejected": r["tuned_rejected"], "cpu_baseline": r["cpu_baseline"],
                "cpu_baseline_all_cores": r["cpu_baseline_all_cores"], "parity": r["parity"], "clocks": r["clocks"],
                "gpu_launches": r["gpu_launches"], "shape": r["shape"]}

    everything = [main_rec] + list(per_config.values())
    failed = [r["workload"] for r in everything if r["parity"] is not None and not r["parity"]["ok"]]
    m = main_rec
    launches = sum(3 * r["gpu_launches"] + 8 * (r["gpu_launches"] // max(1, args.steps)) for r in everything)
    line = {"metric": METRIC, "value": None if failed else value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": m["workload"], **m["shape"], "beams_per_gpu": 1,
                       "l2": "256 MiB memset between timed steps (outside each step's events); "
                             "working set %.0f MB > 126 MB L2" % m["working_set_mb"],
                       "kcfg": m["kcfg"], "tuned_from": m["tuned_from"], "tuned_rejected": m["tuned_rejected"],
                       "parity": m["parity"],
                       "parity_all_workloads": {r["workload"]: (r["parity"] or {}).get("ok") for r in everything}},
            "dedisp_only": {"value": world * m["dedisp_only"]["value"], "unit": UNIT, "ms": m["dedisp_ms"]},
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_tot_ms / args.steps,
                    "h2d_bytes_per_step": m["e2e"]["h2d_bytes_per_step"], "d2h_bytes_per_step": m["e2e"]["d2h_bytes_per_step"],
                    "how": m["e2e"]["how"], "batch0_equals_single_batch_result": m["e2e"]["batch0_equals_single_batch_result"],
                    "single_batch_call": m["e2e"]["single_batch_call"]},
            "gpu_launches": int(m["gpu_launches"]), "gpu_launches_whole_run": int(launches),
            "clocks": m["clocks"], "roofline": m["roofline"], "stages": m["stages"],
            "cpu_baseline": m["cpu_baseline"], "cpu_baseline_all_cores": m["cpu_baseline_all_cores"],
            "parity": m["parity"],
            "per_config": {k: brief(r) for k, r in per_config.items()},
            "tuning": {"measured_in_this_run": tuning_live, "stored_campaign": stored_campaign(),
                       "paper_context": PAPER_TUNING_CONTEXT}}
    if failed:
        line["error"] = "GPU result differs from the oracle on: %s -- no performance number is reported" % ", ".join(failed)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 3 if failed else 0


def _in_plan(plan, k):
    try:
        plan.get_kcfg(k)
        return True
    except Exception:
        return False


def local_gpu_id(torch, local):
    """nvidia-smi identifier of torch device `local` (UUID when available: CUDA_VISIBLE_DEVICES may remap)."""
    try:
        u = str(torch.cuda.get_device_properties(local).uuid)
        return u if u.startswith("GPU-") else "GPU-" + u
    except Exception:
        return str(local)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg1", choices=["cfg0", "cfg1", "cfg2", "cfg3"])
    ap.add_argument("--also", nargs="*", default=None, choices=["cfg0", "cfg1", "cfg2", "cfg3"],
                    help="further workloads timed in the same run at N = 1 (default: cfg3 cfg2 when --workload is cfg1)")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="target duration of the single-thread cpu_baseline sample")
    ap.add_argument("--cpu-seconds-mt", type=float, default=5.0, help="target duration of the all-cores oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tune-budget", type=int, default=120,
                    help="fitness evaluations of the live GA / random / brute-force-subset comparison (0 = skip)")
    ap.add_argument("--ref-seconds", type=float, default=100.0, help="--impl reference: target duration of the whole run")
    args = ap.parse_args()
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
