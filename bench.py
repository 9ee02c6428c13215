#!/usr/bin/env python
"""bench.py -- the headline measurement (BASELINE.json `metric`: DM-trial samples/s, + % of roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2|cfg3|cfg0]
    python bench.py --impl reference ...        # the oracle, on the host cores, same metric
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (dedisperse -> integrate -> snr) over one
batch of synthetic input (BASELINE.json configs[1] by default: Apertif-like direct dedispersion,
1536 channels x 24 414 samples x 2048 DM trials x 9 widths), through the C ABI (include/ddp.h).
`value` = DM-trial samples per second of the whole job with the filterbank resident in HBM;
`e2e` = the same through ddp_search_host with HOST buffers (H2D of the filterbank and D2H of the
S/N table inside the timed region).  Multi-GPU: one process per GPU, each searching its own beam
(no data-path collective) -> weak scaling, time = max over ranks.

One JSON line is printed by rank 0.  DESIGN.md "Measurement" defines every figure in it.
"""
from __future__ import annotations

import argparse
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
# Scalar int32 add rate of one SM.  MEASURED on B200 with ddp_ubench (profiles/r01_ubench.md): a
# dependent-free IADD3 stream sustains 126.4-127.4 thread-adds/clk/SM, the issue-port limit of 4 SMSP x 32
# lanes, i.e. twice the 64/clk of LOP3 / PRMT / IMAD / IDP.4A (63.2-63.9 measured).  Until the end of round 1
# the roofline used 64 (the B300 guide's alu-pipe width), which overstated every fraction by 2x; the old
# figure is still reported as roofline.frac_vs_64_lane_pipe for continuity.
ADD_LANES_PER_CLK_PER_SM = 128
ALU_LANES_PER_CLK_PER_SM = 64  # LOP3 / PRMT / IMAD pipes: 4 SMSP x 16 lanes/clk (B300_MICROARCH "Pipe rates"; measured 63.7)
TUNED_JSON = os.path.join(ROOT, "paper_1811_04165_b200", "tuned_b200.json")
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists for the workload).
# dram__bytes_read.sum + dram__bytes_write.sum of the dedispersion launch(es) from one `ncu --set full` capture
# (stored, not measured by the bench; cold-cache, ncu flushes caches between replay passes):
#   cfg1  profiles/r01_final.md  221.2 MB read + 171.2 MB written (1.54x algorithmic, see the profile)
#   cfg2  profiles/r01_final.md  sub1 49.2 + 48.6 MB, sub2 101.0 + 145.9 MB
#   cfg3  profiles/r01_final.md  1170.0 MB read + 309.8 MB written
NCU_TRAFFIC_BYTES = {"cfg1": 392428032, "cfg2": 344683520, "cfg3": 1479793472}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def get_cfg(name):
    from synth import configs
    return configs.ALL[name]()


def widths_of(cfg):
    return list(cfg.widths)


# ------------------------------------------------------------------------------------ oracle legs
def oracle_rows_chain(cfg, X, rows):
    """The oracle as it stands on the given DM rows: dedisperse (direct or subband) -> integrate ->
    snr.  Returns (Y, snr, argmax).  Only the cpu_baseline / --impl reference legs call this."""
    import oracle
    if cfg.subband is None:
        dms = cfg.dm_list()[np.asarray(rows)]
        delay = oracle.delay_table(cfg.chan_freq_mhz(), dms, cfg.t_samp_s)
        Y = oracle.dedisperse(X, delay, cfg.nsamp_out)
    else:  # rows = coarse-DM indices; every fine DM of them is produced
        sb = cfg.subband
        A = (sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse))[np.asarray(rows)]
        F = sb.fine_step * np.arange(sb.n_fine)
        d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)
        S = oracle.subband_step1(X, d1, sb.n_subbands, cfg.nsamp_out + int(d2.max()))
        Y = oracle.subband_step2(S, d2, cfg.nsamp_out)
    _, S, A = oracle.search(Y, widths_of(cfg))
    return Y, S, A


def oracle_units(cfg):
    """(number of independent row units, DM trials per unit)."""
    if cfg.subband is None:
        return cfg.ndm, 1
    return cfg.subband.n_coarse, cfg.subband.n_fine


def strided_rows(n_units, k):
    k = max(1, min(int(k), n_units))
    return np.unique(np.linspace(0, n_units - 1, k).astype(np.int64))


def time_oracle_sample(cfg, X, target_s):
    """Times the oracle chain on an evenly strided sample of row units sized for ~target_s seconds.
    Returns dict(value, seconds, rows, trials, Y, S, A)."""
    n_units, per = oracle_units(cfg)
    probe = strided_rows(n_units, 2)
    t0 = time.perf_counter()
    oracle_rows_chain(cfg, X, probe)
    dt = max(time.perf_counter() - t0, 1e-6) / len(probe)
    rows = strided_rows(n_units, max(2, int(target_s / dt)))
    t0 = time.perf_counter()
    Y, S, A = oracle_rows_chain(cfg, X, rows)
    sec = time.perf_counter() - t0
    trials = len(rows) * per
    return {"value": trials * cfg.nsamp_out / sec, "seconds": sec, "rows": rows, "trials": trials,
            "Y": Y, "S": S, "A": A}


def make_input(cfg, info_nsamp_in, in_stride, beam=0):
    import dataclasses
    from paper_1811_04165_b200.shard import beam_seed
    from synth import filterbank
    c = cfg if beam == 0 else dataclasses.replace(cfg, seed=beam_seed(cfg.seed, beam))
    X, _ = filterbank.make_filterbank(c, int(info_nsamp_in), int(in_stride))
    return X


def host_geometry(cfg):
    """in_stride / nsamp_in of the workload without touching the GPU (plan creation is host code)."""
    import paper_1811_04165_b200 as ddp
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    i = plan.query()
    out = (int(i.nsamp_in_required), int(i.in_stride_min))
    plan.destroy()
    return out


# ------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = get_cfg(args.workload)
    nsamp_in, in_stride = host_geometry(cfg)
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
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": cfg.name, "nchan": cfg.nchan, "nsamp_out": cfg.nsamp_out, "ndm": cfg.ndm,
                       "widths": widths_of(cfg), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
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


def tuning_report():
    """GA vs brute force vs random search (BASELINE.json metric, configs[4]).  A campaign takes about
    half an hour of GPU time, so it is NOT run inside the bench: this quotes the committed summary of
    the last campaign (campaign.py -> campaign_summary.py) and says so.  None if no campaign is stored."""
    out = {"measured_in_this_run": False, "paper_context": PAPER_TUNING_CONTEXT, "stored": None}
    if not os.path.exists(CAMPAIGN_JSON):
        return out
    with open(CAMPAIGN_JSON) as fh:
        c = json.load(fh)
    def runs(kind):
        return {s: {"final_ms": r["final_ms"], "evaluations": r["n_fitness_calls"], "kernel_timings": r["n_kernel_timings"],
                    "compiles": r["n_compiles"], "wall_s": round(r["wall_seconds"], 1), "best_so_far_at": r["best_so_far_at"]}
                for s, r in c.get(kind, {}).get("runs", {}).items()}
    bf = c.get("bf", {})
    out["stored"] = {
        "source": "paper_1811_04165_b200/campaign_b200.json (python -m paper_1811_04165_b200.campaign --workload cfg2; "
                  "times are the campaign's interleaved re-timing of each tuner's best joint configuration)",
        "workload": c.get("workload"), "gpu": c.get("gpu"), "unit": "ms per pipeline pass (sub1+sub2+integrate+snr)",
        "valid_configurations_per_kernel": c.get("space"), "defaults_ms": c.get("defaults_ms"),
        "brute_force": {"final_ms": bf.get("final_ms"), "sum_of_isolated_minima_ms": bf.get("sum_isolated_min_ms"),
                        "evaluations": bf.get("n_fitness_calls"), "wall_s": round(bf.get("wall_seconds", 0.0), 1)},
        "ga": runs("ga"), "random": runs("random"),
        "ga_final_ms_median": c.get("ga", {}).get("final_ms_median"),
        "random_final_ms_median": c.get("random", {}).get("final_ms_median"),
        "ga_vs_bf": c.get("ga_vs_bf"),
        "note": "wall_s of seeds after the first is warm: compiled code shapes are memoised within the campaign process",
    }
    return out


# ------------------------------------------------------------------------------------ our arm
def apply_tuned(plan, ddp, workload):
    """Loads the committed tuned kernel configurations of the workload (written by the tuners on a
    B200) into the plan; returns the names applied."""
    applied = {}
    if not os.path.exists(TUNED_JSON):
        return applied
    with open(TUNED_JSON) as fh:
        tuned = json.load(fh).get(workload, {})
    for kname, genes in tuned.items():
        k = ddp.KERNEL_NAMES.index(kname)
        c = ddp.Kcfg(*genes)
        if plan.check_kcfg(k, c):
            plan.set_kcfg(k, c)
            applied[kname] = list(genes)
    return applied


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

    cfg = get_cfg(args.workload)
    plan = ddp.plan_from_config(cfg, device=local)
    info = plan.query()
    tuned = apply_tuned(plan, ddp, args.workload)
    buf = ddp.alloc_buffers(plan, dev)
    beam = beams_of_rank(world, rank, world)[0]  # one beam per GPU (weak scaling)
    X = make_input(cfg, info.nsamp_in_required, info.in_stride_min, beam)
    h_in = torch.from_numpy(X).pin_memory()
    buf["d_in"].copy_(h_in)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    h_snr = torch.empty((info.ndm, info.nwidths), dtype=torch.float32).pin_memory()
    h_arg = torch.empty((info.ndm, info.nwidths), dtype=torch.int32).pin_memory()
    kernels_per_step = 3 + (1 if info.subband else 0) - (0 if info.integ_elems > 0 else 1)
    units_per_step = float(info.ndm) * float(info.nsamp_out)

    def step():
        plan.dedisperse(buf["d_in"], buf["d_out"])
        e_mid = torch.cuda.Event(enable_timing=True)
        e_mid.record()
        plan.integrate(buf["d_out"], buf["d_integ"])
        e_int = torch.cuda.Event(enable_timing=True)
        e_int.record()
        plan.snr(buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"])
        return e_mid, e_int

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
    sampler = ClockSampler(local_gpu_id(torch, local))
    ev = []
    for _ in range(args.steps):
        flush.zero_()  # L2 flush between timed iterations, outside the step's events
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        em, ei = step()
        e1.record()
        ev.append((e0, em, ei, e1))
    barrier()
    step_ms = [a.elapsed_time(d) for a, _, _, d in ev]
    dd_ms = [a.elapsed_time(b) for a, b, _, _ in ev]
    int_ms = float(np.mean([b.elapsed_time(c) for _, b, c, _ in ev]))
    snr_ms = float(np.mean([c.elapsed_time(d) for _, _, c, d in ev]))
    local_ms = float(sum(step_ms))
    tot_ms, tot_units = combine(local_ms, units_per_step * args.steps, dev)
    value = tot_units / (tot_ms * 1e-3)

    # ---- end-to-end arm: host buffers through ddp_search_host
    for _ in range(3):
        plan.search_host(h_in, buf["d_in"], buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"], h_snr, h_arg)
    barrier()
    e2e_ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        plan.search_host(h_in, buf["d_in"], buf["d_out"], buf["d_integ"], buf["d_snr"], buf["d_argmax"], h_snr, h_arg)
        e1.record()
        e1.synchronize()
        e2e_ms += e0.elapsed_time(e1)
    barrier()
    clocks = sampler.stop()
    e2e_tot_ms, _ = combine(e2e_ms, 0.0, dev)
    e2e_value = tot_units / (e2e_tot_ms * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (dedispersion)
    peaks, peak_src = measured_peaks()
    dd_avg_ms = float(np.mean(dd_ms))
    adds = float(info.adds_dedisp)
    alu_peak = SM_COUNT * ADD_LANES_PER_CLK_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12  # Tadd/s
    pipe64_peak = SM_COUNT * ALU_LANES_PER_CLK_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12
    achieved = adds / (dd_avg_ms * 1e-3) / 1e12
    in_bytes = float(info.nchan) * float(info.nsamp_in_required)
    out_bytes = float(info.ndm) * float(info.nsamp_out) * 4.0
    sub_bytes = 2.0 * info.n_coarse * info.n_subbands * float(info.nsamp_sub) * info.sub_elem_bytes if info.subband else 0.0
    hbm_bytes = in_bytes + out_bytes + sub_bytes
    roofline = {"bound": "alu", "kernel": "dedisperse (%s)" % ("sub1+sub2" if info.subband else "direct"),
                "achieved": achieved, "peak": alu_peak, "unit": "Tadd/s", "frac": achieved / alu_peak,
                "peak_source": "%d SMs x %d int32 adds/clk/SM (IADD3 issue rate, measured 126.4-127.4 with ddp_ubench, "
                               "profiles/r01_ubench.md) x sm_max_mhz %.0f (%s)" % (
                    SM_COUNT, ADD_LANES_PER_CLK_PER_SM, peaks["sm_max_mhz"], peak_src),
                "frac_vs_64_lane_pipe": achieved / pipe64_peak,  # the denominator used until the end of round 1
                "algorithmic_adds_per_launch": adds, "kernel_ms": dd_avg_ms,
                "traffic": NCU_TRAFFIC_BYTES.get(args.workload),
                "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_gbs": hbm_bytes / (dd_avg_ms * 1e-3) / 1e9,
                        "peak_gbs": peaks["hbm_gbs"], "frac": hbm_bytes / (dd_avg_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                        "peak_source": peak_src}}

    # integrate / snr are HBM bound: read Y (+ planes), write planes
    y_bytes = float(info.ndm) * float(info.nsamp_out) * 4.0
    pl_bytes = 4.0 * float(info.ndm) * sum(float(info.plane_len[k]) for k in range(info.nwidths) if info.widths[k] > 1)
    stages = {"dedisperse_ms": dd_avg_ms,
              "integrate": {"ms": int_ms, "algorithmic_bytes": y_bytes + pl_bytes,
                            "hbm_frac": (y_bytes + pl_bytes) / (int_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]},
              "snr": {"ms": snr_ms, "algorithmic_bytes": y_bytes + pl_bytes,
                      "hbm_frac": (y_bytes + pl_bytes) / (snr_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}}

    # ---- the oracle timed beside it (rank 0, N = 1 only) + parity of the sampled rows
    cpu = None
    parity = None
    if world == 1 and not args.no_cpu_baseline:
        r = time_oracle_sample(cfg, X, args.cpu_seconds)
        n_units, per = oracle_units(cfg)
        sample = "%d of %d %s (evenly strided): dedisperse+integrate+snr, %.1f s" % (
            len(r["rows"]), n_units, "DM rows" if cfg.subband is None else "coarse-DM groups", r["seconds"])
        cpu = {"value": r["value"], "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample}
        rows = r["rows"] if cfg.subband is None else (
            r["rows"][:, None] * per + np.arange(per)[None, :]).reshape(-1)
        Yg = buf["d_out"].cpu().numpy().view(np.uint32)[rows, : cfg.nsamp_out]
        Sg = h_snr.numpy()[rows]
        Ag = h_arg.numpy().view(np.uint32)[rows]
        ok = (np.array_equal(Yg, r["Y"]) and np.array_equal(Ag, r["A"]) and
              bool(np.all(np.abs(Sg - r["S"]) <= 1e-5 * np.maximum(1.0, np.abs(r["S"])))))
        parity = {"rows_checked": int(len(rows)), "ok": bool(ok)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": cfg.name, "nchan": cfg.nchan, "nsamp_out": cfg.nsamp_out, "ndm": cfg.ndm,
                       "widths": widths_of(cfg), "beams_per_gpu": 1,
                       "l2": "256 MiB memset between timed steps (outside each step's events); "
                             "working set %.0f MB > 126 MB L2" % ((hbm_bytes + info.integ_elems * 4.0) / 1e6),
                       "kcfg": {ddp.KERNEL_NAMES[k]: list(plan.get_kcfg(k).astuple())
                                for k in range(5) if _in_plan(plan, k)},
                       "tuned_from": os.path.basename(TUNED_JSON) if tuned else None},
            "dedisp_only": {"value": world * units_per_step / (dd_avg_ms * 1e-3), "unit": UNIT, "ms": dd_avg_ms},
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_tot_ms / args.steps,
                    "h2d_bytes_per_step": int(h_in.numel()),
                    "d2h_bytes_per_step": int(h_snr.numel() * 4 + h_arg.numel() * 4)},
            "gpu_launches": int(kernels_per_step * args.steps),
            "clocks": clocks, "roofline": roofline, "stages": stages, "cpu_baseline": cpu, "parity": parity,
            "tuning": tuning_report()}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


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
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target duration of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-seconds", type=float, default=100.0, help="--impl reference: target duration of the whole run")
    args = ap.parse_args()
    if args.steps < 1:
        raise SystemExit("--steps must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
