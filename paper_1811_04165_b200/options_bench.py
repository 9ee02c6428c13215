"""Timings of the optional paths of SURVEY 8(f) on this GPU, beside the headline workload they derive from.

    python -m paper_1811_04165_b200.options_bench [--reps 20] [--sweep 48] [--out gpurun_out/options_bench.json]

bench.py measures the paths BASELINE.json names (uint8 input, decimating integration, no mask, subband reference =
top channel).  This script times, with the same method (CUDA events on the launch stream, >= 3 warm-up passes,
a 256 MiB memset between timed passes so that nothing is read from L2), the options the library adds to them:

  u16     ddp_options.input_bits = 16 on the geometry of BASELINE.json configs[1] (1536 channels, 2048 trials,
          24 414 samples; widths 1..32 and sliding integration, the only way the overflow proofs admit 65535 x 1536):
          the uint16 code shapes of the direct kernel, best of a strided sample of the valid staged shapes;
  slide   integration_mode = SLIDING: the stride-1 boxcar + S/N kernel on configs[1]'s 2048 x 24 414 result;
  mask    chan_mask with every tenth channel zapped on configs[1], tuned direct shape;
  centre  subband_ref = CENTRE on configs[2], tuned step-1 / step-2 shapes.

Parity of every one of these paths is the business of tests/test_gpu_parity.py (this module never sees the oracle).
Numbers are context for DESIGN.md section 6; the roofline fraction is against the same add peak bench.py uses
(192 int32 adds per clock per SM x SMs x the maximum SM clock, profiles/r02_ubench.md).
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys

ADD_PEAK_PER_CLK_PER_SM = 192.0
HERE = os.path.dirname(os.path.abspath(__file__))


def max_sm_mhz(index: int) -> float:
    import pynvml
    pynvml.nvmlInit()
    h = pynvml.nvmlDeviceGetHandleByIndex(index)
    return float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--sweep", type=int, default=48, help="shapes sampled for the 16-bit direct kernel")
    ap.add_argument("--out", default="gpurun_out/options_bench.json")
    ap.add_argument("--cases", nargs="+", default=["u8", "u16", "slide", "mask", "centre"])
    args = ap.parse_args(argv)

    import numpy as np
    import torch
    import paper_1811_04165_b200 as ddp
    from synth import configs, filterbank

    if not torch.cuda.is_available():
        raise SystemExit("options_bench: no CUDA device -- there is no CPU fallback")
    dev = torch.device("cuda:0")
    props = torch.cuda.get_device_properties(0)
    peak_tadd = ADD_PEAK_PER_CLK_PER_SM * props.multi_processor_count * max_sm_mhz(0) * 1e6 / 1e12
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    with open(os.path.join(HERE, "tuned_b200.json")) as fh:
        tuned = json.load(fh)

    def timed(fn, reps):
        for _ in range(3):
            fn()
        ms = []
        for _ in range(reps):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            b.synchronize()
            ms.append(a.elapsed_time(b))
        ms.sort()
        return ms[len(ms) // 2]

    def setup(cfg, bits=8, **kw):
        plan = ddp.plan_from_config(cfg, input_bits=bits, **kw)
        info = plan.query()
        buf = ddp.alloc_buffers(plan, dev)
        X, _ = filterbank.make_filterbank(cfg, int(info.nsamp_in_required), int(info.in_stride_min), bits=bits)
        buf["d_in"].copy_(torch.from_numpy(X if bits == 8 else X.view(np.int16)))
        torch.cuda.synchronize()
        return plan, info, buf

    def apply(plan, workload, kernels):
        for kname in kernels:
            plan.set_kcfg(ddp.KERNEL_NAMES.index(kname), ddp.Kcfg(*tuned[workload][kname]))

    def record(name, ms, info, extra):
        r = {"ms": ms, "adds": info.adds_dedisp, "tadd_per_s": info.adds_dedisp / (ms * 1e-3) / 1e12,
             "frac_of_add_peak": info.adds_dedisp / (ms * 1e-3) / 1e12 / peak_tadd}
        r.update(extra)
        report["cases"][name] = r
        print(name, json.dumps(r), flush=True)

    report = {"gpu": props.name, "sms": props.multi_processor_count, "add_peak_tadd_per_s": peak_tadd,
              "reps": args.reps, "method": "CUDA events, median, 256 MiB memset between passes", "cases": {}}
    cfg1, cfg2 = configs.apertif_direct(), configs.apertif_subband()

    if "u8" in args.cases:  # the reference point: what bench.py times
        plan, info, buf = setup(cfg1)
        apply(plan, "cfg1", ["direct"])
        ms = timed(lambda: plan.dedisperse(buf["d_in"], buf["d_out"]), args.reps)
        record("cfg1_uint8_dedisperse", ms, info, {"kcfg": tuned["cfg1"]["direct"]})
        plan.destroy()
        del buf

    if "u16" in args.cases:
        c16 = dataclasses.replace(cfg1, name="cfg1_geometry_uint16", widths=(1, 2, 4, 8, 16, 32))
        plan, info, buf = setup(c16, bits=16, integration_mode=1)
        V = [c for c in plan.enumerate_kcfgs(ddp.K_DIRECT) if c.staging != 0 and c.threads_t * c.threads_dm >= 128
             and c.samples_per_thread * c.dms_per_thread >= 32]
        picks = [V[i] for i in sorted(set(np.linspace(0, len(V) - 1, args.sweep).astype(int).tolist()))]
        picks.append(plan.get_kcfg(ddp.K_DIRECT))
        best = (float("inf"), None)
        for c in picks:
            plan.set_kcfg(ddp.K_DIRECT, c)
            try:
                ms = timed(lambda: plan.dedisperse(buf["d_in"], buf["d_out"]), 3)
            except ddp.DdpError:
                continue
            if ms < best[0]:
                best = (ms, c)
        plan.set_kcfg(ddp.K_DIRECT, best[1])
        ms = timed(lambda: plan.dedisperse(buf["d_in"], buf["d_out"]), args.reps)
        ms_isnr = timed(lambda: plan.integrate_snr(buf["d_out"], buf["d_snr"], buf["d_argmax"]), args.reps)
        record("cfg1_geometry_uint16_dedisperse", ms, info,
               {"kcfg": list(best[1].astuple()), "shapes_tried": len(picks), "valid_staged_shapes": len(V),
                "input_bytes": int(info.nchan * info.nsamp_in_required * 2), "sliding_integrate_snr_ms": ms_isnr})
        plan.destroy()
        del buf

    if "slide" in args.cases:
        plan, info, buf = setup(cfg1, integration_mode=1)
        apply(plan, "cfg1", ["direct"])
        plan.dedisperse(buf["d_in"], buf["d_out"])
        ms = timed(lambda: plan.integrate_snr(buf["d_out"], buf["d_snr"], buf["d_argmax"]), args.reps)
        nbytes = float(info.ndm) * info.nsamp_out * 4
        report["cases"]["cfg1_sliding_integrate_snr"] = {
            "ms": ms, "widths": [info.widths[k] for k in range(info.nwidths)], "algorithmic_bytes": nbytes,
            "gb_per_s": nbytes / (ms * 1e-3) / 1e9,
            "window_sums_per_s": sum(info.plane_len[k] for k in range(info.nwidths)) * float(info.ndm) / (ms * 1e-3)}
        print("cfg1_sliding_integrate_snr", json.dumps(report["cases"]["cfg1_sliding_integrate_snr"]), flush=True)
        plan.destroy()
        del buf

    if "mask" in args.cases:
        mask = np.ones(cfg1.nchan, np.uint8)
        mask[::10] = 0
        plan, info, buf = setup(cfg1, chan_mask=mask)
        apply(plan, "cfg1", ["direct"])
        ms = timed(lambda: plan.dedisperse(buf["d_in"], buf["d_out"]), args.reps)
        record("cfg1_masked_dedisperse", ms, info, {"kcfg": tuned["cfg1"]["direct"], "channels_masked": int(info.nchan_masked)})
        plan.destroy()
        del buf

    if "centre" in args.cases:
        for ref, name in ((0, "cfg2_top_reference_dedisperse"), (1, "cfg2_centre_reference_dedisperse")):
            plan, info, buf = setup(cfg2, subband_ref=ref)
            apply(plan, "cfg2", ["sub1", "sub2"])
            ms = timed(lambda: plan.dedisperse(buf["d_in"], buf["d_out"]), args.reps)
            record(name, ms, info, {"max_d2": int(info.max_d2)})
            plan.destroy()
            del buf

    os.makedirs(os.path.dirname(os.path.abspath(args.out)), exist_ok=True)
    with open(args.out, "w") as fh:
        json.dump(report, fh, indent=1)
    return 0


if __name__ == "__main__":
    sys.exit(main())
