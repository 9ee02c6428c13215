"""Host logic of libddp through the C ABI (no GPU needed): exported symbols, plan geometry and
delay tables against the oracle, argument errors, kernel-configuration validity / repair /
enumeration, NVRTC compilation of the kernel template for sm_100a, and the loud failure of every
compute call on a machine without a CUDA device (no CPU fallback exists).
"""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import paper_1811_04165_b200 as ddp
from paper_1811_04165_b200 import binding
from synth import configs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

GENE_DOMAINS = ((16, 32, 64, 128, 256, 512, 1024), (1, 2, 4, 8, 16, 32), (1, 2, 4, 8, 16), (1, 2, 4, 8, 16),
                (1, 2, 4, 8, 16), (0, 1, 2, 3, 4), (1, 4, 8, 16))  # BASELINE.json configs[4] + merged staging 3, 4


def has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


# ----------------------------------------------------------------------------- the boundary
def test_library_exports_every_declared_symbol():
    text = open(os.path.join(ROOT, "include", "ddp.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(ddp_[a-z_0-9]+)\s*\(", text))
    declared -= {"ddp_fitness_fn"}
    assert declared, "no declarations parsed from include/ddp.h"
    assert declared == set(ddp.SYMBOLS), "binding.SYMBOLS and include/ddp.h disagree: %s" % (
        declared ^ set(ddp.SYMBOLS))
    L = ctypes.CDLL(binding.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(L, name), "libddp.so does not export %s" % name
    assert "sm_100a" in ddp.version()
    assert ddp.status_str(0) == "ok" and ddp.status_str(-7).startswith("CUDA")


def test_ctypes_mirrors_have_the_size_the_c_compiler_gives(tmp_path):
    """A layout mismatch between binding.py and include/ddp.h would corrupt every call: compile a
    probe against the header with gcc and compare sizeof() of every struct."""
    import subprocess
    names = {"ddp_kcfg": binding.Kcfg, "ddp_options": binding.Options, "ddp_plan_info": binding.PlanInfo,
             "ddp_tune_io": binding.TuneIo, "ddp_ga_params": binding.GaParams, "ddp_bf_params": binding.BfParams,
             "ddp_rand_params": binding.RandParams, "ddp_tune_result": binding.TuneResult}
    src = tmp_path / "probe.c"
    src.write_text('#include <stdio.h>\n#include "ddp.h"\nint main(void){%s return 0;}\n' % "".join(
        'printf("%s %%zu\\n", sizeof(%s));' % (n, n) for n in names))
    exe = tmp_path / "probe"
    subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    out = dict(line.split() for line in subprocess.check_output([str(exe)]).decode().splitlines())
    for n, t in names.items():
        assert int(out[n]) == ctypes.sizeof(t), n


# ----------------------------------------------------------------------------- plan vs oracle
@pytest.mark.parametrize("mk", [configs.tiny, configs.apertif_direct, configs.ska_mid])
def test_direct_plan_delays_equal_oracle_table(mk):
    cfg = mk()
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    i = plan.query()
    d = plan.get_delays(0)
    do = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    assert d.shape == do.shape and np.array_equal(d, do)  # DD.2: entry for entry
    assert i.max_delay == int(do.max())
    assert i.nsamp_in_required == cfg.nsamp_out + int(do.max())
    assert i.in_stride_min >= i.nsamp_in_required and i.in_stride_min % 16 == 0
    assert i.out_stride_min >= cfg.nsamp_out and i.out_stride_min % 4 == 0
    assert i.adds_dedisp == float(cfg.ndm) * cfg.nchan * cfg.nsamp_out
    assert (d[:, 0] == 0).all() and (d[0] == 0).all()  # DD.3: top channel, DM 0
    plan.destroy()


def test_known_geometry_of_the_configs():
    # SURVEY.md Appendix B (computed independently of both implementations)
    for mk, maxd in ((configs.tiny, 344), (configs.apertif_direct, 11589), (configs.ska_mid, 213777)):
        plan = ddp.plan_from_config(mk(), cache_dir=None)
        assert plan.query().max_delay == maxd
        plan.destroy()
    plan = ddp.plan_from_config(configs.apertif_direct(), cache_dir=None)
    i = plan.query()
    assert [i.plane_len[k] for k in range(i.nwidths)] == [24414, 12207, 6103, 3051, 1525, 762, 381, 190, 95]
    assert i.plane_offset[0] == -1 and i.plane_stride[0] == 0  # w = 1 aliases the dedispersed series
    offs = [i.plane_offset[k] for k in range(1, i.nwidths)]
    assert offs == sorted(offs) and offs[0] == 0
    for k in range(1, i.nwidths):
        assert i.plane_stride[k] >= i.plane_len[k]
        nxt = i.plane_offset[k + 1] if k + 1 < i.nwidths else i.integ_elems
        assert nxt - i.plane_offset[k] == i.plane_stride[k] * i.ndm  # planes tile d_integ without overlap
    plan.destroy()


def test_subband_plan_tables_equal_oracle_tables():
    cfg = configs.apertif_subband()
    sb = cfg.subband
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    i = plan.query()
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    d1o, d2o = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)
    assert np.array_equal(plan.get_delays(1), d1o)
    assert np.array_equal(plan.get_delays(2), d2o)
    assert (i.max_d1, i.max_d2) == (int(d1o.max()), int(d2o.max())) == (11413, 168)  # Appendix B
    assert i.nsamp_sub == cfg.nsamp_out + 168
    assert i.ndm == 2048 and i.subband == 1
    # SB.5: the subband plan needs no more input than config 1's direct plan
    pd = ddp.plan_from_config(configs.apertif_direct(), cache_dir=None)
    assert i.nsamp_in_required <= pd.query().nsamp_in_required
    expect = sb.n_coarse * cfg.nchan * float(i.nsamp_sub) + 2048.0 * sb.n_subbands * cfg.nsamp_out
    assert i.adds_dedisp == expect
    with pytest.raises(ddp.DdpError):
        plan.get_delays(0)
    pd.destroy()
    plan.destroy()


def test_subband_centre_reference_plan_tables_equal_oracle_tables():
    """SB.2 alternative: subband_ref = 1 computes the step-2 delays at the centre of every subband;
    (a lower frequency than its top channel, so the delays grow: max 172 instead of 168 samples at BJ:cfg2);
    step 1 is untouched; a direct plan ignores the option; an unknown value is refused."""
    cfg = configs.apertif_subband()
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    d1o, d2o = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F, ref="centre")
    plan = ddp.plan_from_config(cfg, cache_dir=None, subband_ref=1)
    i = plan.query()
    assert i.subband_ref == 1
    assert np.array_equal(plan.get_delays(1), d1o)
    assert np.array_equal(plan.get_delays(2), d2o)
    assert (i.max_d1, i.max_d2) == (int(d1o.max()), int(d2o.max()))
    assert i.max_d2 == 172 and i.nsamp_sub == cfg.nsamp_out + i.max_d2
    plan.destroy()
    top = ddp.plan_from_config(cfg, cache_dir=None)
    assert top.query().subband_ref == 0 and top.query().max_d2 == 168
    top.destroy()
    pd = ddp.plan_from_config(configs.tiny(), cache_dir=None, subband_ref=1)
    assert pd.query().subband_ref == 0
    pd.destroy()
    with pytest.raises(ddp.DdpError):
        ddp.plan_from_config(cfg, cache_dir=None, subband_ref=2)


def test_sixteen_bit_plan_host_side(tmp_path):
    """ddp_options.input_bits = 16 (P:90 INPUT_BITS): geometry, the uint32 intermediate, overflow
    proofs with 65535 per sample, validity (no merged staging) and offline compilation of the uint16 code shapes."""
    cfg = configs.scaled(configs.apertif_direct(), name="u16", nchan=64, nsamp_out=2300, ndm=41, widths=(1, 2, 4, 8))
    p8 = ddp.plan_from_config(cfg, cache_dir=None)
    p = ddp.plan_from_config(cfg, cache_dir=str(tmp_path), input_bits=16)
    i8, i = p8.query(), p.query()
    assert (i8.input_bits, i.input_bits) == (8, 16)
    assert i.in_stride_min == i8.in_stride_min and i.max_delay == i8.max_delay  # strides are in elements
    assert np.array_equal(p.get_delays(0), p8.get_delays(0))
    V = p.enumerate_kcfgs(ddp.K_DIRECT)
    assert {c.staging for c in V} == {0, 1, 2} and {c.staging for c in p8.enumerate_kcfgs(ddp.K_DIRECT)} >= {3, 4}
    assert p.check_kcfg(ddp.K_DIRECT, p.get_kcfg(ddp.K_DIRECT))
    assert not p.check_kcfg(ddp.K_DIRECT, ddp.Kcfg(64, 4, 16, 4, 8, 4, 16))      # merged staging: uint8 only
    assert not p.check_kcfg(ddp.K_DIRECT, ddp.Kcfg(64, 4, 16, 4, 8, 0, 1))       # vec_bytes >= 4 for uint16
    for c in (p.get_kcfg(ddp.K_DIRECT), ddp.Kcfg(32, 4, 8, 2, 4, 0, 16), ddp.Kcfg(64, 2, 4, 4, 8, 2, 8)):
        assert p.check_kcfg(ddp.K_DIRECT, c), c
        p.compile_kcfg(ddp.K_DIRECT, c)
    assert any(n.startswith("ddp_dedisp_u16_") for n in os.listdir(tmp_path))
    p.destroy()
    p8.destroy()
    sb = configs.scaled(configs.apertif_subband(), name="u16sb", nchan=96, nsamp_out=2500, ndm=30, widths=(1, 2, 4, 8),
                        subband=configs.SubbandPlan(n_subbands=8, n_coarse=6, coarse_first=0.0, coarse_step=8.0,
                                                    n_fine=5, fine_step=0.25))
    q = ddp.plan_from_config(sb, cache_dir=None, input_bits=16)
    assert q.query().sub_elem_bytes == 4 and ddp.plan_from_config(sb, cache_dir=None).query().sub_elem_bytes == 2
    q.compile_kcfg(ddp.K_SUB1, q.get_kcfg(ddp.K_SUB1))
    q.compile_kcfg(ddp.K_SUB2, q.get_kcfg(ddp.K_SUB2))
    q.destroy()
    # 65535 * 1536 channels: the second moments of the widest series would not fit 64 bits
    with pytest.raises(ddp.DdpError) as e:
        ddp.plan_from_config(configs.apertif_direct(), cache_dir=None, input_bits=16)
    assert e.value.status == binding.E_OVERFLOW
    with pytest.raises(ddp.DdpError):
        ddp.plan_from_config(cfg, cache_dir=None, input_bits=12)


def test_step1_diagonal_tiles_are_chosen_from_the_delay_tables(tmp_path):
    """Code flag bit 6 (DIAG) of the packed step-1 kernel: on at BJ:cfg2 (the window of 32 coarse trials shrinks from
    TT + 5616 to TT + ~236 samples, so 8 channels per chunk fit twice where 4 fitted once), off for the same band in
    ascending channel order (relative delays negative) and for direct loads; visible in the kernel's name."""
    import dataclasses
    cfg = configs.apertif_subband()
    p = ddp.plan_from_config(cfg, cache_dir=str(tmp_path))
    c = ddp.Kcfg(128, 4, 16, 8, 8, 2, 16)
    assert p.check_kcfg(ddp.K_SUB1, c)       # two buffers of 8 rows: invalid before (V6, test_validity_rules_named_cases)
    p.compile_kcfg(ddp.K_SUB1, c)
    p.compile_kcfg(ddp.K_SUB1, ddp.Kcfg(64, 4, 16, 2, 8, 0, 16))
    names = sorted(os.listdir(tmp_path))
    assert any(n.startswith("ddp_dedisp_u8_s16_d8_u8_g2_v16_t512_w66.") for n in names), names   # OUT16 | DIAG
    assert any(n.startswith("ddp_dedisp_u8_s16_d2_u8_g0_v16_t256_w2.") for n in names), names    # direct loads: OUT16 only
    p.destroy()
    asc = dataclasses.replace(cfg, f_hi_mhz=cfg.f_lo_mhz, f_lo_mhz=cfg.f_hi_mhz)
    q = ddp.plan_from_config(asc, cache_dir=str(tmp_path / "asc"))
    assert not q.check_kcfg(ddp.K_SUB1, c)   # without the diagonal layout the windows are 7.7 KB again
    c4 = ddp.Kcfg(128, 4, 16, 8, 4, 2, 16)
    q.compile_kcfg(ddp.K_SUB1, c4)
    assert any(n.startswith("ddp_dedisp_u8_s16_d8_u4_g2_v16_t512_w18.") for n in os.listdir(tmp_path / "asc"))  # OUT16 | SINGLE
    q.destroy()


def test_plan_create_rejects_bad_arguments():
    f = np.array([1500.0, 1400.0, 1300.0, 1200.0])
    ok = dict(chan_freq_mhz=f, t_samp_s=1e-3, dm_list=[0.0, 10.0], widths=[1, 2], nsamp_out=64, cache_dir=None)

    def status(**kw):
        a = dict(ok)
        a.update(kw)
        try:
            ddp.plan_create(a.pop("chan_freq_mhz"), a.pop("t_samp_s"), a.pop("dm_list"), a.pop("widths"),
                            a.pop("nsamp_out"), **a).destroy()
            return 0
        except ddp.DdpError as e:
            return e.status

    assert status() == 0
    assert status(t_samp_s=0.0) == binding.E_ARG
    assert status(t_samp_s=float("nan")) == binding.E_ARG
    assert status(chan_freq_mhz=np.array([1500.0, -1.0])) == binding.E_ARG
    assert status(chan_freq_mhz=np.array([1500.0, float("inf")])) == binding.E_ARG
    assert status(dm_list=[10.0, 0.0]) == binding.E_ARG            # not non-decreasing
    assert status(dm_list=[-1.0, 0.0]) == binding.E_ARG
    assert status(widths=[2, 1]) == binding.E_ARG                   # not strictly increasing
    assert status(widths=[0, 1]) == binding.E_ARG
    assert status(widths=[1, 3]) == binding.E_ARG                   # not a power of two (INT.3)
    assert status(widths=[1, 64]) == binding.E_ARG                  # floor(ns / w_max) < 2 (INT.2)
    assert status(widths=list(range(1, 18))) == binding.E_ARG       # > DDP_MAX_WIDTHS
    assert status(nsamp_out=0) == binding.E_ARG
    assert status(snr_ddof=2) == binding.E_ARG
    # SB.3: nchan % n_subbands
    assert status(dm_list=None, n_subbands=3, n_coarse=2, coarse_dm_step=8.0, n_fine=2,
                  fine_dm_step=1.0) == binding.E_SHAPE
    assert status(dm_list=None, n_subbands=2, n_coarse=2, coarse_dm_step=8.0, n_fine=2, fine_dm_step=1.0) == 0
    assert status(dm_list=[0.0, 1.0, 8.0, 9.5], n_subbands=2, n_coarse=2, coarse_dm_step=8.0, n_fine=2,
                  fine_dm_step=1.0) == binding.E_ARG               # DM list is not the coarse+fine grid
    # INT.5: 255 * nchan * w_max must stay below 2^32
    big = np.linspace(1500.0, 1200.0, 70000)
    assert status(chan_freq_mhz=big, widths=[1, 256], nsamp_out=1024) == binding.E_OVERFLOW


def test_unsorted_channel_order_is_accepted_and_reference_is_the_maximum():
    f = np.array([1300.0, 1500.0, 1200.0, 1400.0])
    plan = ddp.plan_create(f, 1e-3, [0.0, 10.0, 20.0], [1], 8, cache_dir=None)
    d = plan.get_delays(0)
    assert d.tolist() == [[0, 0, 0, 0], [6, 0, 10, 3], [12, 0, 21, 5]]  # tests/golden/worked_example.txt, permuted
    plan.destroy()


# ----------------------------------------------------------------------------- configurations
def all_plans():
    small_sub = configs.scaled(configs.apertif_subband(), name="small_sub", nchan=96, nsamp_out=1500, n_pulses=1,
                               subband=configs.SubbandPlan(8, 5, 0.0, 8.0, 6, 1.0))
    return [configs.tiny(), configs.apertif_direct(), configs.apertif_subband(), small_sub]


def kernels_of(plan):
    return [k for k in range(5) if _in_plan(plan, k)]


def _in_plan(plan, k):
    try:
        plan.get_kcfg(k)
        return True
    except ddp.DdpError:
        return False


@pytest.mark.parametrize("cfg", all_plans(), ids=lambda c: c.name)
def test_enumeration_is_exactly_the_valid_subset_of_the_raw_grid(cfg):
    """BF space == {raw tuples the validity predicate accepts}; defaults are members."""
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    rng = np.random.default_rng(7)
    for k in kernels_of(plan):
        V = plan.enumerate_kcfgs(k)
        keys = [c.astuple() for c in V]
        assert len(keys) == len(set(keys)) > 0
        assert plan.get_kcfg(k).astuple() in set(keys)
        for c in V[:: max(1, len(V) // 400)]:
            assert plan.check_kcfg(k, c)
            for g, dom in enumerate(GENE_DOMAINS):
                assert c.astuple()[g] in dom
        # seeded sample of the 105 000-point raw grid: accepted iff enumerated
        vset = set(keys)
        n_valid = 0
        for _ in range(3000):
            raw = tuple(int(dom[rng.integers(len(dom))]) for dom in GENE_DOMAINS)
            ok = plan.check_kcfg(k, ddp.Kcfg(*raw))
            assert ok == (raw in vset)
            n_valid += ok
        assert abs(n_valid / 3000.0 - len(keys) / 105000.0) < 0.03
    plan.destroy()


@pytest.mark.parametrize("cfg", all_plans(), ids=lambda c: c.name)
def test_repair_is_total_deterministic_idempotent_and_identity_on_valid(cfg):
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    rng = np.random.default_rng(11)
    for k in kernels_of(plan):
        for n in range(300):
            if n < 250:
                raw = tuple(int(dom[rng.integers(len(dom))]) for dom in GENE_DOMAINS)
            else:  # values outside the candidate arrays are snapped first
                raw = tuple(int(rng.integers(-5, 3000)) for _ in GENE_DOMAINS)
            c = ddp.Kcfg(*raw)
            r1 = plan.repair_kcfg(k, c)
            assert plan.check_kcfg(k, r1), "repair(%s) = %s is not valid" % (raw, r1)
            assert plan.repair_kcfg(k, c).astuple() == r1.astuple()
            assert plan.repair_kcfg(k, r1).astuple() == r1.astuple()
            if plan.check_kcfg(k, c):
                assert r1.astuple() == raw
    plan.destroy()


def test_repair_moves_to_a_nearest_valid_configuration():
    """Nearest in summed |index distance| over the candidate arrays."""
    plan = ddp.plan_from_config(configs.tiny(), cache_dir=None)
    k = ddp.K_DIRECT
    V = [c.astuple() for c in plan.enumerate_kcfgs(k)]

    def dist(a, b):
        return sum(abs(dom.index(x) - dom.index(y)) for dom, x, y in zip(GENE_DOMAINS, a, b))

    rng = np.random.default_rng(3)
    checked = 0
    while checked < 25:
        raw = tuple(int(dom[rng.integers(len(dom))]) for dom in GENE_DOMAINS)
        if plan.check_kcfg(k, ddp.Kcfg(*raw)):
            continue
        r = plan.repair_kcfg(k, ddp.Kcfg(*raw)).astuple()
        assert dist(raw, r) == min(dist(raw, v) for v in V)
        checked += 1
    plan.destroy()


def test_validity_rules_named_cases():
    plan = ddp.plan_from_config(configs.apertif_subband(), cache_dir=None)
    ok = ddp.Kcfg(64, 4, 16, 2, 8, 1, 16)
    assert plan.check_kcfg(ddp.K_SUB1, ok)
    bad = {
        "V1 too many threads": ddp.Kcfg(1024, 2, 16, 2, 8, 1, 16),
        "V1 too few threads": ddp.Kcfg(16, 1, 16, 2, 8, 0, 16),
        "V2 register budget": ddp.Kcfg(64, 4, 16, 16, 8, 1, 16),
        "V4 unroll 32 not a candidate": ddp.Kcfg(64, 4, 16, 2, 32, 1, 16),
        "V5 vec wider than the thread's samples": ddp.Kcfg(64, 4, 4, 2, 8, 0, 16),
        "V3 DM tile larger than the 64 coarse DMs": ddp.Kcfg(32, 32, 16, 4, 8, 0, 16),
    }
    for why, c in bad.items():
        assert not plan.check_kcfg(ddp.K_SUB1, c), why
    # V4: 48 channels per subband -> unroll 16 divides, and sub2 (32 subbands) accepts 16 too
    assert plan.check_kcfg(ddp.K_SUB1, ddp.Kcfg(64, 4, 16, 2, 16, 0, 16))
    # V6: the same shape staged is valid: 16 rows x shifted copies of a ~1.3 KB window (diagonal time tiles,
    # DESIGN.md 6.1c; ~2.5 KB and single-buffered without them)
    assert plan.check_kcfg(ddp.K_SUB1, ddp.Kcfg(64, 4, 16, 2, 16, 1, 16))
    # a 2048 x 32 tile: 2.3 KB windows with the diagonal layout, so 4 and 8 rows per chunk fit (without it the
    # windows are 7.7 KB and 8 rows do not fit even once: test_step1_diagonal_tiles_are_chosen_from_the_delay_tables);
    # 16 rows of a 4096-sample tile's 4.4 KB windows do not fit
    assert plan.check_kcfg(ddp.K_SUB1, ddp.Kcfg(128, 4, 16, 8, 4, 2, 16))
    assert plan.check_kcfg(ddp.K_SUB1, ddp.Kcfg(128, 4, 16, 8, 8, 2, 16))
    assert not plan.check_kcfg(ddp.K_SUB1, ddp.Kcfg(256, 2, 16, 16, 16, 2, 16))
    # uint32-input kernels need vec_bytes >= 4
    assert not plan.check_kcfg(ddp.K_SUB2, ddp.Kcfg(128, 2, 4, 4, 4, 0, 1))
    # the direct kernel is not part of a subband plan
    assert not plan.check_kcfg(ddp.K_DIRECT, ok)
    with pytest.raises(ddp.DdpError) as e:
        plan.set_kcfg(ddp.K_SUB1, bad["V2 register budget"])
    assert e.value.status == binding.E_CONFIG  # never silently repaired
    plan.destroy()


def test_integrate_time_tile_is_a_multiple_of_every_width():
    plan = ddp.plan_from_config(configs.apertif_direct(), cache_dir=None)
    for c in plan.enumerate_kcfgs(ddp.K_INTEGRATE)[::97]:
        assert (c.threads_t * c.samples_per_thread) % 256 == 0
    plan.destroy()


# ----------------------------------------------------------------------------- NVRTC (host only)
@pytest.mark.parametrize("k,genes", [
    (ddp.K_DIRECT, (64, 4, 8, 2, 4, 2, 8)),      # packed uint8 kernel, TMA staging (UBLKCP)
    (ddp.K_DIRECT, (32, 2, 2, 2, 2, 0, 1)),      # generic kernel, direct byte loads
    (ddp.K_INTEGRATE, (64, 2, 8, 2, 2, 1, 8)),
    (ddp.K_SNR, (128, 2, 2, 2, 1, 2, 8)),
])
def test_template_compiles_for_sm100a_without_a_gpu(tmp_path, k, genes):
    cfg = configs.scaled(configs.tiny(), name="nvrtc", widths=(1, 2, 4, 8))
    plan = ddp.plan_from_config(cfg, cache_dir=str(tmp_path))
    c = ddp.Kcfg(*genes)
    assert plan.check_kcfg(k, c)
    plan.compile_kcfg(k, c)
    cubins = [f for f in os.listdir(tmp_path) if f.endswith(".cubin")]
    assert len(cubins) == 1
    blob = open(os.path.join(tmp_path, cubins[0]), "rb").read()
    assert blob[:4] == b"\x7fELF" and len(blob) > 2000
    with pytest.raises(ddp.DdpError) as e:
        plan.compile_kcfg(k, ddp.Kcfg(64, 4, 8, 2, 3, 2, 8))
    assert e.value.status == binding.E_CONFIG
    plan.destroy()


def test_257_channels_per_subband_compiles_staged_step_one(tmp_path):
    """cps = 257: the uint16 intermediate is still exact (257 * 255 = 65535) and the packed kernel must not
    ask for the wide flush at the same time (the template static_asserts against that combination)."""
    f = 1550.0 - 0.1 * np.arange(514)
    plan = ddp.plan_create(f, 40.96e-6, None, [1, 2], 1000, n_subbands=2, n_coarse=3, coarse_dm_step=8.0,
                           n_fine=4, fine_dm_step=0.25, cache_dir=str(tmp_path))
    assert plan.query().sub_elem_bytes == 2
    c = plan.get_kcfg(ddp.K_SUB1)
    assert c.staging != 0
    plan.compile_kcfg(ddp.K_SUB1, c)
    plan.compile_kcfg(ddp.K_SUB1, ddp.Kcfg(64, 2, 16, 2, 1, 2, 16))
    plan.destroy()
    # 258 channels per subband: uint32 intermediate, wide flush
    plan = ddp.plan_create(1550.0 - 0.1 * np.arange(516), 40.96e-6, None, [1, 2], 1000, n_subbands=2, n_coarse=3,
                           coarse_dm_step=8.0, n_fine=4, fine_dm_step=0.25, cache_dir=str(tmp_path))
    assert plan.query().sub_elem_bytes == 4
    plan.compile_kcfg(ddp.K_SUB1, plan.get_kcfg(ddp.K_SUB1))
    plan.destroy()


# ----------------------------------------------------------------------------- no fallback
@pytest.mark.skipif(has_gpu(), reason="checks the behaviour of a machine WITHOUT a CUDA device")
def test_compute_calls_fail_loudly_without_a_device():
    cfg = configs.scaled(configs.tiny(), name="nogpu", ndm=4, nsamp_out=256, widths=(1, 2))
    plan = ddp.plan_from_config(cfg, cache_dir=None)
    i = plan.query()
    X = np.zeros((i.nchan, i.in_stride_min), dtype=np.uint8)
    Y = np.zeros((i.ndm, i.out_stride_min), dtype=np.uint32)
    L = ddp.lib()
    h = plan._h
    assert L.ddp_dedisperse(h, X.ctypes.data, X.shape[1], Y.ctypes.data, Y.shape[1], None) == binding.E_CUDA
    assert L.ddp_integrate(h, Y.ctypes.data, Y.shape[1], Y.ctypes.data, None) == binding.E_CUDA
    assert L.ddp_plan_bind_workspace(h, X.ctypes.data & ~255, 1 << 30, None) == binding.E_CUDA
    io = ddp.make_tune_io()  # no fitness callback -> hardware harness -> must refuse
    with pytest.raises(ddp.DdpError) as e:
        plan.tune_random(io, seed=1, max_evals=4)
    assert e.value.status == binding.E_CUDA
    assert b"libcuda" in L.ddp_last_error(h) or b"CUDA" in L.ddp_last_error(h)
    with pytest.raises(RuntimeError):
        ddp.alloc_buffers(plan)
    plan.destroy()


def test_sliding_mode_and_channel_mask_plans_host_side():
    """integration_mode = SLIDING and chan_mask as far as the host sees them: geometry, which
    kernels belong to the plan, validity of the fused kernel's shapes, algorithmic work of a masked plan."""
    from synth import configs
    cfg = configs.tiny()
    plan = ddp.plan_from_config(cfg, integration_mode=1)
    i = plan.query()
    assert i.integration_mode == 1 and i.integ_elems == 0
    assert [i.plane_len[k] for k in range(i.nwidths)] == [cfg.nsamp_out - w + 1 for w in cfg.widths]
    for k in (ddp.K_INTEGRATE, ddp.K_SNR):                      # the sums are never materialised in this mode
        with pytest.raises(ddp.DdpError):
            plan.get_kcfg(k)
    V = plan.enumerate_kcfgs(ddp.K_ISNR)
    assert V and all(c.threads_t == 32 and c.staging == 0 and c.unroll == 1 for c in V)
    plan.compile_kcfg(ddp.K_ISNR, V[0])                         # NVRTC, no GPU needed
    with pytest.raises(ddp.DdpError):
        ddp.plan_from_config(cfg, integration_mode=2)
    plan.destroy()
    mask = np.ones(cfg.nchan, np.uint8)
    mask[::4] = 0
    pm = ddp.plan_from_config(cfg, chan_mask=mask)
    im, i0 = pm.query(), ddp.plan_from_config(cfg).query()
    assert im.nchan_masked == cfg.nchan // 4
    assert im.adds_dedisp == pytest.approx(i0.adds_dedisp * 0.75)
    assert im.workspace_bytes > i0.workspace_bytes              # row map + zero row
    assert np.array_equal(pm.get_delays(0), ddp.plan_from_config(cfg).get_delays(0))  # the tables do not change
    with pytest.raises(ValueError):
        ddp.plan_from_config(cfg, chan_mask=np.ones(3, np.uint8))
    pm.destroy()
