"""Parity of the CUDA path (through the C ABI) against the oracle, element by element.

Bar (BASELINE.json north_star): dedispersion and integration bit-exact (uint8 in, uint32
accumulate), S/N within 1e-5 relative, argmax exact.  Small cases span several tiles and ragged
tails; full-size configs are checked on sampled DM rows the oracle computes one by one.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():  # collected on the CPU box, run on the B200 box
    pytest.skip("no CUDA device", allow_module_level=True)

import paper_1811_04165_b200 as ddp  # noqa: E402
from synth import configs  # noqa: E402
from synth.configs import SubbandPlan  # noqa: E402

from gpu_common import (GpuSearch, assert_snr_close, compare_all, oracle_direct_all_rows_mt,  # noqa: E402
                        oracle_direct_rows, oracle_search, oracle_subband, oracle_subband_mt, tuned_shapes, u32)


def small_direct(**kw):
    base = dict(name="small_direct", nchan=80, nsamp_out=3001, ndm=37, widths=(1, 2, 4, 8, 16), n_pulses=3)
    base.update(kw)
    return configs.scaled(configs.apertif_direct(), **base)


def small_subband(**kw):
    base = dict(name="small_subband", nchan=96, nsamp_out=2500, ndm=30, widths=(1, 2, 4, 8), n_pulses=2,
                subband=SubbandPlan(n_subbands=8, n_coarse=6, coarse_first=0.0, coarse_step=8.0, n_fine=5,
                                    fine_step=0.25))
    base.update(kw)
    return configs.scaled(configs.apertif_direct(), **base)


# ---------------------------------------------------------------------------------- whole pipeline
def test_cfg0_full_pipeline_and_pulse_recovery():
    cfg = configs.tiny()
    g = GpuSearch(cfg)
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="cfg0")
    S = g.buf["d_snr"].cpu().numpy()
    i, k = np.unravel_index(np.argmax(S), S.shape)
    assert cfg.dm_list()[i] == 17.0 and cfg.widths[k] == 4  # BJ:cfg0 pulse: DM 17, width 4
    A = u32(g.buf["d_argmax"])
    assert A[i, k] * 4 == 2000                               # t0 = 2000
    g.close()


def test_small_direct_ragged():
    cfg = small_direct()
    g = GpuSearch(cfg)
    g.run_all()
    compare_all(g, oracle_direct_rows(cfg, g.X), what="small_direct")
    g.close()


def test_small_subband_ragged_and_intermediate():
    cfg = small_subband()
    g = GpuSearch(cfg)
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    Sg = g.subband_intermediate()
    assert np.array_equal(Sg, So), "subband intermediate S differs"
    compare_all(g, Yo, what="small_subband")
    # SB.6: rows with zero fine offset equal the direct result at the coarse DM
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    import oracle
    Yd = oracle.dedisperse(g.X, oracle.delay_table(cfg.chan_freq_mhz(), A, cfg.t_samp_s), cfg.nsamp_out)
    Yg = u32(g.buf["d_out"])[:: sb.n_fine, : cfg.nsamp_out]
    assert np.array_equal(Yg, Yd)
    g.close()


# ---------------------------------------------------------------------------------- edge cases
def test_single_dm_zero_is_channel_sum():
    cfg = small_direct(name="dm0", ndm=1, nsamp_out=1000, widths=(1, 2), n_pulses=0)
    g = GpuSearch(cfg)
    Y = g.dedisperse()
    assert np.array_equal(Y[0], g.X[:, :1000].astype(np.uint32).sum(axis=0))  # BJ: DM=0 == plain channel sum
    g.close()


def test_width_one_only_and_tiny_series():
    cfg = small_direct(name="w1", ndm=3, nsamp_out=5, widths=(1,), nchan=16, n_pulses=0)
    g = GpuSearch(cfg)
    g.run_all()
    compare_all(g, oracle_direct_rows(cfg, g.X), what="w1")
    g.close()


def test_saturated_input_maximum_values():
    # all samples 255: the largest sums the accumulators can see for this shape (INT.5)
    cfg = small_direct(name="sat", nchan=64, ndm=9, nsamp_out=2048, widths=(1, 2, 4, 8, 16, 32, 64, 128, 256), n_pulses=0)
    probe = GpuSearch(cfg)
    X = np.full_like(probe.X, 255)
    probe.close()
    g = GpuSearch(cfg, X=X)
    Y, P, S, A = g.run_all()
    assert (Y == 255 * 64).all()
    assert (P[256] == 255 * 64 * 256).all()
    assert (S == 0).all() and (A == 0).all()  # SNR.3: constant series -> 0, argmax 0
    g.close()


def test_error_behaviour():
    cfg = small_direct(name="err", ndm=4, nsamp_out=512, widths=(1, 2), n_pulses=0)
    plan = ddp.plan_from_config(cfg)
    b = ddp.alloc_buffers(plan, bind=False)
    with pytest.raises(ddp.DdpError) as e:
        plan.dedisperse(b["d_in"], b["d_out"])
    assert e.value.status == ddp.binding.E_WORKSPACE
    plan.bind_workspace(b["workspace"])
    with pytest.raises(ddp.DdpError) as e:
        plan.dedisperse(b["d_in"], b["d_out"], in_stride=16)
    assert e.value.status == ddp.binding.E_SHAPE
    bad = ddp.Kcfg(64, 4, 8, 4, 7, 0, 4)
    with pytest.raises(ddp.DdpError) as e:
        plan.set_kcfg(ddp.K_DIRECT, bad)
    assert e.value.status == ddp.binding.E_CONFIG
    plan.destroy()


# ---------------------------------------------------------------------------------- API corners
def test_snr_ddof_one_matches_the_oracle():
    """SNR.2: snr_ddof = 1 (sample standard deviation) against oracle.snr(ddof=1); short series so that
    the two readings differ by far more than the tolerance (0.5 % at n = 95)."""
    cfg = small_direct(name="ddof1", nchan=48, nsamp_out=1530, ndm=21, widths=(1, 2, 4, 8, 16), n_pulses=2)
    g = GpuSearch(cfg, snr_ddof=1)
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="ddof=1", ddof=1)
    _, S0, _ = oracle_search(Yo, list(cfg.widths), 0)
    S1 = g.buf["d_snr"].cpu().numpy()
    assert np.all(np.abs(S1 - S0) > 1e-5 * np.abs(S0)), "ddof=1 result is indistinguishable from ddof=0"
    g.close()


@pytest.mark.parametrize("subband", [False, True])
def test_search_host_end_to_end_call(subband):
    """ddp_search_host (host buffers in, S/N + argmax out) against the oracle: cfg0 and a small subband plan."""
    cfg = small_subband() if subband else configs.tiny()
    g = GpuSearch(cfg)
    i = g.info
    g.buf["d_in"].zero_()                                   # the call must upload the filterbank itself
    h_in = torch.from_numpy(g.X).pin_memory()
    h_snr = torch.full((i.ndm, i.nwidths), -3.0, dtype=torch.float32).pin_memory()
    h_arg = torch.full((i.ndm, i.nwidths), -1, dtype=torch.int32).pin_memory()
    g.plan.search_host(h_in, g.buf["d_in"], g.buf["d_out"], g.buf["d_integ"], g.buf["d_snr"], g.buf["d_argmax"],
                       h_snr, h_arg)                        # synchronises before returning
    Yo = oracle_subband(cfg, g.X)[1] if subband else oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="search_host device side")
    _, So, Ao = oracle_search(Yo, list(cfg.widths), 0)
    assert_snr_close(h_snr.numpy(), So, "search_host host S/N")
    assert np.array_equal(h_arg.numpy().view(np.uint32), Ao)
    # pageable host memory and no argmax request
    h_snr2 = np.full((i.ndm, i.nwidths), -3.0, dtype=np.float32)
    g.plan.search_host(g.X, g.buf["d_in"], g.buf["d_out"], g.buf["d_integ"], g.buf["d_snr"], None, h_snr2, None)
    assert_snr_close(h_snr2, So, "search_host pageable, no argmax")
    # no plane buffer: dedisperse -> fused integrate + S/N (ddp_integrate_snr), same table
    h_snr3 = np.full((i.ndm, i.nwidths), -3.0, dtype=np.float32)
    h_arg3 = np.full((i.ndm, i.nwidths), -1, dtype=np.int32)
    g.plan.search_host(g.X, g.buf["d_in"], g.buf["d_out"], None, g.buf["d_snr"], g.buf["d_argmax"], h_snr3, h_arg3)
    assert_snr_close(h_snr3, So, "search_host without planes")
    assert np.array_equal(h_arg3.view(np.uint32), Ao)
    g.close()


@pytest.mark.parametrize("subband", [False, True])
def test_search_host_batches_equal_one_long_dedispersion(subband):
    """ddp_search_host_batches (8(f) f3): three consecutive batches, only the new samples uploaded, the
    shared max_delay samples carried on the device, uploads overlapped on a second stream -- every batch's S/N table
    equals the oracle's search of the matching columns of ONE long dedispersion of the whole observation."""
    import oracle
    from synth import filterbank
    cfg = small_subband(nsamp_out=1900) if subband else small_direct(name="batches", nchan=40, nsamp_out=2304, ndm=19)
    g = GpuSearch(cfg)
    i = g.info
    nb, ns, md = 3, cfg.nsamp_out, i.max_delay
    nlong = nb * ns + md
    X, _ = filterbank.make_filterbank(cfg, nlong, (nlong + 47) // 16 * 16)
    if subband:
        sb = cfg.subband
        A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
        F = sb.fine_step * np.arange(sb.n_fine)
        d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)
        S = oracle.subband_step1(X, d1, sb.n_subbands, nb * ns + int(d2.max()))
        Ylong = oracle.subband_step2(S, d2, nb * ns)
    else:
        Ylong = oracle.dedisperse(X, oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s), nb * ns)
    d_in1 = torch.empty_like(g.buf["d_in"])
    g.buf["d_in"].zero_()
    d_in1.zero_()
    h_in = torch.from_numpy(X).pin_memory()
    h_snr = torch.full((nb, i.ndm, i.nwidths), -3.0, dtype=torch.float32).pin_memory()
    h_arg = torch.full((nb, i.ndm, i.nwidths), -1, dtype=torch.int32).pin_memory()
    for rep in range(2):  # the second call reuses the plan's copy stream and events
        g.plan.search_host_batches(h_in, nb, g.buf["d_in"], d_in1, g.buf["d_out"], g.buf["d_snr"], g.buf["d_argmax"],
                                   h_snr, h_arg)
        for b in range(nb):
            _, So, Ao = oracle_search(np.ascontiguousarray(Ylong[:, b * ns: (b + 1) * ns]), list(cfg.widths), 0)
            assert_snr_close(h_snr[b].numpy(), So, "batch %d" % b)
            assert np.array_equal(h_arg[b].numpy().view(np.uint32), Ao), "argmax of batch %d" % b
        h_snr.fill_(-3.0)
    # the last batch's dedispersed rows are still on the device
    assert np.array_equal(u32(g.buf["d_out"])[:, :ns], Ylong[:, (nb - 1) * ns:])
    g.close()


def test_snr_without_argmax_wider_strides_and_a_side_stream():
    """d_argmax = NULL; in/out strides larger than the minimum; a caller stream other than the current one."""
    cfg = small_direct(name="strides", nchan=72, nsamp_out=2777, ndm=23, widths=(1, 2, 4, 8), n_pulses=2)
    g = GpuSearch(cfg)
    i = g.info
    Yo = oracle_direct_rows(cfg, g.X)
    _, So, Ao = oracle_search(Yo, list(cfg.widths), 0)
    in_stride, out_stride = int(i.in_stride_min) + 48, int(i.out_stride_min) + 12
    d_in = torch.full((i.nchan, in_stride), 255, dtype=torch.uint8, device="cuda")
    d_in[:, : i.in_stride_min].copy_(torch.from_numpy(g.X))
    d_out = torch.full((i.ndm, out_stride), -1, dtype=torch.int32, device="cuda")
    d_snr = torch.full((i.ndm, i.nwidths), -7.0, dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        pass
    g.plan.dedisperse(d_in, d_out, stream=side)
    g.plan.integrate(d_out, g.buf["d_integ"], stream=side)
    g.plan.snr(d_out, g.buf["d_integ"], d_snr, None, stream=side)
    side.synchronize()
    Yg = u32(d_out)
    assert np.array_equal(Yg[:, : cfg.nsamp_out], Yo)
    assert (Yg[:, i.out_stride_min:] == 0xFFFFFFFF).all(), "columns beyond out_stride_min were written"
    assert_snr_close(d_snr.cpu().numpy(), So, "wide strides / side stream / no argmax")
    # the same through the default-stream path with argmax, for the argmax comparison
    g.plan.snr(d_out, g.buf["d_integ"], d_snr, g.buf["d_argmax"])
    torch.cuda.synchronize()
    assert np.array_equal(u32(g.buf["d_argmax"]), Ao)
    g.close()


def test_subband_257_channels_per_subband_runs_staged_with_the_uint16_intermediate():
    """cps = 257 is the largest subband the uint16 intermediate holds exactly (257 * 255 = 65535): the packed
    kernel must run it without the wide flush (WIDE and OUT16 used to be set together)."""
    cfg = small_subband(name="cps257", nchan=514, nsamp_out=1200, ndm=3 * 4,
                        subband=SubbandPlan(n_subbands=2, n_coarse=3, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=4, fine_step=0.25))
    g = GpuSearch(cfg)
    assert g.info.sub_elem_bytes == 2
    g.X[:] = 255
    g.upload()
    c = g.plan.get_kcfg(ddp.K_SUB1)
    assert c.staging != 0
    Y = g.dedisperse()
    assert np.all(g.subband_intermediate() == 255 * 257)
    assert np.all(Y == 255 * 514)
    g.close()
    g = GpuSearch(cfg)
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="cps257")
    g.close()



# ---------------------------------------------------------------------------------- configuration sweep
def _sample(cfgs, n, seed):
    """n configurations: evenly strided over the canonical enumeration plus seeded random picks, so
    that every staging mode and vector width appears."""
    rng = np.random.default_rng(seed)
    idx = set(np.linspace(0, len(cfgs) - 1, n // 2).astype(int).tolist())
    idx |= set(rng.integers(0, len(cfgs), n - len(idx)).tolist())
    return [cfgs[i] for i in sorted(idx)]


@pytest.mark.parametrize("kernel", [ddp.K_DIRECT, ddp.K_INTEGRATE, ddp.K_SNR])
def test_direct_plan_kernel_configuration_sweep(kernel):
    cfg = small_direct(name="sweep", nchan=64, nsamp_out=2300, ndm=41, widths=(1, 2, 4, 8, 16, 32))
    g = GpuSearch(cfg)
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="sweep default")
    seen = set()
    for c in _sample(g.plan.enumerate_kcfgs(kernel), 48, seed=kernel):
        g.plan.set_kcfg(kernel, c)
        seen.add((c.staging, c.vec_bytes))
        if kernel == ddp.K_DIRECT:
            g.buf["d_out"].fill_(-1)
            g.dedisperse()
        elif kernel == ddp.K_INTEGRATE:
            g.buf["d_integ"].fill_(-1)
            g.integrate()
        g.buf["d_snr"].fill_(-7.0)
        g.buf["d_argmax"].fill_(-1)
        if kernel != ddp.K_SNR:
            g.integrate()
        g.snr()
        compare_all(g, Yo, what="%s %r" % (ddp.KERNEL_NAMES[kernel], c))
    assert {s for s, _ in seen} >= {0, 1, 2}
    g.close()


def test_integrate_and_snr_sparse_wide_widths_sweep():
    """Widths with gaps and boxcars wider than one warp's samples (cross-warp level of the tree),
    ragged length, every block shape family: integrate and snr against the oracle."""
    cfg = small_direct(name="wide", nchan=32, nsamp_out=5203, ndm=19, widths=(1, 2, 8, 64, 512, 1024), n_pulses=2)
    g = GpuSearch(cfg)
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="wide default")
    for kernel in (ddp.K_INTEGRATE, ddp.K_SNR):
        V = g.plan.enumerate_kcfgs(kernel)
        picks = _sample(V, 40, seed=77 + kernel)
        if kernel == ddp.K_INTEGRATE:  # make sure 16-lane rows and the widest blocks are in
            picks += [c for c in V if c.threads_t == 16 and c.staging == 0][:3]
            picks += [c for c in V if c.threads_t == 1024 and c.samples_per_thread == 1][:3]
        for c in picks:
            g.plan.set_kcfg(kernel, c)
            g.buf["d_integ"].fill_(-1)
            g.buf["d_snr"].fill_(-7.0)
            g.buf["d_argmax"].fill_(-1)
            g.integrate()
            g.snr()
            compare_all(g, Yo, what="%s %r" % (ddp.KERNEL_NAMES[kernel], c))
    g.close()


# ---------------------------------------------------------------------------------- fused integration + S/N (8(f) f1)
@pytest.mark.parametrize("widths,ns,ddof", [((1, 2, 4, 8, 16, 32, 64, 128, 256), 4099, 0),
                                            ((1, 2, 8, 64, 512, 1024, 2048), 9217, 0),
                                            ((2, 16, 4096), 12290, 1),
                                            ((1,), 700, 0)])
def test_fused_integrate_snr_equals_oracle(widths, ns, ddof):
    """ddp_integrate_snr (one pass over Y) against the oracle's integrate + snr: S/N within 1e-5, argmax exact, for
    every valid kernel shape (all block-sum levels: in-thread, across lanes, across chunks), ragged lengths, sparse
    width sets, both ddof; with a plane buffer the planes are bit-exact too, without one nothing is written."""
    cfg = small_direct(name="fused%d" % ns, nchan=24, nsamp_out=ns, ndm=21, widths=widths, n_pulses=2)
    g = GpuSearch(cfg, snr_ddof=ddof)
    Yg = g.dedisperse()
    Yo = oracle_direct_rows(cfg, g.X)
    assert np.array_equal(Yg, Yo)
    Po, So, Ao = oracle_search(Yo, list(widths), ddof)
    V = g.plan.enumerate_kcfgs(ddp.K_ISNR)
    assert len(V) >= 10
    for c in V:
        g.plan.set_kcfg(ddp.K_ISNR, c)
        g.buf["d_integ"].fill_(-1)
        g.buf["d_snr"].fill_(-7.0)
        g.buf["d_argmax"].fill_(-1)
        g.plan.integrate_snr(g.buf["d_out"], g.buf["d_snr"], g.buf["d_argmax"])  # no planes
        g.torch.cuda.synchronize()
        assert_snr_close(g.buf["d_snr"].cpu().numpy(), So, "fused %r" % c)
        assert np.array_equal(u32(g.buf["d_argmax"]), Ao), "fused argmax differs for %r" % c
        assert bool((g.buf["d_integ"] == -1).all()), "fused kernel wrote planes it was not given"
    for c in (V[0], V[len(V) // 2], V[-1]):
        g.plan.set_kcfg(ddp.K_ISNR, c)
        g.buf["d_snr"].fill_(-7.0)
        g.plan.integrate_snr(g.buf["d_out"], g.buf["d_snr"], None, d_integ=g.buf["d_integ"])  # planes, no argmax
        g.torch.cuda.synchronize()
        assert_snr_close(g.buf["d_snr"].cpu().numpy(), So, "fused with planes %r" % c)
        Pg = g.planes()
        for w in widths:
            if w > 1:
                assert np.array_equal(Pg[w], Po[w]), "fused plane w=%d differs for %r" % (w, c)
    # the separate kernels give the same bits
    g.integrate()
    S2, A2 = g.snr()
    g.plan.integrate_snr(g.buf["d_out"], g.buf["d_snr"], g.buf["d_argmax"])
    g.torch.cuda.synchronize()
    assert np.array_equal(g.buf["d_snr"].cpu().numpy(), S2) and np.array_equal(u32(g.buf["d_argmax"]), A2)
    g.close()


@pytest.mark.parametrize("widths,ns", [((1, 2, 4, 8, 16, 32, 64, 128, 256), 4099), ((1, 2, 8, 64, 512, 1024), 5203),
                                       ((4,), 777)])
def test_sliding_boxcar_mode_equals_oracle(widths, ns):
    """integration_mode = SLIDING (8(f) f1, INT.1s): the stride-1 boxcar S/N of ddp_integrate_snr against
    oracle.search_sliding (S/N within 1e-5, argmax = first sample of the best window, exact) for every kernel shape;
    the calls that need materialised sums refuse the plan."""
    import oracle
    cfg = small_direct(name="slide%d" % ns, nchan=24, nsamp_out=ns, ndm=13, widths=widths, n_pulses=2)
    g = GpuSearch(cfg, integration_mode=1)
    assert g.info.integration_mode == 1 and g.info.integ_elems == 0
    assert [g.info.plane_len[k] for k in range(len(widths))] == [ns - w + 1 for w in widths]
    Yg = g.dedisperse()
    Yo = oracle_direct_rows(cfg, g.X)
    assert np.array_equal(Yg, Yo)
    _, So, Ao = oracle.search_sliding(Yo, list(widths))
    V = g.plan.enumerate_kcfgs(ddp.K_ISNR)
    assert len(V) >= 10
    for c in V:
        g.plan.set_kcfg(ddp.K_ISNR, c)
        g.buf["d_snr"].fill_(-7.0)
        g.buf["d_argmax"].fill_(-1)
        g.plan.integrate_snr(g.buf["d_out"], g.buf["d_snr"], g.buf["d_argmax"])
        g.torch.cuda.synchronize()
        assert_snr_close(g.buf["d_snr"].cpu().numpy(), So, "sliding %r" % c)
        assert np.array_equal(u32(g.buf["d_argmax"]), Ao), "sliding argmax differs for %r" % c
    for call in (lambda: g.plan.integrate(g.buf["d_out"], g.buf["d_snr"]),
                 lambda: g.plan.snr(g.buf["d_out"], None, g.buf["d_snr"], g.buf["d_argmax"])):
        with pytest.raises(ddp.DdpError) as e:
            call()
        assert e.value.status == ddp.binding.E_CONFIG
    # the end-to-end call works without a plane buffer
    h_snr = np.full(So.shape, -3.0, dtype=np.float32)
    g.plan.search_host(g.X, g.buf["d_in"], g.buf["d_out"], None, g.buf["d_snr"], g.buf["d_argmax"], h_snr, None)
    assert_snr_close(h_snr, So, "sliding search_host")
    g.close()


def test_sliding_boxcar_recovers_the_misaligned_cfg0_pulse_at_its_width():
    """SURVEY INT.1: the BJ:cfg0 pulse moved to t0 = 2002 (not a multiple of its width 4) is found at (DM 17, w 4,
    t 2002) by the sliding search, while the decimating search of the same data peaks at width 2."""
    import dataclasses
    base = configs.tiny()
    cfg = dataclasses.replace(base, fixed_pulses=(dataclasses.replace(base.fixed_pulses[0], t0=2002),))
    gs = GpuSearch(cfg, integration_mode=1)
    gs.dedisperse()
    gs.plan.integrate_snr(gs.buf["d_out"], gs.buf["d_snr"], gs.buf["d_argmax"])
    gs.torch.cuda.synchronize()
    S, A = gs.buf["d_snr"].cpu().numpy(), u32(gs.buf["d_argmax"])
    i, k = np.unravel_index(np.argmax(S), S.shape)
    assert cfg.dm_list()[i] == 17.0 and cfg.widths[k] == 4 and A[i, k] == 2002
    gd = GpuSearch(cfg, X=gs.X)
    gd.run_all()
    Sd = gd.buf["d_snr"].cpu().numpy()
    i2, k2 = np.unravel_index(np.argmax(Sd), Sd.shape)
    assert cfg.dm_list()[i2] == 17.0 and cfg.widths[k2] == 2 and S[i, k] > Sd[i2, k2]
    gs.close()
    gd.close()


# ---------------------------------------------------------------------------------- channel mask (8(f) f4)
def test_channel_mask_direct_every_staging_mode():
    """A plan with zapped channels (reading DD.7m) against oracle.dedisperse_masked, bit-exact, for direct loads,
    cooperative and TMA staging, the packed kernel's wide flush (320 channels) and merged staging; what the masked
    channels hold must not matter (they are filled with 255 here)."""
    import oracle
    nchan = 320
    cfg = small_direct(name="mask", nchan=nchan, nsamp_out=2300, ndm=41, widths=(1, 2, 4, 8), n_pulses=2)
    rng = np.random.default_rng(7)
    mask = (rng.random(nchan) > 0.2).astype(np.uint8)
    mask[:3] = 0
    mask[-1] = 0
    g = GpuSearch(cfg, chan_mask=mask)
    assert g.info.nchan_masked == int((mask == 0).sum()) > 10
    g.X[mask == 0] = 255
    g.upload()
    delay = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    Yo = oracle.dedisperse_masked(g.X, mask, delay, cfg.nsamp_out)
    V = g.plan.enumerate_kcfgs(ddp.K_DIRECT)
    picks = []
    for st in (0, 1, 2, 3, 4):
        picks += _sample([c for c in V if c.staging == st], 6, seed=st)
    assert {c.staging for c in picks} == {0, 1, 2, 3, 4}
    for c in picks:
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        g.buf["d_out"].fill_(-1)
        assert np.array_equal(g.dedisperse(), Yo), "masked direct differs for %r" % c
    g.run_all()
    compare_all(g, Yo, what="masked, whole pipeline")
    # all channels kept == no mask at all
    g2 = GpuSearch(cfg, X=g.X, chan_mask=np.ones(nchan, np.uint8))
    assert np.array_equal(g2.dedisperse(), oracle_direct_rows(cfg, g.X))
    g.close()
    g2.close()


def test_channel_mask_subband_plan():
    """Masked channels in a two-step plan: equal to the subband oracle on a copy of the input whose masked channels
    are zero (a zero row adds nothing), S and Y bit-exact."""
    cfg = small_subband(name="mask_sb")
    mask = np.ones(cfg.nchan, np.uint8)
    mask[[0, 5, 11, 12, 13, 40, 95]] = 0
    g = GpuSearch(cfg, chan_mask=mask)
    Xz = g.X.copy()
    Xz[mask == 0] = 0
    g.X[mask == 0] = 200
    g.upload()
    So, Yo = oracle_subband(cfg, Xz)
    g.run_all()
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="masked subband")
    g.close()


def test_subband_step1_diagonal_tiles_and_the_ascending_band_fallback():
    """Staged step 1 lays its time tiles out in input-aligned time with a per-trial output shift when the delays
    relative to a subband's first channel spread far less than the delays themselves.  Covered
    here: a plan with a coarse DM step large enough to switch it on at every DM-tile size (windows of several
    tiles' length without it), ragged first / last tiles, a ragged DM tile; and the same band in ASCENDING channel
    order, where the first channel of a subband is its latest and the plain layout must be used -- S and Y
    against the oracle for sampled staged shapes of both."""
    import dataclasses
    base = small_subband(name="diag_sb", nchan=192, nsamp_out=3100, ndm=21 * 4,
                         subband=SubbandPlan(n_subbands=8, n_coarse=21, coarse_first=0.0, coarse_step=24.0,
                                             n_fine=4, fine_step=0.5))
    # 96 channels per subband: two delay superchunks of 64 rows, the second one's window bounds are made while the
    # first is summed
    long_sb = small_subband(name="diag_sb96", nchan=384, nsamp_out=2200, ndm=17 * 2,
                            subband=SubbandPlan(n_subbands=4, n_coarse=17, coarse_first=0.0, coarse_step=24.0,
                                                n_fine=2, fine_step=0.5))
    for cfg in (base, dataclasses.replace(base, name="diag_sb_ascending", f_hi_mhz=base.f_lo_mhz, f_lo_mhz=base.f_hi_mhz),
                long_sb):
        g = GpuSearch(cfg)
        So, Yo = oracle_subband(cfg, g.X)
        V = [c for c in g.plan.enumerate_kcfgs(ddp.K_SUB1) if c.staging in (1, 2)]
        picks = _sample(V, 40, seed=31)
        # blocks of fewer threads than a delay superchunk has rows (64): the per-row min / max of the relative
        # delays must still cover every row (a 32-thread block once left half of them unset)
        picks += _sample([c for c in V if c.threads_t * c.threads_dm <= 64], 12, seed=32)
        assert {c.staging for c in picks} == {1, 2}
        for c in picks:
            g.plan.set_kcfg(ddp.K_SUB1, c)
            g.buf["d_out"].fill_(-1)
            Y = g.dedisperse()
            assert np.array_equal(g.subband_intermediate(), So), "%s: S differs for %r" % (cfg.name, c)
            assert np.array_equal(Y, Yo), "%s: Y differs for %r" % (cfg.name, c)
        g.close()
    # the diagonal layout with zapped channels (masked rows read the workspace's row of zeros, which is only
    # in_stride_min long: the shifted tiles must not read past it)
    mask = np.ones(base.nchan, np.uint8)
    mask[[0, 1, 23, 24, 100, 191]] = 0
    g = GpuSearch(base, chan_mask=mask)
    Xz = g.X.copy()
    Xz[mask == 0] = 0
    g.X[mask == 0] = 255
    g.upload()
    So, Yo = oracle_subband(base, Xz)
    for c in _sample([c for c in g.plan.enumerate_kcfgs(ddp.K_SUB1) if c.staging in (1, 2)], 16, seed=33):
        g.plan.set_kcfg(ddp.K_SUB1, c)
        g.buf["d_out"].fill_(-1)
        Y = g.dedisperse()
        assert np.array_equal(g.subband_intermediate(), So), "masked, diagonal: S differs for %r" % c
        assert np.array_equal(Y, Yo), "masked, diagonal: Y differs for %r" % c
    g.close()


# ---------------------------------------------------------------------------------- DM rows split over ranks (8(f) f3)
@pytest.mark.parametrize("subband", [False, True])
def test_dm_sharded_search_equals_the_one_gpu_search(subband):
    """shard.plan_for_rank: one beam's DM trials split over 3 ranks.  Only one GPU is here, so the three ranks' plans
    run in turn on it, each on the same input (a rank's plan needs only its own largest delay of it); their rows,
    stacked, must be the oracle's rows of the whole search, and the S/N tables likewise (what gather_rows
    concatenates; its exchange itself is covered by the gloo test)."""
    from paper_1811_04165_b200.shard import plan_for_rank
    cfg = small_subband(name="shard_sb", ndm=6 * 5) if subband else small_direct(name="shard_d")
    whole = GpuSearch(cfg)
    Yo = oracle_subband(cfg, whole.X)[1] if subband else oracle_direct_rows(cfg, whole.X)
    _, So, Ao = oracle_search(Yo, list(cfg.widths), 0)
    world, rows, snrs, args = 3, [], [], []
    for r in range(world):
        plan, lo, hi = plan_for_rank(cfg, r, world)
        i = plan.query()
        assert i.ndm == hi - lo and i.in_stride_min <= whole.info.in_stride_min
        buf = ddp.alloc_buffers(plan, "cuda:0")
        buf["d_in"].copy_(torch.from_numpy(np.ascontiguousarray(whole.X[:, : i.in_stride_min])))
        plan.dedisperse(buf["d_in"], buf["d_out"])
        plan.integrate_snr(buf["d_out"], buf["d_snr"], buf["d_argmax"])
        torch.cuda.synchronize()
        rows.append(u32(buf["d_out"])[:, : i.nsamp_out])
        snrs.append(buf["d_snr"].cpu().numpy())
        args.append(u32(buf["d_argmax"]))
        plan.destroy()
    assert np.array_equal(np.concatenate(rows, axis=0), Yo)
    assert_snr_close(np.concatenate(snrs, axis=0), So, "sharded search")
    assert np.array_equal(np.concatenate(args, axis=0), Ao)
    whole.close()


# ---------------------------------------------------------------------------------- INPUT_BITS = 16 (8(f) f4)
def test_uint16_input_direct_sweep_saturation_mask_and_host_calls():
    """A 16-bit plan (ddp_options.input_bits = 16): uint16 samples through the uint16 code shapes of the direct
    kernel -- direct loads, cooperative and TMA staging over sampled shapes, bit-exact against the oracle's uint16
    sum; the whole pipeline; all-65535 input (the largest totals the plan's overflow proof admits); a channel
    mask; and the two host entry points, whose copies must move two bytes per sample."""
    import oracle
    from synth import filterbank
    cfg = small_direct(name="u16", nchan=80, nsamp_out=2300, ndm=41, widths=(1, 2, 4, 8), n_pulses=2)
    g = GpuSearch(cfg, input_bits=16)
    i = g.info
    assert i.input_bits == 16 and g.X.dtype == np.uint16 and int(g.X.max()) > 40000
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="u16 default")
    V = g.plan.enumerate_kcfgs(ddp.K_DIRECT)
    assert {c.staging for c in V} == {0, 1, 2}  # merged staging is for uint8 input
    seen = set()
    for c in _sample(V, 60, seed=16):
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        seen.add(c.staging)
        g.buf["d_out"].fill_(-1)
        assert np.array_equal(g.dedisperse(), Yo), "u16 direct differs for %r" % c
    assert seen == {0, 1, 2}
    keep = g.X.copy()
    g.X[:] = 65535
    g.upload()
    for c in _sample(V, 12, seed=17):
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        assert np.all(g.dedisperse() == 65535 * cfg.nchan), "saturated u16 input, %r" % c
    g.X[:] = keep
    g.upload()
    # host entry points
    h_snr = torch.full((i.ndm, i.nwidths), -3.0, dtype=torch.float32).pin_memory()
    h_arg = torch.full((i.ndm, i.nwidths), -1, dtype=torch.int32).pin_memory()
    g.buf["d_in"].zero_()
    g.plan.search_host(torch.from_numpy(g.X.view(np.int16)).pin_memory(), g.buf["d_in"], g.buf["d_out"], None,
                       g.buf["d_snr"], g.buf["d_argmax"], h_snr, h_arg)
    _, So, Ao = oracle_search(Yo, list(cfg.widths), 0)
    assert_snr_close(h_snr.numpy(), So, "u16 search_host")
    assert np.array_equal(h_arg.numpy().view(np.uint32), Ao)
    nb, ns, md = 2, cfg.nsamp_out, i.max_delay
    nlong = nb * ns + md
    Xl, _ = filterbank.make_filterbank(cfg, nlong, (nlong + 47) // 16 * 16, bits=16)
    Ylong = oracle.dedisperse(Xl, oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s), nb * ns)
    d_in1 = torch.zeros_like(g.buf["d_in"])
    g.buf["d_in"].zero_()
    hb_snr = torch.full((nb, i.ndm, i.nwidths), -3.0, dtype=torch.float32).pin_memory()
    hb_arg = torch.full((nb, i.ndm, i.nwidths), -1, dtype=torch.int32).pin_memory()
    g.plan.search_host_batches(torch.from_numpy(Xl.view(np.int16)).pin_memory(), nb, g.buf["d_in"], d_in1,
                               g.buf["d_out"], g.buf["d_snr"], g.buf["d_argmax"], hb_snr, hb_arg)
    for b in range(nb):
        _, Sb, Ab = oracle_search(np.ascontiguousarray(Ylong[:, b * ns: (b + 1) * ns]), list(cfg.widths), 0)
        assert_snr_close(hb_snr[b].numpy(), Sb, "u16 batch %d" % b)
        assert np.array_equal(hb_arg[b].numpy().view(np.uint32), Ab)
    g.close()
    # channel mask on a 16-bit plan
    mask = np.ones(cfg.nchan, np.uint8)
    mask[[0, 7, 8, 33, 79]] = 0
    gm = GpuSearch(cfg, input_bits=16, chan_mask=mask)
    Xz = gm.X.copy()
    Xz[mask == 0] = 0
    gm.X[mask == 0] = 65535
    gm.upload()
    Ym = oracle_direct_rows(cfg, Xz)
    for c in _sample(gm.plan.enumerate_kcfgs(ddp.K_DIRECT), 18, seed=18):
        gm.plan.set_kcfg(ddp.K_DIRECT, c)
        gm.buf["d_out"].fill_(-1)
        assert np.array_equal(gm.dedisperse(), Ym), "masked u16 direct differs for %r" % c
    gm.close()


def test_uint16_input_subband_plan():
    """A 16-bit two-step plan: the intermediate is uint32 (65535 * channels per subband does not fit 16 bits); S and
    Y against the oracle over sampled step-1 and step-2 shapes."""
    cfg = small_subband(name="u16_sb", nchan=96, nsamp_out=2100, ndm=12 * 8,
                        subband=SubbandPlan(n_subbands=8, n_coarse=12, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=8, fine_step=0.25))
    g = GpuSearch(cfg, input_bits=16)
    assert g.info.input_bits == 16 and g.info.sub_elem_bytes == 4
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="u16 subband default")
    for kernel in (ddp.K_SUB1, ddp.K_SUB2):
        keep = g.plan.get_kcfg(kernel)
        seen = set()
        for c in _sample(g.plan.enumerate_kcfgs(kernel), 30, seed=20 + kernel):
            g.plan.set_kcfg(kernel, c)
            seen.add(c.staging)
            g.buf["d_out"].fill_(-1)
            Y = g.dedisperse()
            assert np.array_equal(g.subband_intermediate(), So), "u16 plan: S differs for %r" % c
            assert np.array_equal(Y, Yo), "u16 plan: Y differs for %s %r" % (ddp.KERNEL_NAMES[kernel], c)
        assert seen >= {0, 1}
        g.plan.set_kcfg(kernel, keep)
    g.close()


@pytest.mark.parametrize("kernel", [ddp.K_SUB1, ddp.K_SUB2])
def test_subband_plan_kernel_configuration_sweep(kernel):
    cfg = small_subband(name="sweep_sb", nchan=128, nsamp_out=2100, ndm=24 * 8,
                        subband=SubbandPlan(n_subbands=8, n_coarse=24, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=8, fine_step=0.25))
    g = GpuSearch(cfg)
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    compare_all(g, Yo, what="sweep_sb default")
    seen = set()
    for c in _sample(g.plan.enumerate_kcfgs(kernel), 48, seed=kernel):
        g.plan.set_kcfg(kernel, c)
        seen.add(c.staging)
        g.buf["d_out"].fill_(-1)
        Y = g.dedisperse()
        assert np.array_equal(g.subband_intermediate(), So), "S differs for %r" % c
        assert np.array_equal(Y, Yo), "Y differs for %s %r" % (ddp.KERNEL_NAMES[kernel], c)
    assert seen >= {0, 1, 2}
    g.close()


# ---------------------------------------------------------------------------------- merged staging (genes 3, 4)
def _merged(plan, kernel, n, seed):
    V = [c for c in plan.enumerate_kcfgs(kernel) if c.staging >= 3]
    assert V, "no merged-staging shape is valid for this plan"
    picks = _sample(V, n, seed)
    # make sure both group sizes and several chunk sizes are in
    for st in (3, 4):
        picks += [c for c in V if c.staging == st][:2] + [c for c in V if c.staging == st][-2:]
    return picks


@pytest.mark.parametrize("nchan,ndm,dm_step", [(64, 41, 0.25), (80, 37, 0.25), (320, 41, 0.25), (512, 23, 0.5), (96, 64, 1.0)])
def test_direct_merged_staging_sweep_and_saturation(nchan, ndm, dm_step):
    """Staging genes 3 / 4: 2 / 4 adjacent channels pre-summed per distinct tuple of relative delays, then added
    by the trials.  Bit-exact against the oracle over sampled shapes (ragged time and DM tiles, reductions of
    64 ... 512 channels incl. the 256-row flush with and without a ragged last flush, one and several delay
    superchunks), and with all-255 input (largest lane values)."""
    import dataclasses
    cfg = dataclasses.replace(small_direct(name="merge%d" % nchan, nchan=nchan, nsamp_out=2300, ndm=ndm,
                                           widths=(1, 2, 4, 8), n_pulses=2), dm_step=dm_step)
    g = GpuSearch(cfg)
    Yo = oracle_direct_rows(cfg, g.X)
    picks = _merged(g.plan, ddp.K_DIRECT, 36, seed=nchan)
    assert {c.staging for c in picks} == {3, 4}
    for c in picks:
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        g.buf["d_out"].fill_(-1)
        assert np.array_equal(g.dedisperse(), Yo), "merged direct differs for %r" % c
    g.run_all()
    compare_all(g, Yo, what="merged direct, whole pipeline")
    g.X[:] = 255
    g.upload()
    for c in picks[::4]:
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        g.buf["d_out"].fill_(-1)
        assert np.all(g.dedisperse() == 255 * nchan), "saturated merged direct differs for %r" % c
    g.close()


def test_direct_merged_staging_unsorted_channel_order():
    """Channel order is arbitrary (DD.3): with shuffled channels the relative delays of 'adjacent' rows are
    large and of either sign; shapes that stay valid must still be exact."""
    import dataclasses
    base = small_direct(name="merge_shuffled", nchan=32, nsamp_out=1500, ndm=16, widths=(1, 2), n_pulses=1)
    rng = np.random.default_rng(5)
    perm = rng.permutation(base.nchan)
    f = base.chan_freq_mhz()[perm]
    plan = ddp.plan_create(f, base.t_samp_s, base.dm_list(), base.widths, base.nsamp_out)
    info = plan.query()
    b = ddp.alloc_buffers(plan)
    from synth import filterbank
    X0, _ = filterbank.make_filterbank(base, int(info.nsamp_in_required), int(info.in_stride_min))
    X = np.ascontiguousarray(X0[perm])
    b["d_in"].copy_(torch.from_numpy(X))
    import oracle
    Yo = oracle.dedisperse(X, oracle.delay_table(f, base.dm_list(), base.t_samp_s), base.nsamp_out)
    V = [c for c in plan.enumerate_kcfgs(ddp.K_DIRECT) if c.staging >= 3]
    assert V
    for c in _sample(V, 16, seed=9):
        plan.set_kcfg(ddp.K_DIRECT, c)
        b["d_out"].fill_(-1)
        plan.dedisperse(b["d_in"], b["d_out"])
        torch.cuda.synchronize()
        assert np.array_equal(u32(b["d_out"])[:, : base.nsamp_out], Yo), "merged, shuffled channels: %r" % c
    plan.destroy()


@pytest.mark.parametrize("cps,wide", [(16, False), (48, False), (260, True)])
def test_subband_step1_merged_staging(cps, wide):
    """Step 1 with merged staging: uint16 result (OUT16) and, for more than 257 channels per subband, the
    uint32 intermediate with the 256-row flush; S and Y against the oracle."""
    nsub = 4 if wide else 8
    cfg = small_subband(name="merge_sb%d" % cps, nchan=nsub * cps, nsamp_out=2100, ndm=12 * 8,
                        subband=SubbandPlan(n_subbands=nsub, n_coarse=12, coarse_first=0.0, coarse_step=2.0,
                                            n_fine=8, fine_step=0.25))
    g = GpuSearch(cfg)
    assert g.info.sub_elem_bytes == (4 if wide else 2)
    So, Yo = oracle_subband(cfg, g.X)
    for c in _merged(g.plan, ddp.K_SUB1, 24, seed=cps):
        g.plan.set_kcfg(ddp.K_SUB1, c)
        g.buf["d_out"].fill_(-1)
        Y = g.dedisperse()
        assert np.array_equal(g.subband_intermediate(), So), "merged step 1: S differs for %r" % c
        assert np.array_equal(Y, Yo), "merged step 1: Y differs for %r" % c
    g.close()


def test_subband_centre_reference_against_the_oracle():
    """SB.2 alternative: step-2 delays computed at the centre of every subband (option subband_ref = 1).  Only the
    table changes, so S, Y, the sums and the S/N must equal the oracle run with its own centre-reference table --
    and Y must differ from the default reading's on this input (the option is really in effect)."""
    cfg = small_subband(name="centre_sb", nchan=384, nsamp_out=2500, ndm=12 * 16,
                        subband=SubbandPlan(n_subbands=8, n_coarse=12, coarse_first=0.0, coarse_step=16.0,
                                            n_fine=16, fine_step=1.0))
    g = GpuSearch(cfg, subband_ref=1)
    assert g.info.subband_ref == 1
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X, ref="centre")
    assert np.array_equal(g.subband_intermediate(), So[:, :, : g.info.nsamp_sub])
    compare_all(g, Yo, what="centre reference")
    g2 = GpuSearch(cfg)
    assert g2.info.subband_ref == 0 and g2.info.max_d2 < g.info.max_d2
    assert not np.array_equal(g2.plan.get_delays(2), g.plan.get_delays(2))
    g2.run_all()
    compare_all(g2, oracle_subband(cfg, g2.X)[1], what="top reference")
    g2.close()
    g.close()


@pytest.mark.parametrize("nchan", [320, 512])
def test_direct_wide_reduction_sweep_and_saturation(nchan):
    """More than 257 channels: the packed kernel flushes its 16-bit lanes every 256 rows (WIDE), with a
    ragged last flush (320 = 256 + 64) and without one (512): staged shapes incl. single-buffered ones
    against the oracle, then all-255 input (the largest values the lanes and the flush can see)."""
    cfg = small_direct(name="wide%d" % nchan, nchan=nchan, nsamp_out=2100, ndm=41, widths=(1, 2, 4, 8), n_pulses=2)
    g = GpuSearch(cfg)
    g.run_all()
    Yo = oracle_direct_rows(cfg, g.X)
    compare_all(g, Yo, what="wide default")
    staged = [c for c in g.plan.enumerate_kcfgs(ddp.K_DIRECT) if c.staging in (1, 2)]
    picks = _sample(staged, 40, seed=nchan)
    seen = set()
    for c in picks:
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        seen.add((c.staging, c.unroll))
        g.buf["d_out"].fill_(-1)
        assert np.array_equal(g.dedisperse(), Yo), "wide direct differs for %r" % c
    assert {s for s, _ in seen} >= {1, 2} and len({u for _, u in seen}) >= 3
    g.X[:] = 255
    g.upload()
    for c in picks[::5]:
        g.plan.set_kcfg(ddp.K_DIRECT, c)
        g.buf["d_out"].fill_(-1)
        assert np.all(g.dedisperse() == 255 * nchan), "saturated wide direct differs for %r" % c
    g.close()


@pytest.mark.parametrize("cps", [96, 256])
def test_subband_step2_lane_group_sizes(cps):
    """Step 2 sums G subband words in 16-bit lanes before splitting them: G = 2 for 65..128 channels per
    subband, G = 1 for 129..257 (cfg2 itself has G = 4).  Sweep of staged step-2 shapes, plus all-255 input."""
    cfg = small_subband(name="g_cps%d" % cps, nchan=8 * cps, nsamp_out=1800, ndm=5 * 8,
                        subband=SubbandPlan(n_subbands=8, n_coarse=5, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=8, fine_step=0.25))
    g = GpuSearch(cfg)
    assert g.info.sub_elem_bytes == 2
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="lane group default")
    staged = [c for c in g.plan.enumerate_kcfgs(ddp.K_SUB2) if c.staging != 0]
    picks = _sample(staged, 24, seed=cps)
    assert {c.staging for c in picks} == {1, 2}
    for c in picks:
        g.plan.set_kcfg(ddp.K_SUB2, c)
        g.buf["d_out"].fill_(-1)
        assert np.array_equal(g.dedisperse(), Yo), "step 2 differs for %r" % c
    g.X[:] = 255
    g.upload()
    for c in picks[::4]:
        g.plan.set_kcfg(ddp.K_SUB2, c)
        g.buf["d_out"].fill_(-1)
        assert np.all(g.dedisperse() == 255 * 8 * cps)
    g.close()


def test_subband_wide_subbands_keep_uint32_intermediate():
    """SB.4: more than 257 channels per subband cannot be stored in 16 bits -> uint32 S, generic step 2."""
    cfg = small_subband(name="wide_sb", nchan=1040, nsamp_out=1500, ndm=4 * 6,
                        subband=SubbandPlan(n_subbands=2, n_coarse=4, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=6, fine_step=0.25))
    g = GpuSearch(cfg)
    assert g.info.sub_elem_bytes == 4
    g.run_all()
    So, Yo = oracle_subband(cfg, g.X)
    assert np.array_equal(g.subband_intermediate(), So)
    compare_all(g, Yo, what="wide_sb default")
    for kernel in (ddp.K_SUB1, ddp.K_SUB2):
        for c in _sample(g.plan.enumerate_kcfgs(kernel), 12, seed=7 + kernel):
            g.plan.set_kcfg(kernel, c)
            g.buf["d_out"].fill_(-1)
            Y = g.dedisperse()
            assert np.array_equal(g.subband_intermediate(), So), "S differs for %r" % c
            assert np.array_equal(Y, Yo), "Y differs for %s %r" % (ddp.KERNEL_NAMES[kernel], c)
    g.close()


def test_subband_saturated_input_fills_the_uint16_intermediate():
    """255 everywhere: S = 255 * channels-per-subband is the largest value the narrow storage must hold."""
    cfg = small_subband(name="sat_sb", nchan=8 * 256, nsamp_out=1100, ndm=3 * 4,
                        subband=SubbandPlan(n_subbands=8, n_coarse=3, coarse_first=0.0, coarse_step=8.0,
                                            n_fine=4, fine_step=0.25))
    g = GpuSearch(cfg)
    assert g.info.sub_elem_bytes == 2
    g.X[:] = 255
    g.upload()
    Y = g.dedisperse()
    assert np.all(g.subband_intermediate() == 255 * 256)
    assert np.all(Y == 255 * 8 * 256)
    g.close()


# ---------------------------------------------------------------------------------- full-size configs
# The shapes that are BENCHMARKED are the ones that are compared: every kernel slot is first left at the
# plan default and then set to its entry of tuned_b200.json (what bench.py times), and EVERY row of the
# result is compared with the oracle -- the all-cores leg (oracle_mt.cpp) computes all rows in seconds.
def _shape_sets(workload):
    return [("defaults", False), ("tuned_b200.json:" + workload, True)]


@pytest.mark.slow
def test_cfg1_full_size_every_row_default_and_tuned_shapes():
    cfg = configs.apertif_direct()
    g = GpuSearch(cfg)
    Yo = oracle_direct_all_rows_mt(cfg, g.X)
    assert tuned_shapes("cfg1"), "tuned_b200.json has no cfg1 entry"
    for what, tuned in _shape_sets("cfg1"):
        if tuned:
            g.apply_tuned("cfg1")
        g.buf["d_out"].fill_(-1)
        g.buf["d_integ"].fill_(-1)
        g.buf["d_snr"].fill_(-7.0)
        g.run_all()
        compare_all(g, Yo, what="cfg1 " + what, mt=True)
    # every injected pulse is found at its DM (rows of the pulses' DMs carry the S/N maxima nearby)
    S = g.buf["d_snr"].cpu().numpy()
    for p in g.pulses:
        i = int(round(p.dm / cfg.dm_step))
        lo, hi = max(0, i - 8), min(cfg.ndm, i + 9)
        assert S[lo:hi].max() > 6.0, "pulse %r not detected" % (p,)
    # a shape whose two buffers of shifted copies exceed 227 KB: single-buffered copies + wide flush
    g.plan.set_kcfg(ddp.K_DIRECT, ddp.Kcfg(64, 8, 16, 8, 16, 2, 16))
    g.buf["d_out"].fill_(-1)
    assert np.array_equal(g.dedisperse(), Yo), "single-buffered direct kernel differs"
    g.close()


@pytest.mark.slow
def test_cfg2_full_size_every_row_default_and_tuned_shapes_and_identity_rows():
    cfg = configs.apertif_subband()
    g = GpuSearch(cfg)
    sb = cfg.subband
    So, Yo = oracle_subband_mt(cfg, g.X)
    assert tuned_shapes("cfg2"), "tuned_b200.json has no cfg2 entry"
    for what, tuned in _shape_sets("cfg2"):
        if tuned:
            g.apply_tuned("cfg2")
        g.buf["d_out"].fill_(-1)
        g.buf["d_integ"].fill_(-1)
        g.buf["d_snr"].fill_(-7.0)
        g.run_all()
        assert np.array_equal(g.subband_intermediate(), So), "cfg2 %s: S differs" % what
        compare_all(g, Yo, what="cfg2 " + what, mt=True)
    # SB.6 / BJ:cfg2: zero-fine-offset rows equal config 1's direct rows at the same DM (all 64 of them)
    d = configs.apertif_direct()
    coarse = np.arange(sb.n_coarse)
    Yd = oracle_direct_all_rows_mt(d, g.X, coarse * sb.n_fine)
    assert np.array_equal(u32(g.buf["d_out"])[coarse * sb.n_fine, : cfg.nsamp_out], Yd)
    # step-1 shapes whose two buffers of shifted copies exceed 227 KB run single-buffered (TMA and
    # cooperative staging): same S, same Y
    for genes in ([128, 4, 16, 8, 4, 2, 16], [128, 4, 16, 8, 4, 1, 16]):
        g.plan.set_kcfg(ddp.K_SUB1, ddp.Kcfg(*genes))
        g.buf["d_out"].fill_(-1)
        Y = g.dedisperse()
        assert np.array_equal(g.subband_intermediate(), So), "S differs for single-buffered %r" % genes
        assert np.array_equal(Y, Yo), "Y differs for single-buffered %r" % genes
    g.close()


@pytest.mark.slow
def test_cfg3_full_size_every_row_default_and_tuned_shapes():
    cfg = configs.ska_mid()
    g = GpuSearch(cfg)
    Yo = oracle_direct_all_rows_mt(cfg, g.X)
    assert tuned_shapes("cfg3"), "tuned_b200.json has no cfg3 entry"
    for what, tuned in _shape_sets("cfg3"):
        if tuned:
            g.apply_tuned("cfg3")
        g.buf["d_out"].fill_(-1)
        g.buf["d_integ"].fill_(-1)
        g.buf["d_snr"].fill_(-7.0)
        g.run_all()
        compare_all(g, Yo, what="cfg3 " + what, mt=True)
    g.close()


@pytest.mark.slow
def test_cfg2_subband_vs_direct_snr_at_the_injected_pulses():
    """BJ:cfg2 "the DM-wise SNR peaks are compared against config 1's direct result" (SURVEY SB pin (v)).
    The subband method approximates direct dedispersion, so the two S/N values differ; what is pinned is
    that each GPU leg reproduces ITS oracle at every injected pulse's (DM, width), hence also the
    oracle-vs-oracle ratio, and that zero-fine-offset rows give identical S/N.  The table is printed
    (pytest -s) and quoted in DESIGN.md."""
    d, sbc = configs.apertif_direct(), configs.apertif_subband()
    nf = sbc.subband.n_fine
    widths = list(d.widths)
    gd = GpuSearch(d)
    pulses = gd.pulses
    rows = np.array(sorted({int(round(p.dm / d.dm_step)) for p in pulses} |
                           {int(round(p.dm / d.dm_step)) // nf * nf for p in pulses}))
    gd.run_all()
    Sd = gd.buf["d_snr"].cpu().numpy()[rows].copy()
    _, So_d, _ = oracle_search(oracle_direct_rows(d, gd.X, rows), widths, 0)
    assert_snr_close(Sd, So_d, "direct leg")
    gd.close()

    gs = GpuSearch(sbc)
    assert [(p.dm, p.t0, p.width, p.amplitude) for p in gs.pulses] == [(p.dm, p.t0, p.width, p.amplitude) for p in pulses]
    gs.run_all()
    Ss = gs.buf["d_snr"].cpu().numpy()[rows].copy()
    coarse = sorted({int(r) // nf for r in rows})
    _, Yo_s = oracle_subband(sbc, gs.X, np.array(coarse))
    pick = np.array([coarse.index(int(r) // nf) * nf + int(r) % nf for r in rows])
    _, So_s, _ = oracle_search(Yo_s[pick], widths, 0)
    assert_snr_close(Ss, So_s, "subband leg")
    gs.close()

    at = {int(r): n for n, r in enumerate(rows)}
    for r in rows:                       # SB.6: zero fine offset -> same integers -> same float32 S/N
        if int(r) % nf == 0:
            assert np.array_equal(Sd[at[int(r)]], Ss[at[int(r)]]), "row %d" % r
    print("\n  DM      t0  w amp | direct S/N  subband S/N  ratio | oracle ratio | fine offset b")
    for p in pulses:
        r = int(round(p.dm / d.dm_step))
        k = widths.index(p.width)
        n = at[r]
        ratio, oratio = Ss[n, k] / Sd[n, k], So_s[n, k] / So_d[n, k]
        assert abs(ratio - oratio) <= 3e-5 * max(1.0, abs(oratio))
        assert Sd[n, k] > 5.0 and Ss[n, k] > 0.0        # every pulse stands out in the direct search
        print("%7.2f %6d %2d %3d | %10.3f  %11.3f  %5.3f | %12.3f | %d" % (
            p.dm, p.t0, p.width, p.amplitude, Sd[n, k], Ss[n, k], ratio, oratio, r % nf))
