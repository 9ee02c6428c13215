"""Pins for oracle/ against what the paper and the mathematics fix (CPU only, no CUDA path).

Every test here compares the oracle with something other than itself: a hand-derived fixture,
a closed form, an invariant, a special case that reduces to a numpy routine, or a pure-Python
brute force written from the definition (PAPER.md; BASELINE.json
north_star / cfg0).
"""
import math

import numpy as np
import pytest

import oracle
from synth import configs, filterbank

K = 4.148808e3


# ----------------------------------------------------------------------------- helpers
def py_delays(f, dms, ts):
    fr = max(f)
    return [[math.floor(((K * dm) * (1.0 / (fc * fc) - 1.0 / (fr * fr))) / ts + 0.5) for fc in f] for dm in dms]


def py_dedisperse(X, delay, ns):
    """Brute force from the definition Y[i][t] = sum_c X[c][t + delay[i][c]] (pure Python)."""
    return [[sum(int(X[c][t + delay[i][c]]) for c in range(len(X))) for t in range(ns)]
            for i in range(len(delay))]


def small_case(seed, nchan=6, ndm=5, ns=37, dm_step=3.0):
    rng = np.random.default_rng(seed)
    f = np.sort(rng.uniform(1200.0, 1500.0, nchan))[::-1].copy()
    dms = dm_step * np.arange(ndm)
    ts = 1e-3
    delay = oracle.delay_table(f, dms, ts)
    nin = ns + int(delay.max())
    X = rng.integers(0, 256, size=(nchan, nin), dtype=np.uint8)
    return f, dms, ts, delay, X


# ----------------------------------------------------------------------------- DD: delays
def test_delay_worked_example(worked_example):
    f = [1500.0, 1400.0, 1300.0, 1200.0]
    d = oracle.delay_table(f, [0.0, 10.0, 20.0], 1e-3)
    assert d.tolist() == worked_example["delay"]


def test_delay_closed_form_values():
    # 4148.808 * DM * (f^-2 - fref^-2) / t_samp, hand-evaluated: see tests/golden/worked_example.txt
    d = oracle.delay_table([1500.0, 1400.0], [10.0], 1e-3)
    assert d[0, 0] == 0 and d[0, 1] == 3          # 2.7282 -> 3
    d = oracle.delay_table([1500.0, 1200.0], [20.0], 1e-3)
    assert d[0, 1] == 21                          # 20.744 -> 21
    # doubling t_samp halves the unrounded delay: 10.372 -> 5.186 -> 5
    d = oracle.delay_table([1500.0, 1200.0], [10.0], 2e-3)
    assert d[0, 1] == 5


def test_delay_reference_and_sign():
    cfg = configs.tiny()
    f = cfg.chan_freq_mhz()
    d = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    assert (d[0] == 0).all()                       # DM = 0: no shift
    assert (d[:, np.argmax(f)] == 0).all()         # top channel is the reference (DD.3)
    assert (d >= 0).all()                          # lower frequency arrives later (DD.4)
    assert (np.diff(d, axis=1) >= 0).all()         # descending frequency => non-decreasing delay
    assert (np.diff(d, axis=0) >= 0).all()         # increasing DM => non-decreasing delay
    assert d.max() == 344                          # SURVEY Appendix B, cfg 0 under FRQ.1
    # channel order must not matter (f_ref = max, not f[0])
    perm = np.random.default_rng(0).permutation(f.size)
    dp = oracle.delay_table(f[perm], cfg.dm_list(), cfg.t_samp_s)
    assert (dp == d[:, perm]).all()


def test_delay_matches_python_float64():
    cfg = configs.tiny()
    f = cfg.chan_freq_mhz()
    d = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    assert d.tolist() == py_delays(list(f), list(cfg.dm_list()), cfg.t_samp_s)


@pytest.mark.parametrize("mk,maxd", [(configs.apertif_direct, 11589), (configs.ska_mid, 213777)])
def test_delay_geometry_full_configs(mk, maxd):
    """SURVEY Appendix B max delays; and no entry is a near-tie at x.5 (DD.2), so a 1-ulp change of
    evaluation order cannot flip a rounding."""
    cfg = mk()
    f = cfg.chan_freq_mhz()
    dms = cfg.dm_list()
    d = oracle.delay_table(f, dms, cfg.t_samp_s)
    assert d.max() == maxd
    g = 1.0 / (f * f) - 1.0 / (f.max() ** 2)
    x = (K * dms)[:, None] * g[None, :] / cfg.t_samp_s
    assert (np.floor(x + 0.5).astype(np.int64) == d).all()
    frac = np.abs((x - np.floor(x)) - 0.5)
    assert frac.min() > 1e-9


# ----------------------------------------------------------------------------- DD: sums
def test_dedisperse_worked_example(worked_example):
    f = [1500.0, 1400.0, 1300.0, 1200.0]
    d = oracle.delay_table(f, [0.0, 10.0, 20.0], 1e-3)
    nin = 8 + 21
    X = np.array([[(7 * c + 3 * t) % 11 for t in range(nin)] for c in range(4)], dtype=np.uint8)
    Y = oracle.dedisperse(X, d, 8)
    assert Y.tolist() == worked_example["Y"]
    assert oracle.integrate(Y, 2).tolist() == worked_example["I2"]
    assert oracle.integrate(Y, 4).tolist() == worked_example["I4"]
    for w, Iw in ((1, Y), (2, oracle.integrate(Y, 2)), (4, oracle.integrate(Y, 4))):
        s, a = oracle.snr(np.ascontiguousarray(Iw))
        assert np.allclose(s, worked_example["snr%d" % w][0], rtol=0, atol=1e-6)
        assert a.tolist() == worked_example["argmax%d" % w][0]


def test_dm0_is_plain_channel_sum():
    cfg = configs.tiny()
    f = cfg.chan_freq_mhz()
    d = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    X, _ = filterbank.make_filterbank(cfg, cfg.nsamp_out + int(d.max()))
    Y = oracle.dedisperse(X, d[:1], cfg.nsamp_out)
    assert (Y[0] == X[:, :cfg.nsamp_out].astype(np.uint32).sum(axis=0)).all()


def test_constant_input():
    f, dms, ts, delay, X = small_case(1)
    X[:] = 37
    Y = oracle.dedisperse(X, delay, 37)
    assert (Y == 37 * X.shape[0]).all()


def test_impulse_response_every_delay():
    """A single 1 at (c*, t*) must appear in row i at t* - delay[i][c*] and nowhere else:
    checks the sign of the shift and every table entry individually (DD.4)."""
    f, dms, ts, delay, X = small_case(2)
    ns = 37
    for cstar in range(X.shape[0]):
        tstar = int(delay[:, cstar].max()) + 5
        X[:] = 0
        X[cstar, tstar] = 1
        Y = oracle.dedisperse(X, delay, ns)
        for i in range(delay.shape[0]):
            expect = np.zeros(ns, dtype=np.uint32)
            pos = tstar - int(delay[i, cstar])
            if 0 <= pos < ns:
                expect[pos] = 1
            assert (Y[i] == expect).all()


def test_linearity():
    f, dms, ts, delay, X = small_case(3)
    rng = np.random.default_rng(7)
    X1 = rng.integers(0, 128, size=X.shape, dtype=np.uint8)
    X2 = rng.integers(0, 128, size=X.shape, dtype=np.uint8)
    Y1, Y2 = oracle.dedisperse(X1, delay, 37), oracle.dedisperse(X2, delay, 37)
    assert (oracle.dedisperse((X1 + X2).astype(np.uint8), delay, 37) == Y1 + Y2).all()


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_bruteforce_tiny(seed):
    f, dms, ts, delay, X = small_case(seed)
    Y = oracle.dedisperse(X, delay, 37)
    assert Y.tolist() == py_dedisperse(X.tolist(), delay.tolist(), 37)


def test_numpy_gather_cfg0():
    """Third implementation: vectorised numpy gather over the whole of cfg 0."""
    cfg = configs.tiny()
    f = cfg.chan_freq_mhz()
    d = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    ns = cfg.nsamp_out
    X, _ = filterbank.make_filterbank(cfg, ns + int(d.max()))
    Y = oracle.dedisperse(X, d, ns)
    t = np.arange(ns)
    for i in range(0, cfg.ndm, 5):
        ref = X[np.arange(cfg.nchan)[:, None], t[None, :] + d[i][:, None]].astype(np.uint64).sum(axis=0)
        assert (Y[i] == ref).all()


def test_uint8_saturated_input_no_overflow():
    f, dms, ts, delay, X = small_case(4, nchan=9)
    X[:] = 255
    assert (oracle.dedisperse(X, delay, 37) == 255 * 9).all()


def test_short_input_is_an_error():
    f, dms, ts, delay, X = small_case(5)
    with pytest.raises(ValueError):
        oracle.dedisperse(np.ascontiguousarray(X[:, :-1]), delay, 37)


# ----------------------------------------------------------------------------- SB
def sb_case(seed, nchan=12, nsub=3, ncoarse=4, nfine=4, coarse_step=8.0, ns=41):
    rng = np.random.default_rng(seed)
    f = 1500.0 - np.arange(nchan) * (300.0 / nchan)
    ts = 1e-3
    A = coarse_step * np.arange(ncoarse)
    F = (coarse_step / nfine) * np.arange(nfine)
    d1, d2 = oracle.subband_tables(f, ts, nsub, A, F)
    ns1 = ns + int(d2.max())
    nin = ns1 + int(d1.max())
    X = rng.integers(0, 256, size=(nchan, nin), dtype=np.uint8)
    return f, ts, A, F, d1, d2, ns1, X


def test_subband_bruteforce_tiny():
    ns, nsub = 41, 3
    f, ts, A, F, d1, d2, ns1, X = sb_case(21, ns=ns, nsub=nsub)
    S = oracle.subband_step1(X, d1, nsub, ns1)
    Y = oracle.subband_step2(S, d2, ns)
    cps = f.size // nsub
    fr = f.max()
    # pure-Python restatement of SB.1 reading "B": total shift of channel c in trial (a, b)
    # is d1[a][c] + d2[b][sub(c)], with d1/d2 from the formula evaluated in Python.
    for a in range(len(A)):
        for b in range(len(F)):
            for t in range(0, ns, 7):
                acc = 0
                for c in range(f.size):
                    s = c // cps
                    fs = max(f[s * cps:(s + 1) * cps])
                    dd1 = math.floor(((K * A[a]) * (1 / f[c] ** 2 - 1 / fr ** 2)) / ts + 0.5)
                    dd2 = math.floor(((K * F[b]) * (1 / fs ** 2 - 1 / fr ** 2)) / ts + 0.5)
                    acc += int(X[c][t + dd1 + dd2])
                assert Y[a * len(F) + b][t] == acc


def test_subband_zero_fine_offset_rows_equal_direct():
    """SB.6: rows with b = 0 have d2 == 0 and are bit-identical to direct at DM = A[a]."""
    ns, nsub = 41, 3
    f, ts, A, F, d1, d2, ns1, X = sb_case(22, ns=ns, nsub=nsub)
    assert (d2[0] == 0).all()
    Y = oracle.subband_step2(oracle.subband_step1(X, d1, nsub, ns1), d2, ns)
    direct = oracle.dedisperse(X, oracle.delay_table(f, A, ts), ns)
    assert (Y[::len(F)] == direct).all()


def test_subband_single_subband_equals_direct_at_coarse_dm():
    """nSub = 1: f_sub = f_ref so d2 == 0 and every row (a, b) equals direct at A[a]."""
    ns = 41
    f, ts, A, F, d1, d2, ns1, X = sb_case(23, ns=ns, nsub=1)
    assert (d2 == 0).all()
    Y = oracle.subband_step2(oracle.subband_step1(X, d1, 1, ns1), d2, ns)
    direct = oracle.dedisperse(X, oracle.delay_table(f, A, ts), ns)
    for b in range(len(F)):
        assert (Y[b::len(F)] == direct).all()


def test_subband_one_channel_per_subband_shift_is_d1_plus_d2():
    """cps = 1: f_sub[s] = f[s], so the trial (a, b) shifts channel c by
    round(K A g/ts) + round(K F g/ts) -- a direct sum with that summed delay table."""
    ns, nsub = 41, 12
    f, ts, A, F, d1, d2, ns1, X = sb_case(24, ns=ns, nsub=nsub)
    Y = oracle.subband_step2(oracle.subband_step1(X, d1, nsub, ns1), d2, ns)
    tot = (d1[:, None, :] + d2[None, :, :]).reshape(-1, f.size)
    assert (Y == oracle.dedisperse(X, tot, ns)).all()


def test_subband_cfg2_geometry():
    cfg = configs.apertif_subband()
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)
    assert d1.max() == 11413 and d2.max() == 168
    # per-channel total delay differs from direct by -8..+1 samples (SB.6)
    direct = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    cps = cfg.nchan // sb.n_subbands
    tot = (d1[:, None, :] + np.repeat(d2, cps, axis=1)[None, :, :]).reshape(cfg.ndm, cfg.nchan)
    err = tot.astype(np.int64) - direct
    assert err.min() == -8 and err.max() == 1
    assert (err[::sb.n_fine] == 0).all()


def test_subband_centre_reference_tables():
    """Reading SB.2c (subband reference = centre of the subband): only the step-2 table changes; with one channel
    per subband the centre IS the channel, so it equals the default; at BJ:cfg2 the per-channel total delay then
    differs from direct by -5..+4 samples instead of -8..+1 (computed there independently), and
    a closed-form entry checks the frequency that is used."""
    cfg = configs.apertif_subband()
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    f = cfg.chan_freq_mhz()
    d1t, d2t = oracle.subband_tables(f, cfg.t_samp_s, sb.n_subbands, A, F)
    d1c, d2c = oracle.subband_tables(f, cfg.t_samp_s, sb.n_subbands, A, F, ref="centre")
    assert np.array_equal(d1c, d1t) and not np.array_equal(d2c, d2t)
    direct = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    cps = cfg.nchan // sb.n_subbands
    tot = (d1c[:, None, :] + np.repeat(d2c, cps, axis=1)[None, :, :]).reshape(cfg.ndm, cfg.nchan)
    err = tot.astype(np.int64) - direct
    assert err.min() == -5 and err.max() == 4
    # closed form: last subband, largest fine offset, centre of its 48 channels
    fs = f.reshape(sb.n_subbands, cps)[-1]
    fc = 0.5 * (fs.max() + fs.min())
    x = ((K * F[-1]) * (1.0 / (fc * fc) - 1.0 / (f.max() * f.max()))) / cfg.t_samp_s
    assert d2c[-1, -1] == math.floor(x + 0.5)
    # one channel per subband: centre == the channel
    a1, a2 = oracle.subband_tables(f[:16], cfg.t_samp_s, 16, A[:3], F[:5])
    b1, b2 = oracle.subband_tables(f[:16], cfg.t_samp_s, 16, A[:3], F[:5], ref="centre")
    assert np.array_equal(a1, b1) and np.array_equal(a2, b2)


def test_uint16_input_sums():
    """INPUT_BITS = 16: the same sums over uint16 samples.  Pins: the worked example scaled by
    257 (every sample v -> 257 v, so every sum scales alike); linearity X = 256 H + L  =>  Y(X) = 256 Y(H) + Y(L)
    with the uint8 functions (pinned above) on both bytes; brute force with numpy on the ragged small case;
    saturated input 65535 everywhere; and the same for subband step 1."""
    f = [1500.0, 1400.0, 1300.0, 1200.0]
    d = oracle.delay_table(f, [0.0, 10.0, 20.0], 1e-3)
    X8 = np.array([[(7 * c + 3 * t) % 11 for t in range(8 + 21)] for c in range(4)], dtype=np.uint8)
    Y8 = oracle.dedisperse(X8, d, 8)
    assert np.array_equal(oracle.dedisperse((X8.astype(np.uint16) * 257), d, 8), Y8 * 257)
    cfg = configs.tiny()
    delay = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    nin = cfg.nsamp_out + int(delay.max())
    X, _ = filterbank.make_filterbank(cfg, nin, nin + 5, bits=16)
    assert X.dtype == np.uint16 and X.max() > 255
    H, L = (X >> 8).astype(np.uint8), (X & 0xFF).astype(np.uint8)
    rows = delay[[0, 3, cfg.ndm - 1]]
    Y = oracle.dedisperse(X, rows, cfg.nsamp_out)
    assert np.array_equal(Y, 256 * oracle.dedisperse(H, rows, cfg.nsamp_out) + oracle.dedisperse(L, rows, cfg.nsamp_out))
    t = np.arange(cfg.nsamp_out)
    brute = np.zeros(cfg.nsamp_out, dtype=np.int64)
    for c in range(cfg.nchan):
        brute += X[c, t + rows[2, c]]
    assert np.array_equal(Y[2], brute)
    sat = np.full((cfg.nchan, nin), 65535, dtype=np.uint16)
    assert (oracle.dedisperse(sat, rows, cfg.nsamp_out) == 65535 * cfg.nchan).all()
    # subband step 1
    nsub, A = 8, np.array([0.0, 4.0, 8.0])
    d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, nsub, A, np.array([0.0, 0.5, 1.0]))
    ns1 = cfg.nsamp_out + int(d2.max())
    Xs, _ = filterbank.make_filterbank(cfg, ns1 + int(d1.max()), bits=16)
    S = oracle.subband_step1(Xs, d1, nsub, ns1)
    Hs, Ls = (Xs >> 8).astype(np.uint8), (Xs & 0xFF).astype(np.uint8)
    assert np.array_equal(S, 256 * oracle.subband_step1(Hs, d1, nsub, ns1) + oracle.subband_step1(Ls, d1, nsub, ns1))
    cps = cfg.nchan // nsub
    b = np.zeros(ns1, dtype=np.int64)
    for c in range(5 * cps, 6 * cps):
        b += Xs[c, np.arange(ns1) + d1[2, c]]
    assert np.array_equal(S[2, 5], b)


# ----------------------------------------------------------------------------- INT
def test_integrate_invariants():
    rng = np.random.default_rng(31)
    Y = rng.integers(0, 2 ** 20, size=(5, 1000), dtype=np.uint32)
    for w in (1, 2, 3, 4, 7, 8, 16, 64, 256):
        I = oracle.integrate(Y, w)
        n = 1000 // w
        assert I.shape == (5, n)
        assert (I == Y[:, :n * w].reshape(5, n, w).sum(axis=2)).all()      # numpy routine
        assert (I.sum(axis=1, dtype=np.uint64) == Y[:, :n * w].sum(axis=1, dtype=np.uint64)).all()
    I4, I8 = oracle.integrate(Y, 4), oracle.integrate(Y, 8)
    assert (I8 == I4[:, 0:250:2] + I4[:, 1:250:2]).all()                     # INT.4
    assert (oracle.integrate(Y, 1) == Y).all()


def test_integrate_constant_and_tail():
    Y = np.full((2, 24414), 9, dtype=np.uint32)
    I = oracle.integrate(Y, 256)
    assert I.shape == (2, 95) and (I == 9 * 256).all()                        # 24414 // 256 = 95, tail dropped
    Y[:, 95 * 256:] = 1000                                                    # the dropped tail must not leak
    assert (oracle.integrate(Y, 256) == 9 * 256).all()


# ----------------------------------------------------------------------------- SNR
def test_snr_matches_numpy_float64():
    rng = np.random.default_rng(41)
    V = rng.integers(10 ** 7, 10 ** 7 + 50000, size=(6, 3051), dtype=np.uint32)
    s, a = oracle.snr(V)
    v = V.astype(np.float64)
    ref = (v.max(axis=1) - v.mean(axis=1)) / v.std(axis=1)                    # numpy std: ddof = 0 (SNR.2)
    assert np.allclose(s, ref.astype(np.float32), rtol=1e-6, atol=0)
    assert (a == v.argmax(axis=1)).all()
    s1, _ = oracle.snr(V, ddof=1)
    assert np.allclose(s1, (ref * math.sqrt((3051 - 1) / 3051)).astype(np.float32), rtol=1e-6)


def test_snr_single_spike_closed_form():
    """n-1 values a and one value a+h: mean = a + h/n, var = h^2 (n-1)/n^2 => snr = sqrt(n-1)."""
    for n, a, h, pos in ((100, 5000, 77, 13), (4096, 8192, 1, 4095), (95, 10 ** 8, 12345, 0)):
        V = np.full((1, n), a, dtype=np.uint32)
        V[0, pos] += h
        s, am = oracle.snr(V)
        assert abs(s[0] - math.sqrt(n - 1)) <= 1e-6 * math.sqrt(n - 1)
        assert am[0] == pos


def test_snr_invariances_and_degenerate():
    rng = np.random.default_rng(43)
    v = rng.integers(1000, 5000, size=(1, 777), dtype=np.uint32)
    s, a = oracle.snr(v)
    s2, _ = oracle.snr(v * np.uint32(3) + np.uint32(11))                      # affine, a > 0
    assert abs(s2[0] - s[0]) <= 1e-6 * abs(s[0])
    perm = rng.permutation(777)
    s3, _ = oracle.snr(np.ascontiguousarray(v[:, perm]))
    assert abs(s3[0] - s[0]) <= 1e-6 * abs(s[0])
    c = np.full((2, 50), 123, dtype=np.uint32)
    sc, ac = oracle.snr(c)
    assert (sc == 0).all() and (ac == 0).all() and np.isfinite(sc).all()       # SNR.3
    tie = np.array([[1, 9, 3, 9, 9]], dtype=np.uint32)
    assert oracle.snr(tie)[1][0] == 1                                          # lowest index (SNR.4)


# ----------------------------------------------------------------------------- end to end
def test_cfg0_pulse_recovered_at_its_dm_and_width():
    """BASELINE.json north_star: an injected dispersed pulse is recovered at its DM and width."""
    cfg = configs.tiny()
    f = cfg.chan_freq_mhz()
    d = oracle.delay_table(f, cfg.dm_list(), cfg.t_samp_s)
    X, pulses = filterbank.make_filterbank(cfg, cfg.nsamp_out + int(d.max()))
    Y = oracle.dedisperse(X, d, cfg.nsamp_out)
    _, S, A = oracle.search(Y, cfg.widths)
    i, j = np.unravel_index(np.argmax(S), S.shape)
    p = pulses[0]
    assert cfg.dm_list()[i] == p.dm == 17.0
    assert cfg.widths[j] == p.width == 4
    assert A[i, j] * cfg.widths[j] == p.t0 == 2000
    # closed form (SNR.5): P / sqrt(nchan*w*sigma_q^2 + P^2 (n-1)/n^2), P = A*nchan*w = 5120 -> 16.96
    assert 15.5 < S[i, j] < 18.5
    others = np.delete(S.max(axis=1), i)
    assert others.max() < S[i, j] - 3.0


# ----------------------------------------------------------------------------- all-cores leg
def test_all_cores_leg_equals_pure_python_brute_force_and_single_thread_leg():
    """oracle_mt.cpp only spreads rows over the cores: pinned to the pure-Python brute
    force on a tiny case, and bit-identical to the single-thread functions on cfg0 (direct, subband
    with a ragged coarse/fine grid, integrate + S/N with ddof 0 and 1)."""
    f, dms, ts, delay, X = small_case(11)
    assert oracle.dedisperse_mt(X, delay, 37).tolist() == py_dedisperse(X, delay.tolist(), 37)

    cfg = configs.tiny()
    d = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    Xc, _ = filterbank.make_filterbank(cfg, cfg.nsamp_out + int(d.max()))
    Y = oracle.dedisperse(Xc, d, cfg.nsamp_out)
    assert np.array_equal(oracle.dedisperse_mt(Xc, d, cfg.nsamp_out), Y)
    for ddof in (0, 1):
        P, S, A = oracle.search(Y, cfg.widths, ddof)
        Pm, Sm, Am = oracle.search_mt(Y, cfg.widths, ddof)
        assert all(np.array_equal(P[w], Pm[w]) for w in cfg.widths)
        assert np.array_equal(S, Sm) and np.array_equal(A, Am)
    A_dm, F_dm = 4.0 * np.arange(5), 0.5 * np.arange(7)
    d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, 8, A_dm, F_dm)
    ns = 3000
    S1 = oracle.subband_step1(Xc, d1, 8, ns + int(d2.max()))
    Y2 = oracle.subband_step2(S1, d2, ns)
    Sm, Ym = oracle.subband_mt(Xc, d1, d2, 8, ns)
    assert np.array_equal(S1, Sm) and np.array_equal(Y2, Ym)
    assert oracle.mt_threads() >= 1


# ----------------------------------------------------------------------------- INT.1s: sliding boxcar (8(f) f1)
def test_sliding_boxcar_closed_forms_and_relation_to_block_sums():
    """oracle.integrate_sliding against what fixes it: a constant series gives w*v, a single impulse gives a
    run of w copies ending at its position, numpy's cumulative-sum difference is the third implementation,
    and the block sums of oracle.integrate are its samples at multiples of w (INT.4 invariant)."""
    rng = np.random.default_rng(5)
    ns = 53
    c = np.full((2, ns), 7, dtype=np.uint32)
    for w in (1, 2, 3, 4, 8, 53):
        I = oracle.integrate_sliding(c, w)
        assert I.shape == (2, ns - w + 1) and (I == 7 * w).all()
    imp = np.zeros((1, ns), dtype=np.uint32)
    imp[0, 20] = 9
    for w in (1, 2, 4, 8):
        I = oracle.integrate_sliding(imp, w)[0]
        want = np.zeros(ns - w + 1, dtype=np.uint32)
        want[20 - w + 1: 21] = 9                      # windows t .. t+w-1 that contain sample 20
        assert np.array_equal(I, want)
    Y = rng.integers(0, 400000, size=(3, ns), dtype=np.uint32)
    cs = np.concatenate([np.zeros((3, 1), dtype=np.uint64), np.cumsum(Y.astype(np.uint64), axis=1)], axis=1)
    for w in (1, 2, 3, 4, 5, 8, 16, 32):
        I = oracle.integrate_sliding(Y, w)
        assert np.array_equal(I.astype(np.uint64), cs[:, w:] - cs[:, :-w])
        D = oracle.integrate(Y, w)
        assert np.array_equal(I[:, ::w][:, : D.shape[1]], D)      # decimated planes are a subset
    with pytest.raises(ValueError):
        oracle.integrate_sliding(Y, ns + 1)


def test_sliding_boxcar_recovers_a_misaligned_pulse_at_its_width():
    """SURVEY INT.1: with decimating block sums a width-4 pulse starting 1-2 samples off a multiple of 4 peaks
    at a narrower width; the stride-1 boxcar recovers width 4 and the true start sample."""
    import dataclasses
    base = configs.tiny()
    p = dataclasses.replace(base.fixed_pulses[0], t0=2002)
    cfg = dataclasses.replace(base, fixed_pulses=(p,))
    d = oracle.delay_table(cfg.chan_freq_mhz(), cfg.dm_list(), cfg.t_samp_s)
    X, pulses = filterbank.make_filterbank(cfg, cfg.nsamp_out + int(d.max()))
    assert pulses[0].t0 == 2002 and pulses[0].width == 4
    Y = oracle.dedisperse(X, d, cfg.nsamp_out)
    _, S, A = oracle.search_sliding(Y, cfg.widths)
    i, j = np.unravel_index(np.argmax(S), S.shape)
    assert cfg.dm_list()[i] == 17.0 and cfg.widths[j] == 4 and A[i, j] == 2002
    _, Sd, _ = oracle.search(Y, cfg.widths)
    id_, jd = np.unravel_index(np.argmax(Sd), Sd.shape)
    assert cfg.dm_list()[id_] == 17.0 and cfg.widths[jd] == 2     # decimation splits the pulse over two blocks
    assert S[i, j] > Sd[id_, jd]


# ----------------------------------------------------------------------------- DD.7m: channel mask (8(f) f4)
def test_masked_dedispersion_equals_dedispersion_of_the_kept_channels():
    """oracle.dedisperse_masked against the definitions that fix it: an all-ones mask is the plain sum; a
    masked channel contributes nothing whatever it holds; the result equals the pure-Python brute force over
    the kept channels only; and linearity: masked + complement = full."""
    f, dms, ts, delay, X = small_case(21, nchan=7, ndm=6, ns=41)
    full = oracle.dedisperse(X, delay, 41)
    assert np.array_equal(oracle.dedisperse_masked(X, np.ones(7, np.uint8), delay, 41), full)
    mask = np.array([1, 0, 1, 1, 0, 1, 1], dtype=np.uint8)
    got = oracle.dedisperse_masked(X, mask, delay, 41)
    keep = [c for c in range(7) if mask[c]]
    want = py_dedisperse([X[c] for c in keep], [[row[c] for c in keep] for row in delay.tolist()], 41)
    assert got.tolist() == want
    X2 = X.copy()
    X2[mask == 0] = 255                                  # what a zapped channel holds does not matter
    assert np.array_equal(oracle.dedisperse_masked(X2, mask, delay, 41), got)
    assert np.array_equal(got + oracle.dedisperse_masked(X, 1 - mask, delay, 41), full)
    assert (oracle.dedisperse_masked(X, np.zeros(7, np.uint8), delay, 41) == 0).all()


# ----------------------------------------------------------------------------- batches (8(f) f3)
def test_consecutive_batches_with_carried_samples_equal_one_long_dedispersion():
    """The paper searches consecutive batches of one observation ("10 batches").  Dedispersing
    batch b from samples [b*ns, b*ns + ns + max_delay) -- i.e. keeping the last max_delay samples of the
    previous upload and appending ns new ones -- gives exactly the columns [b*ns, (b+1)*ns) of one long
    dedispersion: pure-Python brute force on the long series is the reference."""
    f, dms, ts, delay, _ = small_case(31, nchan=5, ndm=4, ns=20)
    md = int(delay.max())
    nb, ns = 3, 20
    rng = np.random.default_rng(32)
    X = rng.integers(0, 256, size=(5, nb * ns + md), dtype=np.uint8)
    long_ = np.array(py_dedisperse(X, delay.tolist(), nb * ns), dtype=np.uint32)
    window = np.zeros((5, ns + md), dtype=np.uint8)
    for b in range(nb):
        if b == 0:
            window[:] = X[:, : ns + md]
        else:
            window[:, :md] = window[:, ns: ns + md].copy()      # carried tail of the previous batch
            window[:, md:] = X[:, b * ns + md: (b + 1) * ns + md]  # ns new samples
        Yb = oracle.dedisperse(np.ascontiguousarray(window), delay, ns)
        assert np.array_equal(Yb, long_[:, b * ns: (b + 1) * ns])
