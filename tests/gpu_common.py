"""Shared helpers of the `-m gpu` parity tests: run the CUDA path through the C ABI binding and
the oracle on the same seeded inputs (synth/), and compare.

The CUDA path and the oracle share only the input generator (synth/, data only).
"""
from __future__ import annotations

import json
import os

import numpy as np

import oracle
import paper_1811_04165_b200 as ddp
from synth import filterbank

SNR_RTOL = 1e-5  # BASELINE.json north_star: "SNR within 1e-5 relative"
TUNED_JSON = os.path.join(os.path.dirname(os.path.abspath(ddp.__file__)), "tuned_b200.json")


def tuned_shapes(workload):
    """{kernel name: gene list} of the workload in tuned_b200.json -- the shapes bench.py times."""
    with open(TUNED_JSON) as fh:
        return json.load(fh).get(workload, {})


def u32(t) -> np.ndarray:
    """torch int32-typed device tensor -> numpy uint32 host array."""
    return t.cpu().numpy().view(np.uint32)


class GpuSearch:
    """One plan + its device buffers + the uploaded synthetic filterbank of a SearchConfig."""

    def __init__(self, cfg, X: np.ndarray = None, device="cuda:0", **plan_kw):
        import torch
        self.torch = torch
        self.cfg = cfg
        self.plan = ddp.plan_from_config(cfg, **plan_kw)
        self.info = self.plan.query()
        self.buf = ddp.alloc_buffers(self.plan, device)
        i = self.info
        if X is None:
            X, self.pulses = filterbank.make_filterbank(cfg, int(i.nsamp_in_required), int(i.in_stride_min),
                                                        bits=int(i.input_bits))
        assert X.shape == (i.nchan, i.in_stride_min) and X.dtype == (np.uint8 if i.input_bits == 8 else np.uint16)
        self.X = X
        self.upload()

    def apply_tuned(self, workload):
        """Sets every kernel slot to its shape in tuned_b200.json (what bench.py runs); a shape that is
        not valid for the plan is a test failure, not a skip."""
        applied = {}
        for kname, genes in tuned_shapes(workload).items():
            k = ddp.KERNEL_NAMES.index(kname)
            c = ddp.Kcfg(*genes)
            assert self.plan.check_kcfg(k, c), "tuned %s %r is not valid for %s" % (kname, genes, workload)
            self.plan.set_kcfg(k, c)
            applied[kname] = genes
        return applied

    def upload(self):
        """Re-uploads self.X after the test changed it in place."""
        host = self.X if self.X.dtype == np.uint8 else self.X.view(np.int16)  # the device tensor is int16-typed
        self.buf["d_in"].copy_(self.torch.from_numpy(host))
        self.torch.cuda.synchronize()

    def dedisperse(self):
        self.plan.dedisperse(self.buf["d_in"], self.buf["d_out"])
        self.torch.cuda.synchronize()
        return u32(self.buf["d_out"])[:, : self.info.nsamp_out]

    def integrate(self):
        self.plan.integrate(self.buf["d_out"], self.buf["d_integ"])
        self.torch.cuda.synchronize()
        return self.planes()

    def planes(self):
        i = self.info
        flat = u32(self.buf["d_integ"])
        out = {}
        for k in range(i.nwidths):
            w = i.widths[k]
            if w == 1:
                continue
            off, st, n = i.plane_offset[k], i.plane_stride[k], i.plane_len[k]
            out[w] = flat[off: off + st * i.ndm].reshape(i.ndm, st)[:, :n]
        return out

    def snr(self):
        self.plan.snr(self.buf["d_out"], self.buf["d_integ"], self.buf["d_snr"], self.buf["d_argmax"])
        self.torch.cuda.synchronize()
        return self.buf["d_snr"].cpu().numpy(), u32(self.buf["d_argmax"])

    def run_all(self):
        Y = self.dedisperse()
        P = self.integrate()
        S, A = self.snr()
        return Y, P, S, A

    def subband_intermediate(self):
        """S[ncoarse][nsub][nsamp_sub] read back through the debug accessor."""
        import ctypes
        i = self.info
        n = i.n_coarse * i.n_subbands * i.sub_stride
        dt = {2: np.uint16, 4: np.uint32}[i.sub_elem_bytes]  # SB.4: narrow storage where exact
        ptr = self.plan.subband_buffer()
        assert ptr
        # the buffer lives inside the torch workspace tensor: find its offset there
        base = self.buf["workspace"].data_ptr()
        off = ptr - base
        host = self.buf["workspace"][off: off + n * i.sub_elem_bytes].cpu().numpy().view(dt).astype(np.uint32)
        return host.reshape(i.n_coarse, i.n_subbands, i.sub_stride)[:, :, : i.nsamp_sub]

    def close(self):
        self.plan.destroy()


# ---------------------------------------------------------------------------- oracle legs
def oracle_direct_rows(cfg, X, rows=None):
    """Oracle dedispersion of the given DM rows (all when None) -> uint32 [nrows][ns]."""
    dms = cfg.dm_list()
    if rows is not None:
        dms = dms[np.asarray(rows)]
    delay = oracle.delay_table(cfg.chan_freq_mhz(), dms, cfg.t_samp_s)
    return oracle.dedisperse(np.ascontiguousarray(X), delay, cfg.nsamp_out)


def oracle_subband(cfg, X, coarse_rows=None, ref="top"):
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    if coarse_rows is not None:
        A = A[np.asarray(coarse_rows)]
    d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F, ref=ref)
    ns1 = cfg.nsamp_out + int(d2.max())
    S = oracle.subband_step1(np.ascontiguousarray(X), d1, sb.n_subbands, ns1)
    Y = oracle.subband_step2(S, d2, cfg.nsamp_out)
    return S, Y


def oracle_search(Y, widths, ddof=0):
    return oracle.search(np.ascontiguousarray(Y), widths, ddof)


# all-cores legs (oracle_mt.cpp: the same single-thread functions, rows spread over the host cores) --
# what makes every row of the full-size configs affordable
def oracle_direct_all_rows_mt(cfg, X, rows=None):
    dms = cfg.dm_list()
    if rows is not None:
        dms = dms[np.asarray(rows)]
    delay = oracle.delay_table(cfg.chan_freq_mhz(), dms, cfg.t_samp_s)
    return oracle.dedisperse_mt(np.ascontiguousarray(X), delay, cfg.nsamp_out)


def oracle_subband_mt(cfg, X):
    sb = cfg.subband
    A = sb.coarse_first + sb.coarse_step * np.arange(sb.n_coarse)
    F = sb.fine_step * np.arange(sb.n_fine)
    d1, d2 = oracle.subband_tables(cfg.chan_freq_mhz(), cfg.t_samp_s, sb.n_subbands, A, F)
    return oracle.subband_mt(np.ascontiguousarray(X), d1, d2, sb.n_subbands, cfg.nsamp_out)


def assert_snr_close(gpu, ref, what=""):
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    tol = SNR_RTOL * np.maximum(1.0, np.abs(ref))
    bad = np.abs(gpu - ref) > tol
    assert not bad.any(), "%s S/N mismatch at %s: gpu %s oracle %s" % (
        what, np.argwhere(bad)[:5].tolist(), gpu[bad][:5], ref[bad][:5])


def compare_all(g: GpuSearch, Yo, rows=None, what="", ddof=0, mt=False):
    """Full element-by-element comparison of the CUDA results (already computed in g's buffers)
    against the oracle chain applied to the oracle's own dedispersed rows Yo."""
    i = g.info
    widths = [i.widths[k] for k in range(i.nwidths)]
    Yg = u32(g.buf["d_out"])[:, : i.nsamp_out]
    Pg = g.planes()
    Sg, Ag = g.buf["d_snr"].cpu().numpy(), u32(g.buf["d_argmax"])
    if rows is not None:
        rows = np.asarray(rows)
        Yg, Sg, Ag = Yg[rows], Sg[rows], Ag[rows]
        Pg = {w: p[rows] for w, p in Pg.items()}
    assert Yg.shape == Yo.shape
    assert np.array_equal(Yg, Yo), "%s dedispersion differs (bit-exact required)" % what
    Po, So, Ao = (oracle.search_mt if mt else oracle.search)(np.ascontiguousarray(Yo), widths, ddof)
    for w in widths:
        if w > 1:
            assert np.array_equal(Pg[w], Po[w]), "%s integration plane w=%d differs" % (what, w)
    assert_snr_close(Sg, So, what)
    assert np.array_equal(Ag, Ao), "%s argmax differs" % what
