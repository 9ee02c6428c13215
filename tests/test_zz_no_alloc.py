"""The allocation-free entry point (include/ddp_static.h, libddp_static.so): two-step subband dedispersion whose
intermediate lives in a `static __device__` array inside the library.

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a
failure here must not hide the tests of the main path.  The GPU test compares the new entry point with the EXISTING
path (`ddp_dedisperse` on a subband plan, itself checked against the oracle in test_gpu_parity.py), bit for bit --
the sums are integers, which is the tolerance every dedispersion test here uses -- on calls in a row that share the
scratch array: a small plan, a plan whose intermediate does not fit the array at once (coarse trials in groups), and
the small plan again on top of the larger one's leftovers.
"""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_1811_04165_b200 import static_entry

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_static_library_exports_every_declared_symbol_and_states_its_limit():
    text = open(os.path.join(ROOT, "include", "ddp_static.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(ddp_static_[a-z_0-9]+)\s*\(", code))
    assert declared == set(static_entry.SYMBOLS)
    L = ctypes.CDLL(static_entry.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(L, name), "libddp_static.so does not export %s" % name
    m = re.search(r"#define\s+DDP_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", text)
    assert m and static_entry.scratch_bytes() == int(m.group(1)) << int(m.group(2)) == 16 << 20
    # the product sources of this entry point call no allocator
    src = open(os.path.join(ROOT, "paper_1811_04165_b200", "csrc", "ddp_static.cu")).read()
    src = re.sub(r"//[^\n]*", "", src)
    assert not re.search(r"cudaMalloc|cudaFree|cuMemAlloc|cuMemFree|\bmalloc\s*\(|\bnew\b", src)
    assert "cudaGetSymbolAddress" in src and "static __device__ __align__(256)" in src


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def _subband_cfg(name, nchan, nsamp_out, n_sub, n_coarse, n_fine, coarse_step=8.0, fine_step=0.25):
    from synth import configs
    from synth.configs import SubbandPlan
    return configs.scaled(configs.apertif_direct(), name=name, nchan=nchan, nsamp_out=nsamp_out, ndm=n_coarse * n_fine,
                          widths=(1, 2, 4), n_pulses=2,
                          subband=SubbandPlan(n_subbands=n_sub, n_coarse=n_coarse, coarse_first=0.0, coarse_step=coarse_step,
                                              n_fine=n_fine, fine_step=fine_step))


class _Case:
    """One subband plan, its input on the device, the existing path's result, and the tables the new call takes."""

    def __init__(self, cfg):
        import torch
        import paper_1811_04165_b200 as ddp
        from synth import filterbank
        self.cfg = cfg
        self.plan = ddp.plan_from_config(cfg)
        self.info = i = self.plan.query()
        self.buf = ddp.alloc_buffers(self.plan, "cuda:0")
        X, _ = filterbank.make_filterbank(cfg, int(i.nsamp_in_required), int(i.in_stride_min))
        self.buf["d_in"].copy_(torch.from_numpy(X))
        self.d1 = torch.from_numpy(np.ascontiguousarray(self.plan.get_delays(1), dtype=np.int32)).cuda()
        self.d2 = torch.from_numpy(np.ascontiguousarray(self.plan.get_delays(2), dtype=np.int32)).cuda()
        self.plan.dedisperse(self.buf["d_in"], self.buf["d_out"])
        torch.cuda.synchronize()
        self.expect = self.buf["d_out"].cpu().numpy().view(np.uint32)[:, : i.nsamp_out].copy()
        self.out = torch.full_like(self.buf["d_out"], -1)  # preallocated: the call under test allocates nothing

    def run_static(self):
        import torch
        i = self.info
        self.out.fill_(-1)
        static_entry.subband_dedisperse(self.buf["d_in"], self.d1, i.max_d1, self.d2, i.max_d2, i.nsamp_out, self.out)
        torch.cuda.synchronize()
        return self.out.cpu().numpy().view(np.uint32)

    def check(self, what):
        got = self.run_static()
        ns = self.info.nsamp_out
        assert np.array_equal(got[:, :ns], self.expect), "%s: static-scratch result differs from ddp_dedisperse" % what
        assert np.all(got[:, ns:] == 0xFFFFFFFF), "%s: columns >= nsamp_out were written" % what


@pytest.mark.gpu
@pytest.mark.skipif(not _has_gpu(), reason="no CUDA device")
def test_static_scratch_subband_dedispersion_equals_the_plan_path_on_calls_in_a_row():
    import torch
    small = _Case(_subband_cfg("static_small", nchan=96, nsamp_out=2500, n_sub=8, n_coarse=6, n_fine=5))
    # 40 coarse trials x 16 subbands x 8 288 samples x 4 bytes = 21 MB: more than the 16 MiB array -> groups of coarse trials
    large = _Case(_subband_cfg("static_large", nchan=128, nsamp_out=8200, n_sub=16, n_coarse=40, n_fine=8, coarse_step=4.0))
    per_coarse = large.info.n_subbands * ((large.info.nsamp_out + large.info.max_d2 + 32 + 31) // 32 * 32) * 4
    assert per_coarse * large.info.n_coarse > static_entry.scratch_bytes() >= per_coarse
    before = torch.cuda.memory_allocated()
    small.check("first call")
    small.check("second call, same plan")
    large.check("third call, larger plan in groups")
    small.check("fourth call, on top of the larger plan's leftovers")
    large.check("fifth call")
    assert torch.cuda.memory_allocated() == before  # nothing was allocated through torch's allocator either
    # a side stream
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        small.check("side stream")
    small.plan.destroy()
    large.plan.destroy()


@pytest.mark.gpu
@pytest.mark.skipif(not _has_gpu(), reason="no CUDA device")
def test_static_scratch_rejects_what_does_not_fit_and_bad_shapes():
    import torch
    n_sub, ns = 64, 70000  # 64 subbands x 70 048 samples x 4 bytes = 17.9 MB for ONE coarse trial
    d_in = torch.zeros((n_sub, 70048), dtype=torch.uint8, device="cuda:0")
    d1 = torch.zeros((1, n_sub), dtype=torch.int32, device="cuda:0")
    d2 = torch.zeros((1, n_sub), dtype=torch.int32, device="cuda:0")
    out = torch.zeros((1, ns), dtype=torch.int32, device="cuda:0")
    with pytest.raises(static_entry.DdpStaticError) as e:
        static_entry.subband_dedisperse(d_in, d1, 0, d2, 0, ns, out)
    assert e.value.status == static_entry.E_TOO_LARGE and "static scratch holds" in str(e.value)
    with pytest.raises(static_entry.DdpStaticError) as e:  # input rows shorter than nsamp_out + delays + slack
        static_entry.subband_dedisperse(d_in, d1, 100, d2, 0, ns, out)
    assert e.value.status == static_entry.E_SHAPE
    d1_bad = torch.zeros((1, 60), dtype=torch.int32, device="cuda:0")
    with pytest.raises(ValueError):
        static_entry.subband_dedisperse(d_in, d1_bad, 0, d2, 0, ns, out)
    d2_bad = torch.zeros((1, 7), dtype=torch.int32, device="cuda:0")  # 7 subbands do not divide 64 channels
    with pytest.raises(static_entry.DdpStaticError) as e:
        static_entry.subband_dedisperse(d_in, d1, 0, d2_bad, 0, 1000, out)
    assert e.value.status == static_entry.E_ARG
    torch.cuda.synchronize()
