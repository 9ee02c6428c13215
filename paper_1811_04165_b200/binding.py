"""Thin ctypes binding of libddp (include/ddp.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; nothing here computes.  PyTorch
tensors (or raw integer device pointers) supply device memory and streams.  The library must have
been built in-tree (`python -m paper_1811_04165_b200.build`); importing this module without it
raises -- there is no fallback of any kind.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libddp.so")
KCACHE_DIR = os.path.join(_HERE, "kcache")

DDP_MAX_WIDTHS = 16
DDP_NSLOTS = 4
K_DIRECT, K_SUB1, K_SUB2, K_INTEGRATE, K_SNR, K_ISNR = 0, 1, 2, 3, 4, 5
KERNEL_NAMES = ("direct", "sub1", "sub2", "integrate", "snr", "isnr")
STAGE_DIRECT, STAGE_SMEM, STAGE_TMA = 0, 1, 2
E_ARG, E_SHAPE, E_OVERFLOW, E_WORKSPACE, E_CONFIG, E_COMPILE, E_CUDA, E_BUDGET = -1, -2, -3, -4, -5, -6, -7, -8

# every symbol include/ddp.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "ddp_plan_create", "ddp_plan_destroy", "ddp_plan_query", "ddp_plan_get_delays",
    "ddp_plan_bind_workspace", "ddp_dedisperse", "ddp_integrate", "ddp_snr", "ddp_integrate_snr", "ddp_search_host", "ddp_search_host_batches",
    "ddp_plan_subband_buffer", "ddp_get_kcfg", "ddp_set_kcfg", "ddp_check_kcfg", "ddp_repair_kcfg",
    "ddp_compile_kcfg", "ddp_enumerate_kcfgs", "ddp_tune_ga", "ddp_tune_bruteforce",
    "ddp_tune_random", "ddp_time_pipeline", "ddp_status_str", "ddp_last_error", "ddp_version",
)


class DdpError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        super().__init__("%s failed: status %d (%s)%s" % (what, status, status_str(status),
                                                           (": " + detail) if detail else ""))


class Kcfg(C.Structure):
    _fields_ = [(n, C.c_int) for n in ("threads_t", "threads_dm", "samples_per_thread", "dms_per_thread",
                                       "unroll", "staging", "vec_bytes")]

    def astuple(self):
        return tuple(getattr(self, n) for n, _ in self._fields_)

    def __repr__(self):
        return "Kcfg(tt=%d, tdm=%d, spt=%d, dpt=%d, unroll=%d, staging=%d, vec=%d)" % self.astuple()

    def copy(self):
        return Kcfg(*self.astuple())


class Options(C.Structure):
    _fields_ = [("n_subbands", C.c_int), ("n_coarse", C.c_int), ("coarse_dm_first", C.c_double),
                ("coarse_dm_step", C.c_double), ("n_fine", C.c_int), ("fine_dm_step", C.c_double),
                ("snr_ddof", C.c_int), ("device", C.c_int), ("cache_dir", C.c_char_p), ("integration_mode", C.c_int),
                ("chan_mask", C.c_void_p), ("subband_ref", C.c_int), ("input_bits", C.c_int)]


class PlanInfo(C.Structure):
    _fields_ = [("subband", C.c_int), ("nchan", C.c_int), ("ndm", C.c_int), ("nwidths", C.c_int),
                ("nsamp_out", C.c_int), ("n_subbands", C.c_int), ("n_coarse", C.c_int), ("n_fine", C.c_int),
                ("max_delay", C.c_int), ("max_d1", C.c_int), ("max_d2", C.c_int),
                ("nsamp_in_required", C.c_int64), ("in_stride_min", C.c_int64), ("out_stride_min", C.c_int64),
                ("nsamp_sub", C.c_int64), ("sub_stride", C.c_int64),
                ("widths", C.c_int * DDP_MAX_WIDTHS), ("plane_len", C.c_int64 * DDP_MAX_WIDTHS),
                ("plane_stride", C.c_int64 * DDP_MAX_WIDTHS), ("plane_offset", C.c_int64 * DDP_MAX_WIDTHS),
                ("integ_elems", C.c_int64), ("workspace_bytes", C.c_int64), ("adds_dedisp", C.c_double),
                ("sub_elem_bytes", C.c_int), ("integration_mode", C.c_int), ("nchan_masked", C.c_int),
                ("subband_ref", C.c_int), ("input_bits", C.c_int)]


FITNESS_FN = C.CFUNCTYPE(C.c_double, C.c_void_p, C.POINTER(Kcfg))


class TuneIo(C.Structure):
    _fields_ = [("d_in", C.c_void_p), ("in_stride", C.c_size_t), ("d_out", C.c_void_p), ("out_stride", C.c_size_t),
                ("d_integ", C.c_void_p), ("d_snr", C.c_void_p), ("d_argmax", C.c_void_p), ("stream", C.c_void_p),
                ("d_flush", C.c_void_p), ("flush_bytes", C.c_size_t), ("fitness", FITNESS_FN), ("user", C.c_void_p),
                ("reps", C.c_int), ("warmup", C.c_int), ("cutoff_factor", C.c_double)]


class GaParams(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("population", C.c_int), ("generations", C.c_int), ("tournament", C.c_int),
                ("p_cross", C.c_double), ("crossover_kind", C.c_int), ("p_mut", C.c_double),
                ("mutation_kind", C.c_int), ("elitism", C.c_int), ("replacement", C.c_int),
                ("max_evals", C.c_int64)]


class BfParams(C.Structure):
    _fields_ = [("max_evals_per_kernel", C.c_int64), ("isolated", C.c_int), ("slots", C.c_uint)]


class RandParams(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("max_evals", C.c_int64)]


class TuneResult(C.Structure):
    _fields_ = [("best", Kcfg * DDP_NSLOTS), ("best_ms", C.c_double), ("kernel_ms", C.c_double * DDP_NSLOTS),
                ("n_fitness_calls", C.c_int64), ("n_kernel_timings", C.c_int64), ("n_compiles", C.c_int64),
                ("wall_seconds", C.c_double), ("history", C.POINTER(C.c_double)), ("history_cap", C.c_size_t),
                ("history_len", C.c_size_t), ("sum_isolated_min_ms", C.c_double),
                ("final_pop", C.POINTER(Kcfg)), ("final_fit", C.POINTER(C.c_double)), ("final_cap", C.c_size_t),
                ("final_len", C.c_size_t)]


_lib = None


def lib():
    """The loaded C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libddp.so is missing at %s -- build it with "
                              "`python -m paper_1811_04165_b200.build` (there is no fallback path)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, st = C.c_void_p, C.c_int
        L.ddp_plan_create.argtypes = [C.POINTER(vp), vp, C.c_int, C.c_double, vp, C.c_int, vp, C.c_int, C.c_int,
                                      C.POINTER(Options)]
        L.ddp_plan_destroy.argtypes = [vp]
        L.ddp_plan_query.argtypes = [vp, C.POINTER(PlanInfo)]
        L.ddp_plan_get_delays.argtypes = [vp, C.c_int, vp]
        L.ddp_plan_bind_workspace.argtypes = [vp, vp, C.c_size_t, vp]
        L.ddp_dedisperse.argtypes = [vp, vp, C.c_size_t, vp, C.c_size_t, vp]
        L.ddp_integrate.argtypes = [vp, vp, C.c_size_t, vp, vp]
        L.ddp_snr.argtypes = [vp, vp, C.c_size_t, vp, vp, vp, vp]
        L.ddp_integrate_snr.argtypes = [vp, vp, C.c_size_t, vp, vp, vp, vp]
        L.ddp_search_host.argtypes = [vp, vp, C.c_size_t, vp, vp, C.c_size_t, vp, vp, vp, vp, vp, vp]
        L.ddp_search_host_batches.argtypes = [vp, vp, C.c_size_t, C.c_int, vp, vp, C.c_size_t, vp, C.c_size_t, vp, vp, vp,
                                              vp, vp]
        L.ddp_plan_subband_buffer.argtypes = [vp, C.POINTER(vp)]
        for f in ("ddp_get_kcfg", "ddp_set_kcfg", "ddp_check_kcfg", "ddp_repair_kcfg", "ddp_compile_kcfg"):
            getattr(L, f).argtypes = [vp, C.c_int, C.POINTER(Kcfg)]
        L.ddp_enumerate_kcfgs.argtypes = [vp, C.c_int, C.POINTER(Kcfg), C.c_size_t, C.POINTER(C.c_size_t)]
        L.ddp_tune_ga.argtypes = [vp, C.POINTER(TuneIo), C.POINTER(GaParams), C.POINTER(TuneResult)]
        L.ddp_tune_bruteforce.argtypes = [vp, C.POINTER(TuneIo), C.POINTER(BfParams), C.POINTER(TuneResult)]
        L.ddp_tune_random.argtypes = [vp, C.POINTER(TuneIo), C.POINTER(RandParams), C.POINTER(TuneResult)]
        L.ddp_time_pipeline.argtypes = [vp, C.POINTER(TuneIo), C.POINTER(Kcfg), C.POINTER(C.c_double),
                                        C.POINTER(C.c_double)]
        for name in SYMBOLS:
            getattr(L, name).restype = st
        L.ddp_status_str.argtypes = [C.c_int]
        L.ddp_status_str.restype = C.c_char_p
        L.ddp_last_error.argtypes = [vp]
        L.ddp_last_error.restype = C.c_char_p
        L.ddp_version.argtypes = []
        L.ddp_version.restype = C.c_char_p
        _lib = L
    return _lib


def status_str(status: int) -> str:
    return lib().ddp_status_str(status).decode()


def version() -> str:
    return lib().ddp_version().decode()


def _ptr(x) -> Optional[int]:
    """Device/host address of a tensor-like (torch tensor, numpy array) or a raw int; None -> NULL."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return int(x.data_ptr())


def _row_stride(x, given: Optional[int]) -> int:
    if given is not None:
        return int(given)
    if isinstance(x, np.ndarray):
        return x.strides[0] // x.itemsize
    return int(x.stride(0))


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream) or None
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream) or None


class Plan:
    """Owner of one ddp_plan*; methods mirror the C entry points one to one."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)
        self._keep = []  # tensors the C side points into (workspace)

    # ---- helpers
    def _check(self, status: int, what: str):
        if status != 0:
            raise DdpError(status, what, lib().ddp_last_error(self._h).decode(errors="replace"))

    def destroy(self):
        if self._h:
            lib().ddp_plan_destroy(self._h)
            self._h = C.c_void_p(None)
            self._keep = []

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- geometry
    def query(self) -> PlanInfo:
        info = PlanInfo()
        self._check(lib().ddp_plan_query(self._h, C.byref(info)), "ddp_plan_query")
        return info

    def get_delays(self, step: int = 0) -> np.ndarray:
        i = self.query()
        shape = {0: (i.ndm, i.nchan), 1: (i.n_coarse, i.nchan), 2: (i.n_fine, i.n_subbands)}[step]
        out = np.empty(shape, dtype=np.int32)
        self._check(lib().ddp_plan_get_delays(self._h, step, out.ctypes.data), "ddp_plan_get_delays")
        return out

    def bind_workspace(self, d_workspace, nbytes: Optional[int] = None, stream=None):
        if nbytes is None:
            nbytes = d_workspace.numel() * d_workspace.element_size()
        self._check(lib().ddp_plan_bind_workspace(self._h, _ptr(d_workspace), nbytes, _stream(stream)),
                    "ddp_plan_bind_workspace")
        self._keep = [d_workspace]

    def subband_buffer(self) -> int:
        p = C.c_void_p()
        self._check(lib().ddp_plan_subband_buffer(self._h, C.byref(p)), "ddp_plan_subband_buffer")
        return p.value or 0

    # ---- compute
    def dedisperse(self, d_in, d_out, in_stride=None, out_stride=None, stream=None):
        self._check(lib().ddp_dedisperse(self._h, _ptr(d_in), _row_stride(d_in, in_stride), _ptr(d_out),
                                         _row_stride(d_out, out_stride), _stream(stream)), "ddp_dedisperse")

    def integrate(self, d_dedisp, d_integ, stride=None, stream=None):
        self._check(lib().ddp_integrate(self._h, _ptr(d_dedisp), _row_stride(d_dedisp, stride), _ptr(d_integ),
                                        _stream(stream)), "ddp_integrate")

    def snr(self, d_dedisp, d_integ, d_snr, d_argmax=None, stride=None, stream=None):
        self._check(lib().ddp_snr(self._h, _ptr(d_dedisp), _row_stride(d_dedisp, stride), _ptr(d_integ),
                                  _ptr(d_snr), _ptr(d_argmax), _stream(stream)), "ddp_snr")

    def integrate_snr(self, d_dedisp, d_snr, d_argmax=None, d_integ=None, stride=None, stream=None):
        """Fused integration + S/N; the planes are written only when d_integ is given."""
        self._check(lib().ddp_integrate_snr(self._h, _ptr(d_dedisp), _row_stride(d_dedisp, stride), _ptr(d_integ),
                                            _ptr(d_snr), _ptr(d_argmax), _stream(stream)), "ddp_integrate_snr")

    def search_host(self, h_in, d_in, d_out, d_integ, d_snr, d_argmax, h_snr, h_argmax=None, stream=None):
        self._check(lib().ddp_search_host(self._h, _ptr(h_in), _row_stride(h_in, None), _ptr(d_in), _ptr(d_out),
                                          _row_stride(d_out, None), _ptr(d_integ), _ptr(d_snr), _ptr(d_argmax),
                                          _ptr(h_snr), _ptr(h_argmax), _stream(stream)), "ddp_search_host")

    def search_host_batches(self, h_in, nbatches, d_in0, d_in1, d_out, d_snr, d_argmax, h_snr, h_argmax=None,
                            stream=None):
        """Consecutive batches of one observation: h_in [nchan][>= nbatches*ns + max_delay], results [nbatches][ndm][nW]."""
        self._check(lib().ddp_search_host_batches(self._h, _ptr(h_in), _row_stride(h_in, None), int(nbatches),
                                                  _ptr(d_in0), _ptr(d_in1), _row_stride(d_in0, None), _ptr(d_out),
                                                  _row_stride(d_out, None), _ptr(d_snr), _ptr(d_argmax), _ptr(h_snr),
                                                  _ptr(h_argmax), _stream(stream)), "ddp_search_host_batches")

    # ---- kernel configurations
    def get_kcfg(self, k: int) -> Kcfg:
        c = Kcfg()
        self._check(lib().ddp_get_kcfg(self._h, k, C.byref(c)), "ddp_get_kcfg")
        return c

    def set_kcfg(self, k: int, cfg: Kcfg):
        self._check(lib().ddp_set_kcfg(self._h, k, C.byref(cfg)), "ddp_set_kcfg")

    def check_kcfg(self, k: int, cfg: Kcfg) -> bool:
        return lib().ddp_check_kcfg(self._h, k, C.byref(cfg)) == 0

    def repair_kcfg(self, k: int, cfg: Kcfg) -> Kcfg:
        c = cfg.copy()
        self._check(lib().ddp_repair_kcfg(self._h, k, C.byref(c)), "ddp_repair_kcfg")
        return c

    def compile_kcfg(self, k: int, cfg: Kcfg):
        self._check(lib().ddp_compile_kcfg(self._h, k, C.byref(cfg)), "ddp_compile_kcfg")

    def enumerate_kcfgs(self, k: int) -> List[Kcfg]:
        n = C.c_size_t(0)
        self._check(lib().ddp_enumerate_kcfgs(self._h, k, None, 0, C.byref(n)), "ddp_enumerate_kcfgs")
        arr = (Kcfg * max(1, n.value))()
        self._check(lib().ddp_enumerate_kcfgs(self._h, k, arr, n.value, C.byref(n)), "ddp_enumerate_kcfgs")
        return [arr[i].copy() for i in range(n.value)]

    # ---- tuning
    def _result(self, history_cap: int, final_cap: int = 0):
        res = TuneResult()
        hist = (C.c_double * max(1, history_cap))()
        res.history = C.cast(hist, C.POINTER(C.c_double))
        res.history_cap = history_cap
        if final_cap > 0:  # the configurations the run ends with
            res._final_pop = (Kcfg * (final_cap * DDP_NSLOTS))()
            res._final_fit = (C.c_double * final_cap)()
            res.final_pop = C.cast(res._final_pop, C.POINTER(Kcfg))
            res.final_fit = C.cast(res._final_fit, C.POINTER(C.c_double))
            res.final_cap = final_cap
        return res, hist

    @staticmethod
    def _pack(res: TuneResult, hist) -> dict:
        return {"best": [res.best[i].copy() for i in range(DDP_NSLOTS)], "best_ms": res.best_ms,
                "kernel_ms": list(res.kernel_ms), "n_fitness_calls": res.n_fitness_calls,
                "n_kernel_timings": res.n_kernel_timings, "n_compiles": res.n_compiles,
                "wall_seconds": res.wall_seconds, "history": [hist[i] for i in range(res.history_len)],
                "sum_isolated_min_ms": res.sum_isolated_min_ms,
                "final": [([res._final_pop[i * DDP_NSLOTS + s].copy() for s in range(DDP_NSLOTS)], res._final_fit[i])
                          for i in range(res.final_len)] if res.final_cap else []}

    def tune_ga(self, io: TuneIo, seed=1, population=64, generations=50, tournament=3, p_cross=0.8,
                crossover_kind=0, p_mut=0.05, mutation_kind=0, elitism=2, replacement=0, max_evals=0,
                history_cap=1 << 16, final_cap=0) -> dict:
        gp = GaParams(seed, population, generations, tournament, p_cross, crossover_kind, p_mut, mutation_kind,
                      elitism, replacement, max_evals)
        res, hist = self._result(history_cap, final_cap)
        self._check(lib().ddp_tune_ga(self._h, C.byref(io), C.byref(gp), C.byref(res)), "ddp_tune_ga")
        return self._pack(res, hist)

    def tune_bruteforce(self, io: TuneIo, max_evals_per_kernel=0, isolated=0, slots=0, history_cap=1 << 18) -> dict:
        bp = BfParams(max_evals_per_kernel, isolated, slots)
        res, hist = self._result(history_cap)
        self._check(lib().ddp_tune_bruteforce(self._h, C.byref(io), C.byref(bp), C.byref(res)),
                    "ddp_tune_bruteforce")
        return self._pack(res, hist)

    def tune_random(self, io: TuneIo, seed=1, max_evals=1000, history_cap=1 << 16, final_cap=0) -> dict:
        rp = RandParams(seed, max_evals)
        res, hist = self._result(history_cap, final_cap)
        self._check(lib().ddp_tune_random(self._h, C.byref(io), C.byref(rp), C.byref(res)), "ddp_tune_random")
        return self._pack(res, hist)

    def time_pipeline(self, io: TuneIo, cfgs: Sequence[Kcfg]):
        arr = (Kcfg * DDP_NSLOTS)(*[c.copy() for c in cfgs])
        ms = C.c_double(0.0)
        per = (C.c_double * DDP_NSLOTS)()
        self._check(lib().ddp_time_pipeline(self._h, C.byref(io), arr, C.byref(ms), per), "ddp_time_pipeline")
        return ms.value, list(per)


def plan_create(chan_freq_mhz, t_samp_s: float, dm_list, widths, nsamp_out: int, *, n_subbands: int = 0,
                n_coarse: int = 0, coarse_dm_first: float = 0.0, coarse_dm_step: float = 0.0, n_fine: int = 0,
                fine_dm_step: float = 0.0, snr_ddof: int = 0, device: int = 0,
                cache_dir: Optional[str] = KCACHE_DIR, integration_mode: int = 0, chan_mask=None,
                subband_ref: int = 0, input_bits: int = 8) -> Plan:
    f = np.ascontiguousarray(chan_freq_mhz, dtype=np.float64)
    w = np.ascontiguousarray(widths, dtype=np.int32)
    dm = None if dm_list is None else np.ascontiguousarray(dm_list, dtype=np.float64)
    if cache_dir:
        os.makedirs(cache_dir, exist_ok=True)
    mask = None if chan_mask is None else np.ascontiguousarray(chan_mask, dtype=np.uint8)
    if mask is not None and mask.size != f.size:
        raise ValueError("chan_mask needs one byte per channel")
    opt = Options(n_subbands, n_coarse, coarse_dm_first, coarse_dm_step, n_fine, fine_dm_step, snr_ddof, device,
                  cache_dir.encode() if cache_dir else None, int(integration_mode),
                  None if mask is None else mask.ctypes.data, int(subband_ref), int(input_bits))
    h = C.c_void_p()
    st = lib().ddp_plan_create(C.byref(h), f.ctypes.data, f.size, float(t_samp_s),
                               None if dm is None else dm.ctypes.data, 0 if dm is None else dm.size,
                               w.ctypes.data, w.size, int(nsamp_out), C.byref(opt))
    if st != 0:
        raise DdpError(st, "ddp_plan_create")
    return Plan(h.value)


def make_tune_io(d_in=None, d_out=None, d_integ=None, d_snr=None, d_argmax=None, stream=None, d_flush=None,
                 fitness=None, reps: int = 5, warmup: int = 1, cutoff_factor: float = 0.0) -> TuneIo:
    io = TuneIo()
    if d_in is not None:
        io.d_in, io.in_stride = _ptr(d_in), _row_stride(d_in, None)
        io.d_out, io.out_stride = _ptr(d_out), _row_stride(d_out, None)
        io.d_integ, io.d_snr, io.d_argmax = _ptr(d_integ), _ptr(d_snr), _ptr(d_argmax)
        io.stream = _stream(stream)
        if d_flush is not None:
            io.d_flush, io.flush_bytes = _ptr(d_flush), d_flush.numel() * d_flush.element_size()
    if fitness is not None:
        io.fitness = fitness if isinstance(fitness, FITNESS_FN) else FITNESS_FN(fitness)
        io._keep_fitness = io.fitness
    io.reps, io.warmup, io.cutoff_factor = reps, warmup, cutoff_factor
    return io
