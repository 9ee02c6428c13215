"""ORACLE -- test infrastructure only (see oracle.cpp header).

Thin ctypes/numpy wrapper around `oracle.cpp`.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s cpu_baseline / `--impl reference` legs may import this package; nothing under
`paper_1811_04165_b200/` does, and this package imports nothing from there.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_SRC_MT = os.path.join(_HERE, "oracle_mt.cpp")
_LIB_MT = os.path.join(_HERE, "liboracle_mt.so")
_lib = None
_lib_mt = None


def build(force: bool = False) -> str:
    """Compile oracle.cpp with g++ (plain -O2, no contraction, single thread)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC",
                               _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    # the all-cores leg: oracle.cpp (unchanged) + oracle_mt.cpp (omp parallel for over rows)
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_MT))
    if force or not os.path.exists(_LIB_MT) or os.path.getmtime(_LIB_MT) < newest:
        tmp = _LIB_MT + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, _SRC_MT, "-o", tmp])
        os.replace(tmp, _LIB_MT)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def _load_mt():
    global _lib_mt
    if _lib_mt is None:
        build()
        _lib_mt = ctypes.CDLL(_LIB_MT)
    return _lib_mt


def mt_threads() -> int:
    """Threads the all-cores leg uses (OpenMP default: one per host core unless OMP_NUM_THREADS says otherwise)."""
    return int(_load_mt().oracle_mt_threads())


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def delay_table(f_mhz, dm, t_samp_s: float, f_ref_mhz: Optional[float] = None) -> np.ndarray:
    """int32 [ndm][nchan]; f_ref defaults to max f (DD.3)."""
    f = np.ascontiguousarray(f_mhz, dtype=np.float64)
    d = np.ascontiguousarray(dm, dtype=np.float64)
    if f_ref_mhz is None:
        f_ref_mhz = float(f.max())
    out = np.empty((d.size, f.size), dtype=np.int32)
    rc = _load().oracle_delay_table(_p(f), ctypes.c_int(f.size), ctypes.c_double(f_ref_mhz), _p(d),
                                    ctypes.c_int(d.size), ctypes.c_double(t_samp_s), _p(out))
    if rc != 0:
        raise ValueError("oracle_delay_table rc=%d" % rc)
    return out


def dedisperse(X: np.ndarray, delay: np.ndarray, ns: int) -> np.ndarray:
    """uint32 [nrows][ns] for the delay rows given (X: uint8, or uint16 for INPUT_BITS = 16, [nchan][in_stride])."""
    assert X.dtype in (np.uint8, np.uint16) and X.ndim == 2 and X.flags.c_contiguous
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nrows, nchan = delay.shape
    assert nchan == X.shape[0]
    Y = np.empty((nrows, ns), dtype=np.uint32)
    fn = _load().oracle_dedisperse if X.dtype == np.uint8 else _load().oracle_dedisperse_u16
    rc = fn(_p(X), ctypes.c_int(nchan), ctypes.c_size_t(X.shape[1]), _p(delay),
                                   ctypes.c_int(nrows), ctypes.c_int(ns), _p(Y), ctypes.c_size_t(ns))
    if rc != 0:
        raise ValueError("oracle_dedisperse rc=%d (input too short for the delays?)" % rc)
    return Y


def subband_step1(X: np.ndarray, d1: np.ndarray, nsub: int, ns1: int) -> np.ndarray:
    """uint32 S[ncoarse][nsub][ns1] (X: uint8, or uint16 for INPUT_BITS = 16)."""
    assert X.dtype in (np.uint8, np.uint16) and X.ndim == 2 and X.flags.c_contiguous
    d1 = np.ascontiguousarray(d1, dtype=np.int32)
    ncoarse, nchan = d1.shape
    S = np.empty((ncoarse, nsub, ns1), dtype=np.uint32)
    fn = _load().oracle_subband_step1 if X.dtype == np.uint8 else _load().oracle_subband_step1_u16
    rc = fn(_p(X), ctypes.c_int(nchan), ctypes.c_size_t(X.shape[1]),
                                      ctypes.c_int(nsub), _p(d1), ctypes.c_int(ncoarse), ctypes.c_int(ns1),
                                      _p(S), ctypes.c_size_t(ns1))
    if rc != 0:
        raise ValueError("oracle_subband_step1 rc=%d" % rc)
    return S


def subband_step2(S: np.ndarray, d2: np.ndarray, ns: int) -> np.ndarray:
    """uint32 Y[ncoarse*nfine][ns]; row a*nfine+b."""
    assert S.dtype == np.uint32 and S.ndim == 3 and S.flags.c_contiguous
    d2 = np.ascontiguousarray(d2, dtype=np.int32)
    ncoarse, nsub, ns1 = S.shape
    nfine = d2.shape[0]
    assert d2.shape[1] == nsub
    Y = np.empty((ncoarse * nfine, ns), dtype=np.uint32)
    rc = _load().oracle_subband_step2(_p(S), ctypes.c_int(nsub), ctypes.c_size_t(ns1), ctypes.c_int(ns1),
                                      _p(d2), ctypes.c_int(nfine), ctypes.c_int(ncoarse), ctypes.c_int(ns),
                                      _p(Y), ctypes.c_size_t(ns))
    if rc != 0:
        raise ValueError("oracle_subband_step2 rc=%d" % rc)
    return Y


def subband_tables(f_mhz, t_samp_s: float, nsub: int, coarse_dm, fine_dm, ref: str = "top") -> Tuple[np.ndarray, np.ndarray]:
    """(d1[ncoarse][nchan], d2[nfine][nsub]) for reading SB.1 "B" -- both tables relative to the global f_ref.
    SB.2: the subband reference frequency is its highest channel frequency (ref="top", default) or, reading SB.2c
    (SURVEY 8(c) SB.2 alternative, 8(f) f4), the centre of the subband, (highest + lowest channel frequency) / 2
    (ref="centre")."""
    f = np.asarray(f_mhz, dtype=np.float64)
    cps = f.size // nsub
    assert cps * nsub == f.size and ref in ("top", "centre")
    f_ref = float(f.max())
    fs = f.reshape(nsub, cps)
    f_sub = fs.max(axis=1) if ref == "top" else 0.5 * (fs.max(axis=1) + fs.min(axis=1))
    d1 = delay_table(f, coarse_dm, t_samp_s, f_ref)
    d2 = delay_table(f_sub, fine_dm, t_samp_s, f_ref)
    return d1, d2


def integrate(Y: np.ndarray, w: int, ns: Optional[int] = None) -> np.ndarray:
    """uint32 [nrows][ns // w] block sums of width w (INT.1, INT.2)."""
    assert Y.dtype == np.uint32 and Y.ndim == 2 and Y.flags.c_contiguous
    if ns is None:
        ns = Y.shape[1]
    nw = ns // w
    out = np.empty((Y.shape[0], nw), dtype=np.uint32)
    rc = _load().oracle_integrate(_p(Y), ctypes.c_size_t(Y.shape[1]), ctypes.c_int(Y.shape[0]),
                                  ctypes.c_int(ns), ctypes.c_int(w), _p(out), ctypes.c_size_t(max(nw, 1)))
    if rc != 0:
        raise ValueError("oracle_integrate rc=%d" % rc)
    return out


def snr(V: np.ndarray, ddof: int = 0, n: Optional[int] = None) -> Tuple[np.ndarray, np.ndarray]:
    """(snr float32 [nrows], argmax uint32 [nrows]) over the first n values of every row."""
    assert V.dtype == np.uint32 and V.ndim == 2 and V.flags.c_contiguous
    if n is None:
        n = V.shape[1]
    s = np.empty(V.shape[0], dtype=np.float32)
    a = np.empty(V.shape[0], dtype=np.uint32)
    rc = _load().oracle_snr(_p(V), ctypes.c_size_t(V.shape[1]), ctypes.c_int(V.shape[0]), ctypes.c_int(n),
                            ctypes.c_int(ddof), _p(s), _p(a))
    if rc != 0:
        raise ValueError("oracle_snr rc=%d" % rc)
    return s, a


def search(Y: np.ndarray, widths: Sequence[int], ddof: int = 0):
    """integrate + snr for every width: (planes dict w -> I_w, snr [nrows][nW], argmax [nrows][nW])."""
    planes, S, A = {}, [], []
    for w in widths:
        I = Y if w == 1 else integrate(Y, w)
        planes[w] = I
        s, a = snr(np.ascontiguousarray(I), ddof)
        S.append(s)
        A.append(a)
    return planes, np.stack(S, axis=1), np.stack(A, axis=1)


def integrate_sliding(Y: np.ndarray, w: int, ns: Optional[int] = None) -> np.ndarray:
    """uint32 [nrows][ns - w + 1] stride-1 boxcar sums of width w (reading INT.1s)."""
    assert Y.dtype == np.uint32 and Y.ndim == 2 and Y.flags.c_contiguous
    if ns is None:
        ns = Y.shape[1]
    n = ns - w + 1
    out = np.empty((Y.shape[0], max(n, 1)), dtype=np.uint32)
    rc = _load().oracle_integrate_sliding(_p(Y), ctypes.c_size_t(Y.shape[1]), ctypes.c_int(Y.shape[0]),
                                          ctypes.c_int(ns), ctypes.c_int(w), _p(out), ctypes.c_size_t(max(n, 1)))
    if rc != 0:
        raise ValueError("oracle_integrate_sliding rc=%d" % rc)
    return out


def search_sliding(Y: np.ndarray, widths: Sequence[int], ddof: int = 0):
    """integrate_sliding + snr for every width: (planes dict w -> I^s_w, snr [nrows][nW], argmax [nrows][nW])."""
    planes, S, A = {}, [], []
    for w in widths:
        I = Y if w == 1 else integrate_sliding(Y, w)
        planes[w] = I
        s, a = snr(np.ascontiguousarray(I), ddof)
        S.append(s)
        A.append(a)
    return planes, np.stack(S, axis=1), np.stack(A, axis=1)


def dedisperse_masked(X: np.ndarray, mask: np.ndarray, delay: np.ndarray, ns: int) -> np.ndarray:
    """oracle dedispersion leaving out the channels whose mask byte is 0 (reading DD.7m)."""
    assert X.dtype == np.uint8 and X.ndim == 2 and X.flags.c_contiguous
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nrows, nchan = delay.shape
    assert nchan == X.shape[0] == mask.size
    Y = np.empty((nrows, ns), dtype=np.uint32)
    rc = _load().oracle_dedisperse_masked(_p(X), ctypes.c_int(nchan), ctypes.c_size_t(X.shape[1]), _p(mask),
                                          _p(delay), ctypes.c_int(nrows), ctypes.c_int(ns), _p(Y),
                                          ctypes.c_size_t(ns))
    if rc != 0:
        raise ValueError("oracle_dedisperse_masked rc=%d" % rc)
    return Y


# ---------------------------------------------------------------------------- all-cores leg (oracle_mt.cpp)
# Same arithmetic: every row is computed by the single-thread function above, rows are spread over
# the host cores with `omp parallel for`.
def dedisperse_mt(X: np.ndarray, delay: np.ndarray, ns: int) -> np.ndarray:
    assert X.dtype == np.uint8 and X.ndim == 2 and X.flags.c_contiguous
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    nrows, nchan = delay.shape
    assert nchan == X.shape[0]
    Y = np.empty((nrows, ns), dtype=np.uint32)
    rc = _load_mt().oracle_mt_dedisperse(_p(X), ctypes.c_int(nchan), ctypes.c_size_t(X.shape[1]), _p(delay),
                                         ctypes.c_int(nrows), ctypes.c_int(ns), _p(Y), ctypes.c_size_t(ns))
    if rc != 0:
        raise ValueError("oracle_mt_dedisperse rc=%d" % rc)
    return Y


def subband_mt(X: np.ndarray, d1: np.ndarray, d2: np.ndarray, nsub: int, ns: int):
    """(S uint32 [ncoarse][nsub][ns + max d2], Y uint32 [ncoarse*nfine][ns]), coarse DMs spread over the cores."""
    assert X.dtype == np.uint8 and X.ndim == 2 and X.flags.c_contiguous
    d1 = np.ascontiguousarray(d1, dtype=np.int32)
    d2 = np.ascontiguousarray(d2, dtype=np.int32)
    ncoarse, nchan = d1.shape
    nfine = d2.shape[0]
    ns1 = ns + int(d2.max())
    S = np.empty((ncoarse, nsub, ns1), dtype=np.uint32)
    Y = np.empty((ncoarse * nfine, ns), dtype=np.uint32)
    rc = _load_mt().oracle_mt_subband(_p(X), ctypes.c_int(nchan), ctypes.c_size_t(X.shape[1]), ctypes.c_int(nsub),
                                      _p(d1), ctypes.c_int(ncoarse), ctypes.c_int(ns1), _p(S), ctypes.c_size_t(ns1),
                                      _p(d2), ctypes.c_int(nfine), ctypes.c_int(ns), _p(Y), ctypes.c_size_t(ns))
    if rc != 0:
        raise ValueError("oracle_mt_subband rc=%d" % rc)
    return S, Y


def search_mt(Y: np.ndarray, widths: Sequence[int], ddof: int = 0):
    """integrate + snr for every width with the rows spread over the cores: (planes, snr, argmax)."""
    assert Y.dtype == np.uint32 and Y.ndim == 2 and Y.flags.c_contiguous
    L = _load_mt()
    planes, S, A = {}, [], []
    nrows, ns = Y.shape
    for w in widths:
        if w == 1:
            I = Y
        else:
            nw = ns // w
            I = np.empty((nrows, nw), dtype=np.uint32)
            rc = L.oracle_mt_integrate(_p(Y), ctypes.c_size_t(ns), ctypes.c_int(nrows), ctypes.c_int(ns),
                                       ctypes.c_int(w), _p(I), ctypes.c_size_t(max(nw, 1)))
            if rc != 0:
                raise ValueError("oracle_mt_integrate rc=%d" % rc)
        planes[w] = I
        s = np.empty(nrows, dtype=np.float32)
        a = np.empty(nrows, dtype=np.uint32)
        rc = L.oracle_mt_snr(_p(I), ctypes.c_size_t(I.shape[1]), ctypes.c_int(nrows), ctypes.c_int(I.shape[1]),
                             ctypes.c_int(ddof), _p(s), _p(a))
        if rc != 0:
            raise ValueError("oracle_mt_snr rc=%d" % rc)
        S.append(s)
        A.append(a)
    return planes, np.stack(S, axis=1), np.stack(A, axis=1)
