"""ctypes binding of include/ddp_static.h (libddp_static.so): the one entry point that allocates nothing.

Argument marshalling only.  The two-step subband dedispersion runs with its intermediate in a 16 MiB
`static __device__` array inside the library (see the header for why, the limit, and the sharing rules: calls that
overlap on one GPU race on that array).  There is no CPU fallback: a missing library is an error.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libddp_static.so")
SYMBOLS = ("ddp_static_subband_dedisperse", "ddp_static_scratch_bytes", "ddp_static_last_error")
OK, E_ARG, E_SHAPE, E_TOO_LARGE, E_CUDA = 0, -1, -2, -3, -4

_lib = None


class DdpStaticError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("ddp_static_subband_dedisperse failed: status %d (%s)" % (status, text))
        self.status = status


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s is missing: run `python -m paper_1811_04165_b200.build` (no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.ddp_static_subband_dedisperse.argtypes = [vp, C.c_size_t, C.c_int, C.c_int, vp, C.c_int, C.c_int, vp, C.c_int,
                                                    C.c_int, C.c_int, vp, C.c_size_t, vp]
        L.ddp_static_subband_dedisperse.restype = C.c_int
        L.ddp_static_scratch_bytes.restype = C.c_size_t
        L.ddp_static_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def scratch_bytes() -> int:
    return int(lib().ddp_static_scratch_bytes())


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream) or None
    if isinstance(stream, int):
        return stream or None
    return int(stream.cuda_stream) or None


def subband_dedisperse(d_in, d_d1, max_d1: int, d_d2, max_d2: int, nsamp_out: int, d_out, stream=None) -> None:
    """d_in uint8 [nchan][in_stride], d_d1 int32 [n_coarse][nchan], d_d2 int32 [n_fine][n_subbands],
    d_out int32-typed uint32 [n_coarse * n_fine][out_stride] -- device tensors; asynchronous on `stream`."""
    nchan, in_stride = int(d_in.shape[0]), int(d_in.stride(0))
    n_coarse, n_fine, n_sub = int(d_d1.shape[0]), int(d_d2.shape[0]), int(d_d2.shape[1])
    if int(d_d1.shape[1]) != nchan or not d_d1.is_contiguous() or not d_d2.is_contiguous():
        raise ValueError("d_d1 must be contiguous [n_coarse][nchan], d_d2 contiguous [n_fine][n_subbands]")
    if int(d_out.shape[0]) != n_coarse * n_fine:
        raise ValueError("d_out needs n_coarse * n_fine rows")
    st = lib().ddp_static_subband_dedisperse(d_in.data_ptr(), in_stride, nchan, n_sub, d_d1.data_ptr(), n_coarse,
                                             int(max_d1), d_d2.data_ptr(), n_fine, int(max_d2), int(nsamp_out),
                                             d_out.data_ptr(), int(d_out.stride(0)), _stream(stream))
    if st != OK:
        raise DdpStaticError(st, lib().ddp_static_last_error().decode())
