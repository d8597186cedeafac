"""ctypes binding of the allocation-free entry point of liblcf.so (include/lcf_noalloc.h).  Marshalling only."""
from __future__ import annotations

import ctypes as C

from . import lcf

MAX_FRAMES = 128          # LCF_NOALLOC_MAX_FRAMES
EXPORTS = ["lcf_gram_global_noalloc", "lcf_noalloc_last_error"]


def _lib() -> C.CDLL:
    L = lcf.load()         # raises if liblcf.so is missing: no fallback
    L.lcf_gram_global_noalloc.argtypes = [C.c_void_p, C.c_int, C.c_longlong, C.c_void_p, C.c_void_p]
    L.lcf_gram_global_noalloc.restype = C.c_int
    L.lcf_noalloc_last_error.argtypes = []
    L.lcf_noalloc_last_error.restype = C.c_char_p
    return L


def last_error() -> str:
    return _lib().lcf_noalloc_last_error().decode()


def gram_global_noalloc(iq_dev, N: int, P: int, R_dev, stream=None) -> None:
    """R[i][j] = sum_p conj(S[i][p]) S[j][p] (Eq. 1) of the device-resident complex64 [N][P] cube into the device-resident
    N x N complex128 matrix R_dev; asynchronous on `stream`; allocates nothing (N <= MAX_FRAMES)."""
    st = _lib().lcf_gram_global_noalloc(lcf._ptr(iq_dev), int(N), int(P), lcf._ptr(R_dev), lcf._stream(stream))
    if st != lcf.OK:
        raise lcf.LcfError(st, last_error() or "lcf_gram_global_noalloc")
