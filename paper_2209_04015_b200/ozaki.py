"""ctypes binding of include/afqmc_ozaki.h (the Ozaki-scheme experiment).  Marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import torch

from .binding import AfqmcError, _require_cuda, _stream_ptr

_LIB = None
OZAKI_EXPORTS = ["afqmc_ozaki_gemm", "afqmc_ozaki_last_error"]


def load_ozaki_library():
    global _LIB
    if _LIB is None:
        path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libafqmc_ozaki.so")
        if not os.path.exists(path):
            raise AfqmcError(f"{path} not found: build it first (python -c 'import __graft_entry__ as g; g.build()')")
        lib = C.CDLL(path)
        vp, ip = C.c_void_p, C.c_int
        lib.afqmc_ozaki_gemm.argtypes = [vp, vp, ip, ip, ip, ip, vp, C.POINTER(C.c_double), C.POINTER(C.c_float),
                                         C.POINTER(C.c_float), ip, vp]
        lib.afqmc_ozaki_gemm.restype = ip
        lib.afqmc_ozaki_last_error.argtypes = []
        lib.afqmc_ozaki_last_error.restype = C.c_char_p
        _LIB = lib
    return _LIB


def ozaki_gemm(A, B, slices, store=True, repeats=1, stream=None):
    """afqmc_ozaki_gemm: C = A @ B.T through `slices` INT8 digit planes on tcgen05.  A [M, K], B [Ncol, K] contiguous CUDA
    float64.  Returns dict(C (or None), checksum, ms_slice, ms_gemm)."""
    _require_cuda()
    lib = load_ozaki_library()
    for t in (A, B):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == torch.float64 and t.dim() == 2):
            raise AfqmcError("ozaki_gemm: A and B must be contiguous 2-D CUDA float64 tensors")
    if A.shape[1] != B.shape[1]:
        raise AfqmcError("ozaki_gemm: A [M, K] and B [Ncol, K] must share K")
    M, K = A.shape
    Ncol = B.shape[0]
    out = torch.empty((M, Ncol), dtype=torch.float64, device=A.device) if store else None
    cs, ms_s, ms_g = C.c_double(0.0), C.c_float(0.0), C.c_float(0.0)
    rc = lib.afqmc_ozaki_gemm(A.data_ptr(), B.data_ptr(), M, Ncol, K, int(slices), out.data_ptr() if store else None,
                              C.byref(cs), C.byref(ms_s), C.byref(ms_g), int(repeats), _stream_ptr(stream))
    if rc != 0:
        raise AfqmcError(f"afqmc_ozaki_gemm failed ({rc}): {lib.afqmc_ozaki_last_error().decode()}")
    return dict(C=out, checksum=cs.value, ms_slice=ms_s.value, ms_gemm=ms_g.value)
