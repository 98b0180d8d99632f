"""ctypes binding of libpsd_peaks.so (include/psd_peaks.h): roofline-denominator micro-benchmarks.

Argument marshalling only; every number is measured by the CUDA kernels in csrc/psd_peaks.cu.
"""
from __future__ import annotations

import ctypes as C
import os

from . import _build

EXPORTS = ("psd_peak_fp64_fma", "psd_peak_fp32_fma", "psd_peak_shared_atomic_f64",
           "psd_peak_global_red_f64")

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        path = _build.PEAKS_LIB
        if _build.is_stale(path):
            _build.build(target=path)
        if not os.path.exists(path):
            raise ImportError("libpsd_peaks.so is missing and could not be built")
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        L.psd_peak_fp64_fma.argtypes = [C.c_int, C.c_void_p, C.c_int, dp]
        L.psd_peak_fp32_fma.argtypes = [C.c_int, C.c_void_p, C.c_int, dp]
        L.psd_peak_shared_atomic_f64.argtypes = [C.c_int, C.c_void_p, C.c_int, dp]
        L.psd_peak_global_red_f64.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, dp]
        _lib = L
    return _lib


def _call(fn, *args) -> float:
    out = C.c_double(0.0)
    rc = fn(*args, C.byref(out))
    if rc:
        raise RuntimeError(f"libpsd_peaks: {fn.__name__} failed with status {rc}")
    return out.value


def measure(device: int = 0, stream=None, reps: int = 5) -> dict:
    """All peaks, as a dict (FLOP/s and atomics/s)."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libpsd_peaks needs a CUDA device")
    L = lib()
    st = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    return {
        "fp64_fma_flops": _call(L.psd_peak_fp64_fma, device, st, reps),
        "fp32_fma_flops": _call(L.psd_peak_fp32_fma, device, st, reps),
        "shared_atomic_f64_per_s": _call(L.psd_peak_shared_atomic_f64, device, st, reps),
        "global_red_f64_tile_per_s": _call(L.psd_peak_global_red_f64, device, st, 0, reps),
        "global_red_f64_scatter_per_s": _call(L.psd_peak_global_red_f64, device, st, 1, reps),
    }
