"""Binding of librpa_probes.so (include/rpa_probes.h): issue-rate probes of the FP64 and int8 tensor pipes.
Measurement helpers for bench.py and the tests -- not part of the product library, nothing on the chi0 path calls them."""
from __future__ import annotations

import ctypes as C

from . import build as _build

EXPORTS = ("rpa_probe_fp64_tensor_peak", "rpa_probe_int8_tensor_peak", "rpa_probe_last_error")

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build_probes())
        L.rpa_probe_fp64_tensor_peak.restype = C.c_int
        L.rpa_probe_fp64_tensor_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.rpa_probe_int8_tensor_peak.restype = C.c_int
        L.rpa_probe_int8_tensor_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
        L.rpa_probe_last_error.restype = C.c_char_p
        L.rpa_probe_last_error.argtypes = []
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise RuntimeError(f"librpa_probes error {rc}: " + lib().rpa_probe_last_error().decode("utf-8", "replace"))


def _stream(device):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("the probes need a CUDA device")
    return torch, torch.device(device)


def rpa_probe_fp64_tensor_peak(device="cuda:0") -> float:
    """Measured FP64 tensor (DMMA) TFLOP/s of this GPU."""
    torch, dev = _stream(device)
    with torch.cuda.device(dev):
        t = C.c_double(0.0)
        _check(lib().rpa_probe_fp64_tensor_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(t)))
    return float(t.value)


def rpa_probe_int8_tensor_peak(device="cuda:0"):
    """(int8 tcgen05 Top/s, mismatches of the self-checked first MMA)."""
    torch, dev = _stream(device)
    with torch.cuda.device(dev):
        t, bad = C.c_double(0.0), C.c_int32(-1)
        _check(lib().rpa_probe_int8_tensor_peak(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(t), C.byref(bad)))
    return float(t.value), int(bad.value)
