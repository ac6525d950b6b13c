"""Measured FP32 FMA-chain peak (bench.py's second denominator for the walk's roofline).

A measurement aid with its own small library (csrc/fma_peak.cu -> libbh_fma_peak.so); it is not part of
libbh, not declared in include/bh.h and nothing on the product path calls it."""
from __future__ import annotations

import ctypes as C

from . import build as _build


def measure(device: int = 0):
    """(packed FFMA2, scalar FFMA) register-resident FMA-chain rates in TFLOP/s on `device`."""
    L = C.CDLL(_build.build_fma_peak())
    L.bh_fma_peak_measure.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.bh_fma_peak_measure.restype = C.c_int
    a, b = C.c_double(0.0), C.c_double(0.0)
    rc = L.bh_fma_peak_measure(int(device), C.byref(a), C.byref(b))
    if rc != 0:
        raise RuntimeError(f"bh_fma_peak_measure: cudaError {rc}")
    return a.value, b.value
