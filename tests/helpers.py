"""Shared test helpers: device upload/download of bit-pattern arrays and the GEMM acceptance metric.

No method arithmetic lives here: the metric compares two given arrays (BASELINE.json:
"rel. error <= 1e-2, max-abs normalised by |A||B| row/column norms").
"""
from __future__ import annotations

import numpy as np

GEMM_TOL = 1e-2


def to_dev(a: np.ndarray):
    """numpy -> cuda tensor with the same bytes (uint16/uint64 go through same-width signed views)."""
    import torch
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        a = a.view(np.int16)
    elif a.dtype == np.uint64:
        a = a.view(np.int64)
    elif a.dtype == np.uint32:
        a = a.view(np.int32)
    return torch.from_numpy(a.copy()).cuda()


def to_host(t, dtype) -> np.ndarray:
    return t.detach().cpu().numpy().view(dtype)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def gemm_norm_err(gpu_bits: np.ndarray, ref: np.ndarray, rowA: np.ndarray, colB: np.ndarray, alpha: float = 1.0,
                  beta: float = 0.0, cin_bits: np.ndarray | None = None) -> float:
    gpu = bf16_bits_to_f64(gpu_bits)
    assert np.all(np.isfinite(gpu)), "NaN/Inf in GPU result"
    den = abs(alpha) * np.outer(rowA, colB) + 1e-30
    if beta != 0.0 and cin_bits is not None:
        den = den + abs(beta) * np.abs(bf16_bits_to_f64(cin_bits))
    return float(np.max(np.abs(gpu - ref) / den))
