"""Seeded synthetic inputs for the ra-overlap hot path (host side, numpy out).

The single module both sides of every parity test draw their inputs from.  It
contains no arithmetic of the method itself: only the counter-based generator
in ``gen.c`` (SplitMix64 finaliser keyed by (seed, stream, element index)) and
the workload shapes of BASELINE.json's five configs.

bf16 tensors are returned as ``numpy.uint16`` bit patterns.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libra_inputs.so")

BASE_SEED = 20260609  # seed of config c is BASE_SEED + c  (input recipe)

# stream ids: one per tensor so tensors of one config are independent
STREAM_A, STREAM_B, STREAM_C, STREAM_AR, STREAM_A2A = 1, 2, 3, 16, 64


def build(force: bool = False) -> str:
    """Compile gen.c into libra_inputs.so (gcc, generic x86-64, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, sz, vp = ctypes.c_uint64, ctypes.c_size_t, ctypes.c_void_p
        lib.ra_inputs_bits_u64.argtypes = [vp, sz, u64, u64]
        lib.ra_inputs_uniform_f32.argtypes = [vp, sz, u64, u64]
        lib.ra_inputs_normal_bf16.argtypes = [vp, sz, u64, u64]
        lib.ra_inputs_smallint_bf16.argtypes = [vp, sz, u64, u64, ctypes.c_int, ctypes.c_int]
        lib.ra_inputs_tagged_chunks_u64.argtypes = [vp, ctypes.c_int, sz]
        for f in (lib.ra_inputs_bits_u64, lib.ra_inputs_uniform_f32, lib.ra_inputs_normal_bf16,
                  lib.ra_inputs_smallint_bf16, lib.ra_inputs_tagged_chunks_u64):
            f.restype = None
        _lib = lib
    return _lib


def _ptr(a: np.ndarray) -> int:
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def normal_bf16(shape, seed: int, stream: int, out: np.ndarray | None = None) -> np.ndarray:
    """N(0,1) rounded to bf16 (RNE); uint16 bit patterns."""
    a = np.empty(shape, dtype=np.uint16) if out is None else out
    _L().ra_inputs_normal_bf16(_ptr(a), a.size, seed, stream)
    return a


def uniform_f32(shape, seed: int, stream: int, out: np.ndarray | None = None) -> np.ndarray:
    """U[-1,1) fp32 with 24-bit resolution."""
    a = np.empty(shape, dtype=np.float32) if out is None else out
    _L().ra_inputs_uniform_f32(_ptr(a), a.size, seed, stream)
    return a


def bits_u64(n_words: int, seed: int, stream: int, out: np.ndarray | None = None) -> np.ndarray:
    """Raw 64-bit draws (alltoall payload: arbitrary bit patterns)."""
    a = np.empty(n_words, dtype=np.uint64) if out is None else out
    _L().ra_inputs_bits_u64(_ptr(a), a.size, seed, stream)
    return a


def smallint_bf16(shape, seed: int, stream: int, lo: int = -2, hi: int = 2) -> np.ndarray:
    """Integers uniform in [lo, hi] as bf16 bit patterns (integer-exact GEMM pin)."""
    a = np.empty(shape, dtype=np.uint16)
    _L().ra_inputs_smallint_bf16(_ptr(a), a.size, seed, stream, lo, hi)
    return a


def tagged_chunks(P: int, chunk_bytes: int) -> np.ndarray:
    """P*P chunks; 64-bit word w of chunk (i,j) is i<<56 | j<<48 | w."""
    assert chunk_bytes % 8 == 0
    a = np.empty(P * P * (chunk_bytes // 8), dtype=np.uint64)
    _L().ra_inputs_tagged_chunks_u64(_ptr(a), P, chunk_bytes // 8)
    return a


# ----------------------------------------------------------------------------
# bf16 <-> fp32 helpers for building structured test inputs (identity, ones...).
# Plain bit manipulation; values used with these are exactly representable.
def f32_to_bf16_bits_exact(x: np.ndarray) -> np.ndarray:
    """Truncate fp32 -> bf16 bits; asserts the value is exactly representable."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    assert not np.any(u & 0xFFFF), "value not exactly representable in bf16"
    return (u >> 16).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << 16).view(np.float32)


# ----------------------------------------------------------------------------
# BASELINE.json configs (index 0..4).  GEMM layout: transA=0, transB=1 (A is
# M x K, B is N x K, both K-contiguous), ld = K; C is M x N, ld = N.
@dataclass(frozen=True)
class Config:
    index: int
    name: str
    M: int
    N: int
    K: int
    coll: str            # "allreduce" | "alltoall"
    P: int
    ar_count: int = 0    # fp32 elements per rank buffer
    chunk_bytes: int = 0  # alltoall chunk size
    n_iters: int = 20

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def gemm_flops(self) -> float:
        return 2.0 * self.M * self.N * self.K

    @property
    def gemm_bytes(self) -> int:      # algorithmic minimum, beta == 0
        return 2 * (self.M * self.K + self.K * self.N + self.M * self.N)

    @property
    def coll_bytes(self) -> int:      # bytes moved (read + written)
        if self.coll == "allreduce":
            return 2 * 4 * self.P * self.ar_count
        return 2 * self.P * self.P * self.chunk_bytes


MiB = 1 << 20
CONFIGS = (
    Config(0, "tiny", 256, 256, 256, "allreduce", 4, ar_count=65536, n_iters=4),
    Config(1, "cb-ar", 8192, 8192, 8192, "allreduce", 8, ar_count=16 * MiB),
    Config(2, "mb-ar", 64, 16384, 16384, "allreduce", 8, ar_count=16 * MiB),
    Config(3, "cb-a2a", 8192, 8192, 8192, "alltoall", 8, chunk_bytes=8 * MiB),
    Config(4, "mb-a2a", 64, 16384, 16384, "alltoall", 8, chunk_bytes=8 * MiB),
    # The paper's literal Table 1 workloads: 4 GPUs, 896 MB collectives.  896 MiB is
    # exactly the bf16 output of the 8192 x 57344 GEMM, read here as the PER-RANK message: allreduce over P = 4 rank
    # buffers of 896 MiB (fp32 elements), alltoall with 4 chunks of 224 MiB per rank.
    Config(5, "paper-cb-ar", 8192, 8192, 8192, "allreduce", 4, ar_count=224 * MiB, n_iters=10),
    Config(6, "paper-mb-ar", 8192, 57344, 8192, "allreduce", 4, ar_count=224 * MiB, n_iters=10),
    Config(7, "paper-cb-a2a", 8192, 8192, 8192, "alltoall", 4, chunk_bytes=224 * MiB, n_iters=10),
    Config(8, "paper-mb-a2a", 8192, 57344, 8192, "alltoall", 4, chunk_bytes=224 * MiB, n_iters=10),
)


def gemm_operands(cfg: Config):
    """(A[M,K], B[N,K]) bf16 bit patterns, N(0,1)."""
    A = normal_bf16((cfg.M, cfg.K), cfg.seed, STREAM_A)
    B = normal_bf16((cfg.N, cfg.K), cfg.seed, STREAM_B)
    return A, B


def allreduce_buffers(cfg: Config, count: int | None = None):
    """List of P fp32 rank buffers, U[-1,1)."""
    n = cfg.ar_count if count is None else count
    return [uniform_f32(n, cfg.seed, STREAM_AR + r) for r in range(cfg.P)]


def alltoall_payload(cfg: Config, chunk_bytes: int | None = None) -> np.ndarray:
    """send buffer: P*P chunks of random bits (uint64 words)."""
    cb = cfg.chunk_bytes if chunk_bytes is None else chunk_bytes
    assert cb % 8 == 0
    return bits_u64(cfg.P * cfg.P * (cb // 8), cfg.seed, STREAM_A2A)
