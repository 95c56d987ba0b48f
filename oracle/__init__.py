"""CPU oracle for the ra-overlap hot path -- TEST INFRASTRUCTURE, NOT PRODUCT.

Thin ctypes wrapper over ``oracle.c`` (plain C, fp64 GEMM from the definition,
strict rank-order fp32 allreduce, memcpy alltoall).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl
reference`` legs import this package; ``paper_2606_09200_b200`` never does, and
this package imports nothing from it.

bf16 tensors are ``numpy.uint16`` bit patterns throughout.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

# strict IEEE: no fast-math, no FMA contraction, SSE (x86-64 default), FTZ/DAZ untouched.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i, f, vp, sz = ctypes.c_int, ctypes.c_float, ctypes.c_void_p, ctypes.c_size_t
        lib.oracle_gemm.argtypes = [i, i, i, i, i, f, vp, i, vp, i, f, vp, i, vp, vp]
        lib.oracle_gemm_samples.argtypes = [i, i, i, i, i, f, vp, i, vp, i, f, vp, i, vp, vp, sz, vp]
        lib.oracle_gemm_norms.argtypes = [i, i, i, i, i, vp, i, vp, i, vp, vp]
        lib.oracle_allreduce.argtypes = [vp, i, sz]
        lib.oracle_alltoall.argtypes = [vp, vp, i, sz]
        lib.oracle_bf16_to_f32.argtypes = [vp, vp, sz]
        lib.oracle_f32_to_bf16.argtypes = [vp, vp, sz]
        lib.oracle_num_threads.restype = i
        lib.oracle_set_threads.argtypes = [i]
        for fn in (lib.oracle_gemm, lib.oracle_gemm_samples, lib.oracle_gemm_norms, lib.oracle_allreduce,
                   lib.oracle_alltoall, lib.oracle_bf16_to_f32, lib.oracle_f32_to_bf16, lib.oracle_set_threads):
            fn.restype = None
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_L().oracle_num_threads())


def set_threads(n: int) -> None:
    _L().oracle_set_threads(int(n))


def _c(a: np.ndarray, dtype) -> np.ndarray:
    assert a.dtype == dtype, (a.dtype, dtype)
    assert a.flags["C_CONTIGUOUS"]
    return a


def bf16_to_f32(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    out = np.empty(b.shape, dtype=np.float32)
    _L().oracle_bf16_to_f32(b.ctypes.data, out.ctypes.data, b.size)
    return out


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, dtype=np.uint16)
    _L().oracle_f32_to_bf16(x.ctypes.data, out.ctypes.data, x.size)
    return out


def _gemm_args(transA, transB, M, N, K, A, lda, B, ldb, Cin, ldc):
    _c(A, np.uint16), _c(B, np.uint16)
    lda = lda if lda is not None else (M if transA else K)
    ldb = ldb if ldb is not None else (K if transB else N)
    ldc = ldc if ldc is not None else N
    need_a = ((K - 1) * lda + M) if transA else ((M - 1) * lda + K)
    need_b = ((N - 1) * ldb + K) if transB else ((K - 1) * ldb + N)
    assert A.size >= need_a and B.size >= need_b, "operand buffer too small for (shape, ld)"
    cin_ptr = None
    if Cin is not None:
        _c(Cin, np.uint16)
        assert Cin.size >= (M - 1) * ldc + N
        cin_ptr = Cin.ctypes.data
    return lda, ldb, ldc, cin_ptr


def gemm(transA: int, transB: int, M: int, N: int, K: int, alpha: float, A: np.ndarray, B: np.ndarray,
         beta: float = 0.0, Cin: np.ndarray | None = None, lda=None, ldb=None, ldc=None):
    """O1.  Returns (ref fp64 [M,N], ref rounded to bf16 bits [M,N])."""
    lda, ldb, ldc, cin_ptr = _gemm_args(transA, transB, M, N, K, A, lda, B, ldb, Cin, ldc)
    assert beta == 0.0 or Cin is not None
    ref = np.empty((M, N), dtype=np.float64)
    ref16 = np.empty((M, N), dtype=np.uint16)
    _L().oracle_gemm(transA, transB, M, N, K, alpha, A.ctypes.data, lda, B.ctypes.data, ldb, beta, cin_ptr, ldc,
                     ref.ctypes.data, ref16.ctypes.data)
    return ref, ref16


def gemm_samples(transA, transB, M, N, K, alpha, A, B, ii, jj, beta=0.0, Cin=None, lda=None, ldb=None, ldc=None):
    """O1 on sampled entries (ii[s], jj[s]); fp64."""
    lda, ldb, ldc, cin_ptr = _gemm_args(transA, transB, M, N, K, A, lda, B, ldb, Cin, ldc)
    ii = np.ascontiguousarray(ii, dtype=np.int64)
    jj = np.ascontiguousarray(jj, dtype=np.int64)
    assert ii.shape == jj.shape and ii.min(initial=0) >= 0 and ii.max(initial=0) < M and jj.max(initial=0) < N
    ref = np.empty(ii.shape, dtype=np.float64)
    _L().oracle_gemm_samples(transA, transB, M, N, K, alpha, A.ctypes.data, lda, B.ctypes.data, ldb, beta, cin_ptr,
                             ldc, ii.ctypes.data, jj.ctypes.data, ii.size, ref.ctypes.data)
    return ref


def gemm_norms(transA, transB, M, N, K, A, B, lda=None, ldb=None):
    """(||op(A)(i,:)||_2 for all i, ||op(B)(:,j)||_2 for all j), fp64."""
    lda, ldb, _, _ = _gemm_args(transA, transB, M, N, K, A, lda, B, ldb, None, None)
    ra = np.empty(M, dtype=np.float64)
    cb = np.empty(N, dtype=np.float64)
    _L().oracle_gemm_norms(transA, transB, M, N, K, A.ctypes.data, lda, B.ctypes.data, ldb, ra.ctypes.data,
                           cb.ctypes.data)
    return ra, cb


def allreduce(bufs: list[np.ndarray]) -> None:
    """O2, in place: every buffer <- ((b0+b1)+...)+b_{P-1}, fp32, this order."""
    P = len(bufs)
    n = bufs[0].size
    for b in bufs:
        _c(b, np.float32)
        assert b.size == n
    ptrs = (ctypes.c_void_p * P)(*[b.ctypes.data for b in bufs])
    _L().oracle_allreduce(ptrs, P, n)


def alltoall(send: np.ndarray, P: int, chunk_bytes: int) -> np.ndarray:
    """O3, out of place: recv chunk (j,i) <- send chunk (i,j).  Byte arrays (any dtype, viewed as bytes)."""
    s = np.ascontiguousarray(send).view(np.uint8).reshape(-1)
    assert s.size == P * P * chunk_bytes
    r = np.empty_like(s)
    _L().oracle_alltoall(s.ctypes.data, r.ctypes.data, P, chunk_bytes)
    return r.view(send.dtype)


def overlap_replay(n_iters: int, ar_bufs: list[np.ndarray] | None = None,
                   a2a_a: np.ndarray | None = None, P: int = 0, chunk_bytes: int = 0):
    """O4: the schedule has no arithmetic of its own; its result is
    O2 / O3 applied n_iters times in program order (allreduce in place; alltoall
    ping-pong a->b on even iterations, b->a on odd).  The GEMM has beta=0 and fixed
    A, B, so its result is O1's, every iteration.  Returns (a, b) for alltoall."""
    if ar_bufs is not None:
        for _ in range(n_iters):
            allreduce(ar_bufs)
        return None
    a = a2a_a.copy()
    b = np.zeros_like(a)
    for it in range(n_iters):
        if it % 2 == 0:
            b = alltoall(a, P, chunk_bytes)
        else:
            a = alltoall(b, P, chunk_bytes)
    return a, b
