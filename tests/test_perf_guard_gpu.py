"""Performance guard: every hot kernel against a library yardstick measured in the same process on the same box
(boxes of the pool differ by ~4 %, so absolute thresholds would be either loose or flaky).

Round 2 lost 4-5 % on three kernels to "harmless" generalisations -- a run-time tile_k, a run-time store predicate in the
allreduce, a run-time branch for the dynamic tile order -- and found them only by re-timing against round 1's library and
against cuBLAS.  These checks would have failed on each of them.  Yardsticks are library code (torch.matmul = cuBLAS,
Tensor.copy_) and are used here only as a ruler: nothing in the product path calls them.  Timing: CUDA events, back to
back launches, best of 5 repetitions for both sides.
"""
import numpy as np
import pytest

import ra_inputs
from helpers import to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def _best_ms(fn, inner, reps=5):
    import torch
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(True), torch.cuda.Event(True)
        e0.record()
        for _ in range(inner):
            fn()
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1) / inner)
    return best


def _gemm_pair(ra, M, N, K):
    import torch
    A = to_dev(ra_inputs.normal_bf16((M, K), 5, ra_inputs.STREAM_A)).view(torch.bfloat16)
    B = to_dev(ra_inputs.normal_bf16((N, K), 5, ra_inputs.STREAM_B)).view(torch.bfloat16)
    C = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(max(ra.ra_gemm_workspace_bytes(0, 1, M, N, K), 16), dtype=torch.uint8, device="cuda")
    ours = lambda: ra.ra_gemm(0, 1, M, N, K, 1.0, A, K, B, K, 0.0, C, N, workspace=ws)
    lib = lambda: torch.matmul(A, B.t(), out=C)
    return ours, lib


@pytest.mark.parametrize("M,N,K,inner,slack", [
    (64, 16384, 16384, 50, 1.12),      # weight streaming (mb-*): measured ratio 1.047-1.054 (88 vs 84 us); the run-time tile_k made it 1.10
    (8192, 8192, 8192, 4, 1.08),       # tensor-bound (cb-*), short bursts before the power cap settles: measured ratio 1.004-1.011
    (2048, 2048, 2048, 50, 1.45),      # single-wave pair tiles: measured ratio 1.13-1.24 (not a benchmark shape: wide margin)
])
def test_gemm_is_within_reach_of_the_library_gemm(ra, M, N, K, inner, slack):
    ours, lib = _gemm_pair(ra, M, N, K)
    for attempt in range(3):                     # a guard must not be flaky: a miss is re-measured before it counts
        t_lib = _best_ms(lib, inner)
        t_ours = _best_ms(ours, inner)
        if t_ours <= slack * t_lib:
            return
    assert t_ours <= slack * t_lib, f"ra_gemm {t_ours * 1e3:.1f} us vs library {t_lib * 1e3:.1f} us on {M}x{N}x{K}"


def test_collectives_move_bytes_at_copy_speed(ra):
    """allreduce emul (P = 8 x 64 MiB) and alltoall emul (64 chunks x 8 MiB) each move 1 GiB; a device-to-device copy of
    512 MiB moves the same.  Measured ratios: allreduce 0.996-1.006, alltoall 1.025-1.03 (the store predicate made the allreduce 1.04)."""
    import torch
    src = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    dst = torch.empty_like(src)
    bufs = [torch.zeros(16 << 20, dtype=torch.float32, device="cuda") for _ in range(8)]       # zeros: the in-place sum stays finite
    a = torch.zeros((64 * (8 << 20)) // 8, dtype=torch.int64, device="cuda")
    b = torch.empty_like(a)
    for attempt in range(3):                     # a guard must not be flaky: a miss is re-measured before it counts
        t_copy = _best_ms(lambda: dst.copy_(src), 10)
        t_ar = _best_ms(lambda: ra.ra_allreduce_emul(bufs), 10)
        t_a2a = _best_ms(lambda: ra.ra_alltoall_emul(a, b, 8, 8 << 20), 10)
        if t_ar <= 1.06 * t_copy and t_a2a <= 1.08 * t_copy:
            return
    assert t_ar <= 1.06 * t_copy, f"allreduce {t_ar * 1e3:.1f} us vs copy {t_copy * 1e3:.1f} us"
    assert t_a2a <= 1.08 * t_copy, f"alltoall {t_a2a * 1e3:.1f} us vs copy {t_copy * 1e3:.1f} us"
