"""ra_gemm_static_ws: the GEMM entry point for callers that cannot allocate device memory.

Who that is: code that lives inside someone else's process -- a plug-in of a serving runtime or training framework whose
memory pool took the whole HBM at start-up and hands none of it out -- and code on a latency path where cudaMalloc /
cudaFree are off limits because they stall every stream of the device, which is the very compute / communication
concurrency this library is about.  ra_gemm asks such a caller for a workspace it has no means to get (stream-K plans:
the memory-bound GEMM on a reduced sm_budget, config 5's sweep).  ra_gemm_static_ws takes that workspace from a 16 MiB
array that is part of libra.so's device image instead.

What is checked here: on the same inputs it must produce exactly the bytes ra_gemm produces with a caller-allocated
workspace (same plan, same kernel, same reduction order -- the GEMM tests' own bar for a fixed plan is bit equality), on
two calls in a row, the second of which finds the array as the first left it (stale tile counters and partial sums);
also with a different shape in between, and against the CPU oracle.  A plan that needs more scratch than the array holds
must be refused with RA_ERR_SCRATCH_LIMIT and leave C untouched.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a problem in this extra
entry point must not hide the parity tests of the main path.  It does not depend on anything the other tests leave
behind (and passes in a fresh process on its own): every test zeroes / poisons its own output buffers, and the shared
array is deliberately NOT cleaned between tests.
"""
import numpy as np
import pytest

import oracle
import ra_inputs
from helpers import GEMM_TOL, gemm_norm_err, to_dev, to_host

pytestmark = pytest.mark.gpu

MIB = 1 << 20
NAN_BITS = 0x7FC0


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def _poisoned_c(M, N):
    import torch
    return torch.full((M, N), NAN_BITS, dtype=torch.int16, device="cuda")   # every element must be overwritten


def _existing_path(ra, M, N, K, dA, dB, occ, alpha=1.0):
    """ra_gemm with a workspace the caller allocated -- the path every other test pins against the oracle."""
    import torch
    need = ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ)
    ws = torch.empty(max(need, 16), dtype=torch.uint8, device="cuda")
    dC = _poisoned_c(M, N)
    ra.ra_gemm(0, 1, M, N, K, alpha, dA, K, dB, K, 0.0, dC, N, occ=occ, workspace=ws)
    torch.cuda.synchronize()
    return to_host(dC, np.uint16).reshape(M, N)


def _static_path(ra, M, N, K, dA, dB, occ, alpha=1.0):
    import torch
    dC = _poisoned_c(M, N)
    ra.ra_gemm_static_ws(0, 1, M, N, K, alpha, dA, K, dB, K, 0.0, dC, N, occ=occ)
    torch.cuda.synchronize()
    return to_host(dC, np.uint16).reshape(M, N)


# stream-K plans (they are the ones that use scratch), all within the 16 MiB the library carries
STREAM_K_CASES = [
    (64, 4096, 8192, dict(cluster_k=1)),                                   # 148 CTAs, 9.25 MiB of scratch
    (64, 4096, 8192, dict(cluster_k=1, sm_budget=74)),                     # same shape, other grid: other counter layout
    (64, 4096, 8192, dict(cluster_k=1, sm_budget=110, smem_reserve_bytes=128 * 1024, tile_k=32)),
]


@pytest.mark.parametrize("M,N,K,occ", STREAM_K_CASES)
def test_static_ws_matches_caller_workspace_twice_in_a_row(ra, M, N, K, occ):
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    need = ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ)
    assert plan["split_k"] > 1 and 0 < need <= ra.RA_GEMM_STATIC_WS_BYTES, (plan, need)   # the case really uses scratch
    A = ra_inputs.normal_bf16((M, K), 301, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 301, ra_inputs.STREAM_B)
    dA, dB = to_dev(A), to_dev(B)
    want = _existing_path(ra, M, N, K, dA, dB, occ)
    first = _static_path(ra, M, N, K, dA, dB, occ)
    second = _static_path(ra, M, N, K, dA, dB, occ)      # finds the first call's counters and partial sums in the array
    assert first.tobytes() == want.tobytes()
    assert second.tobytes() == want.tobytes()
    # and the existing path is itself right (so "equal to it" means "equal to the oracle's GEMM within the GEMM bound")
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B, 0.0, None)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B)
    assert gemm_norm_err(second, ref, rowA, colB) <= GEMM_TOL


def test_static_ws_integer_exact_after_a_different_shape(ra):
    """The array holds another launch's leftovers (more tiles, more CTAs) when this one starts; small-integer operands
    make every partial sum exact, so the result must equal the oracle bit for bit."""
    occ = dict(cluster_k=1)
    M0, N0, K0 = 64, 4096, 8192
    dA0 = to_dev(ra_inputs.normal_bf16((M0, K0), 302, ra_inputs.STREAM_A))
    dB0 = to_dev(ra_inputs.normal_bf16((N0, K0), 302, ra_inputs.STREAM_B))
    _static_path(ra, M0, N0, K0, dA0, dB0, occ)
    M, N, K = 48, 2048, 8192
    occ2 = dict(cluster_k=1, sm_budget=40)
    assert ra.ra_gemm_plan_query(0, 1, M, N, K, occ2)["split_k"] > 1
    A = ra_inputs.smallint_bf16((M, K), 303, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 303, ra_inputs.STREAM_B)
    ref_bits = oracle.gemm(0, 1, M, N, K, 1.0, A, B, 0.0, None)[1]
    dA, dB = to_dev(A), to_dev(B)
    for _ in range(2):
        got = _static_path(ra, M, N, K, dA, dB, occ2)
        assert got.tobytes() == np.ascontiguousarray(ref_bits).tobytes()


def test_static_ws_without_scratch_is_plain_ra_gemm(ra):
    M, N, K = 512, 768, 1024                                   # data-parallel plan: no workspace at all
    assert ra.ra_gemm_workspace_bytes(0, 1, M, N, K, None) == 0
    dA = to_dev(ra_inputs.normal_bf16((M, K), 304, ra_inputs.STREAM_A))
    dB = to_dev(ra_inputs.normal_bf16((N, K), 304, ra_inputs.STREAM_B))
    want = _existing_path(ra, M, N, K, dA, dB, None, alpha=0.5)
    for _ in range(2):
        assert _static_path(ra, M, N, K, dA, dB, None, alpha=0.5).tobytes() == want.tobytes()


def test_static_ws_refuses_plans_beyond_its_limit(ra):
    import torch
    M, N, K = 200, 10000, 1024                                 # stream-K over 256-wide tiles on 148 CTAs: 37 MiB
    assert ra.ra_gemm_workspace_bytes(0, 1, M, N, K, None) > ra.RA_GEMM_STATIC_WS_BYTES
    dA = to_dev(ra_inputs.normal_bf16((M, K), 305, ra_inputs.STREAM_A))
    dB = to_dev(ra_inputs.normal_bf16((N, K), 305, ra_inputs.STREAM_B))
    dC = _poisoned_c(M, N)
    with pytest.raises(ra.RaError) as e:
        ra.ra_gemm_static_ws(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, dC, N)
    assert e.value.status == ra.RA_ERR_SCRATCH_LIMIT and "RA_ERR_SCRATCH_LIMIT" in str(e.value)
    torch.cuda.synchronize()
    assert bool((dC == NAN_BITS).all())                        # refused before anything was enqueued
    # the same problem on fewer SMs fits, and then it works
    occ = dict(sm_budget=48)
    need = ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ)
    if 0 < need <= ra.RA_GEMM_STATIC_WS_BYTES:
        want = _existing_path(ra, M, N, K, dA, dB, occ)
        assert _static_path(ra, M, N, K, dA, dB, occ).tobytes() == want.tobytes()
