"""GPU robustness: canary (guard-band) checks for out-of-bounds writes and a seeded fuzz over shapes / layouts / knobs.

compute-sanitizer is not available on this pool, so every kernel's writes are fenced in by hand: the output lives in
the middle of a larger allocation filled with a sentinel, and everything outside the output (guard bands before and
after, pad columns between rows) must be untouched afterwards.  TMA stores clip in hardware, direct stores are
predicated in the kernels -- both are exercised (planner paths: big tiles, pair tiles, single-CTA tiles, stream-K,
skinny/swapped, squeezed-by-reserve without store staging).
"""
import numpy as np
import pytest

import oracle
import ra_inputs
from helpers import GEMM_TOL, gemm_norm_err, to_dev, to_host

pytestmark = pytest.mark.gpu

SENT16 = 0x7FA5          # a NaN pattern no computation produces
GUARD = 4096             # elements of guard band on each side


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def _gemm_with_guards(ra, M, N, K, ldc, occ, transA=0, transB=1, alpha=1.0, beta=0.0, seed=1):
    import torch
    lda = (M if transA else K)
    ldb = (K if transB else N)
    A = ra_inputs.normal_bf16((K if transA else M, lda), seed, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N if transB else K, ldb), seed, ra_inputs.STREAM_B)
    big = torch.full((GUARD + M * ldc + GUARD,), SENT16, dtype=torch.int16, device="cuda")
    cin = None
    if beta != 0.0:
        cin = ra_inputs.normal_bf16((M, ldc), seed, ra_inputs.STREAM_C)
        cin[:, N:] = SENT16                                     # pad columns keep the sentinel
        big[GUARD:GUARD + M * ldc] = to_dev(cin).reshape(-1)
    C = big[GUARD:GUARD + M * ldc]
    assert C.data_ptr() % 16 == 0
    ws = torch.empty(max(ra.ra_gemm_workspace_bytes(transA, transB, M, N, K, occ), 16), dtype=torch.uint8, device="cuda")
    ra.ra_gemm(transA, transB, M, N, K, alpha, to_dev(A), lda, to_dev(B), ldb, beta, C, ldc, occ=occ, workspace=ws)
    torch.cuda.synchronize()
    h = to_host(big, np.uint16)
    assert np.all(h[:GUARD] == SENT16), "write before C"
    assert np.all(h[GUARD + M * ldc:] == SENT16), "write after C"
    body = h[GUARD:GUARD + M * ldc].reshape(M, ldc)
    assert np.all(body[:, N:] == SENT16), "pad columns of C were written"
    ref, _ = oracle.gemm(transA, transB, M, N, K, alpha, A, B, beta, cin, ldc=ldc if cin is not None else None)
    rowA, colB = oracle.gemm_norms(transA, transB, M, N, K, A, B)
    err = gemm_norm_err(body[:, :N].copy(), ref, rowA, colB, alpha, beta, cin[:, :N] if cin is not None else None)
    assert err <= GEMM_TOL, (err, ra.ra_gemm_plan_query(transA, transB, M, N, K, occ))


@pytest.mark.parametrize("M,N,K,occ", [
    (1000, 520, 200, dict(cta_group=2, m_blocks=2)),                      # big tiles, ragged both ways (TMA store clips)
    (1000, 520, 200, dict(cta_group=2, m_blocks=1)),                      # pair tiles
    (200, 136, 72, None),                                                 # single-CTA tile, one ragged tile
    (200, 10000, 1024, None),                                             # stream-K: partial tiles + fix-up stores
    (64, 1000, 512, None),                                                # skinny / swapped: transposed direct stores
    (1000, 520, 200, dict(cta_group=2, smem_reserve_bytes=128 * 1024)),   # squeezed: no store staging, direct stores
    (513, 257 + 7, 64, dict(cta_group=2, m_blocks=2)),                    # one row / a few columns into the next tile
    # N % 8 != 0: a TMA store clips at 16-byte granularity and would spill into the pad columns (regression: it did)
    (256, 1100, 64, None), (128, 12, 64, None), (700, 1097, 72, dict(cta_group=2, m_blocks=2)), (130, 65, 136, None),
])
@pytest.mark.parametrize("beta", [0.0, -0.5])
def test_gemm_writes_stay_inside_c(ra, M, N, K, occ, beta):
    ldc = (N + 7) // 8 * 8 + 8                                            # at least 8 pad columns per row
    _gemm_with_guards(ra, M, N, K, ldc, occ, beta=beta, alpha=1.0 if beta == 0.0 else 2.0, seed=M + N + K)


@pytest.mark.parametrize("variant", [0, 1])
@pytest.mark.parametrize("P,count", [(1, 5), (3, 4099), (8, 1 << 16), (16, 100003)])
def test_allreduce_writes_stay_inside_buffers(ra, P, count, variant):
    import torch
    pad = (count + 3) // 4 * 4                                            # keeps every rank buffer 16-byte aligned
    stride = 64 + pad + 64
    sent = np.float32(-123456.0)
    big = torch.full((P * stride,), float(sent), dtype=torch.float32, device="cuda")
    host = [ra_inputs.uniform_f32(count, 77, ra_inputs.STREAM_AR + r) for r in range(P)]
    bufs = []
    for r in range(P):
        b = big[r * stride + 64: r * stride + 64 + count]
        b.copy_(torch.from_numpy(host[r]))
        bufs.append(b)
    ra.ra_allreduce_emul_ex(bufs, count, variant=variant)
    torch.cuda.synchronize()
    oracle.allreduce(host)
    h = to_host(big, np.float32)
    for r in range(P):
        seg = h[r * stride:(r + 1) * stride]
        assert np.all(seg[:64] == sent) and np.all(seg[64 + count:] == sent), f"rank {r}: write outside the buffer"
        assert seg[64:64 + count].tobytes() == host[r].tobytes()


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("P,chunk", [(1, 16), (3, 48 * 1024 + 16), (5, 4096)])
def test_alltoall_writes_stay_inside_recv(ra, variant, P, chunk):
    import torch
    n = P * P * chunk // 8
    send = ra_inputs.tagged_chunks(P, chunk)
    sent = np.int64(0x5A5A5A5A5A5A5A5A)
    big = torch.full((512 + n + 512,), int(sent), dtype=torch.int64, device="cuda")
    recv = big[512:512 + n]
    s = to_dev(send)
    ra.ra_alltoall_emul_ex(s, recv, P, chunk, variant=variant)
    torch.cuda.synchronize()
    h = to_host(big, np.int64)
    assert np.all(h[:512] == sent) and np.all(h[512 + n:] == sent), "write outside recv"
    assert h[512:512 + n].tobytes() == oracle.alltoall(send, P, chunk).tobytes()
    assert to_host(s, np.uint64).tobytes() == send.tobytes(), "send was modified"


def test_gemm_fuzz_shapes_layouts_knobs(ra):
    """Seeded fuzz: 72 random problems over all four (transA, transB), ragged sizes, alpha/beta and planner knobs."""
    rng = np.random.default_rng(20260609)
    sizes = [1, 7, 8, 63, 64, 65, 127, 128, 129, 200, 255, 256, 257, 384, 511, 512, 520, 777, 1024, 1100]
    ks = [8, 24, 64, 72, 136, 512, 1000, 2048]
    knobs = [None, dict(cta_group=1), dict(cta_group=2), dict(cta_group=2, m_blocks=2), dict(sm_budget=9),
             dict(smem_reserve_bytes=96 * 1024), dict(tiles_per_cta=2), dict(sm_budget=33, smem_reserve_bytes=160 * 1024),
             dict(cluster_k=2), dict(cluster_k=4), dict(cta_group=2, m_blocks=1, cluster_k=2), dict(cluster_k=1)]
    for case in range(72):
        M, N = int(rng.choice(sizes)), int(rng.choice(sizes))
        K = int(rng.choice(ks))
        tA, tB = int(rng.integers(0, 2)), int(rng.integers(0, 2))
        # TMA pitch: leading dimensions must be multiples of 8 elements
        if (tA and M % 8) or (not tA and K % 8) or (tB and K % 8) or (not tB and N % 8):
            M, N, K = (M + 7) // 8 * 8, (N + 7) // 8 * 8, (K + 7) // 8 * 8
        occ = knobs[int(rng.integers(0, len(knobs)))]
        alpha, beta = [(1.0, 0.0), (2.0, 0.0), (-0.5, 1.0), (1.0, -2.0)][int(rng.integers(0, 4))]
        ldc = (N + 7) // 8 * 8 + (8 if case % 2 else 0)
        _gemm_with_guards(ra, M, N, K, ldc, occ, transA=tA, transB=tB, alpha=alpha, beta=beta, seed=1000 + case)
