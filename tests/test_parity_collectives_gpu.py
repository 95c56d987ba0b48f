"""GPU parity: K2 allreduce stand-in and K3 alltoall stand-in vs the CPU oracle, through the C ABI.

Acceptance: BIT-EXACT (BASELINE.json north_star).
"""
import numpy as np
import pytest

import oracle
import ra_inputs
from helpers import to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def _run_allreduce(ra, bufs_np, sm_budget=0, variant=0, smem=0):
    import torch
    dev = [to_dev(b) for b in bufs_np]
    if variant == 0 and smem == 0:
        ra.ra_allreduce_emul(dev, count=bufs_np[0].size, sm_budget=sm_budget)
    else:
        ra.ra_allreduce_emul_ex(dev, count=bufs_np[0].size, sm_budget=sm_budget, smem_bytes_per_cta=smem, variant=variant)
    torch.cuda.synchronize()
    return [to_host(d, np.float32) for d in dev]


def _assert_bits_equal(a: np.ndarray, b: np.ndarray):
    assert a.tobytes() == b.tobytes()


@pytest.mark.parametrize("P", [1, 2, 3, 4, 8, 9, 16])
@pytest.mark.parametrize("count", [1, 3, 4, 1000, 65536, 2 * 148 * 512 * 4 * 3 + 7])
def test_allreduce_matches_oracle(ra, P, count):
    bufs = [ra_inputs.uniform_f32(count, 777 + P, ra_inputs.STREAM_AR + r) for r in range(P)]
    ref = [b.copy() for b in bufs]
    oracle.allreduce(ref)
    got = _run_allreduce(ra, bufs)
    for r in range(P):
        _assert_bits_equal(got[r], ref[r])


@pytest.mark.parametrize("P", [1, 2, 3, 8, 16])
@pytest.mark.parametrize("count", [1, 3, 4, 100, 1000, 65536 + 36, 2 * 148 * 1024 * 3 + 7])
@pytest.mark.parametrize("smem", [0, 16 * 1024, 200 * 1024])
def test_allreduce_tma_variant_matches_oracle(ra, P, count, smem):
    """variant 1 (TMA ring + shared-memory sum): same rank order, so bit-exact too; several slot sizes, ragged tails."""
    bufs = [ra_inputs.uniform_f32(count, 888 + P, ra_inputs.STREAM_AR + r) for r in range(P)]
    ref = [b.copy() for b in bufs]
    oracle.allreduce(ref)
    got = _run_allreduce(ra, bufs, variant=1, smem=smem)
    for r in range(P):
        _assert_bits_equal(got[r], ref[r])


def test_allreduce_tma_variant_order_and_denormals(ra):
    n = 4099
    bufs = [np.full(n, 2.0 ** 24, np.float32)] + [np.ones(n, np.float32) for _ in range(7)]
    assert np.all(_run_allreduce(ra, bufs, variant=1)[5] == np.float32(16777216.0))
    bufs = [np.ones(n, np.float32)] + [np.full(n, 2.0 ** -24, np.float32) for _ in range(7)]
    assert np.all(_run_allreduce(ra, bufs, variant=1)[0] == np.float32(1.0))
    tiny = np.float32(2.0 ** -140)
    bufs = [np.full(n, tiny, np.float32), np.full(n, tiny, np.float32)] + [np.zeros(n, np.float32) for _ in range(2)]
    assert np.all(_run_allreduce(ra, bufs, variant=1, sm_budget=3)[2] == np.float32(2.0 ** -139))


def test_allreduce_order_detectors(ra):
    # left-to-right gives 16777216; a tree gives 16777222; right-to-left 16777224
    n = 4099
    bufs = [np.full(n, 2.0 ** 24, np.float32)] + [np.ones(n, np.float32) for _ in range(7)]
    got = _run_allreduce(ra, bufs)
    assert np.all(got[0] == np.float32(16777216.0))
    bufs = [np.ones(n, np.float32)] + [np.full(n, 2.0 ** -24, np.float32) for _ in range(7)]
    got = _run_allreduce(ra, bufs)
    assert np.all(got[3] == np.float32(1.0))


def test_allreduce_denormals_kept(ra):
    n = 1031
    tiny = np.float32(2.0 ** -140)
    bufs = [np.full(n, tiny, np.float32), np.full(n, tiny, np.float32)] + [np.zeros(n, np.float32) for _ in range(2)]
    got = _run_allreduce(ra, bufs)
    assert np.all(got[0] == np.float32(2.0 ** -139))


@pytest.mark.parametrize("budget", [1, 37, 74, 148])
def test_allreduce_budget_invariant(ra, budget):
    cfg = ra_inputs.CONFIGS[0]
    bufs = ra_inputs.allreduce_buffers(cfg)
    ref = [b.copy() for b in bufs]
    oracle.allreduce(ref)
    got = _run_allreduce(ra, bufs, sm_budget=budget)
    for r in range(cfg.P):
        _assert_bits_equal(got[r], ref[r])


def test_allreduce_errors(ra):
    import torch
    a = torch.zeros(64, dtype=torch.float32, device="cuda")
    with pytest.raises(ra.RaError) as e:
        ra.ra_allreduce_emul([a, a], count=64)          # aliasing
    assert e.value.status == ra.RA_ERR_INVALID_ARG
    with pytest.raises(ra.RaError):
        ra.ra_allreduce_emul([a[1:], torch.zeros(64, device="cuda")], count=32)   # misaligned
    with pytest.raises(ra.RaError):
        ra.ra_allreduce_emul([torch.zeros(4, device="cuda") for _ in range(17)], count=4)  # P > 16
    ra.ra_allreduce_emul([a], count=0)                  # empty: OK, no launch


# ---------------------------------------------------------------------------------------------
def _run_alltoall(ra, send_np, P, chunk_bytes, **kw):
    import torch
    s = to_dev(send_np)
    r = torch.full_like(s, -1)
    if kw:
        ra.ra_alltoall_emul_ex(s, r, P, chunk_bytes, **kw)
    else:
        ra.ra_alltoall_emul(s, r, P, chunk_bytes)
    torch.cuda.synchronize()
    return to_host(r, send_np.dtype), s, r


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("P,chunk", [(1, 16), (2, 48), (3, 1024), (4, 16 * 1024), (8, 16 * 1024 + 16),
                                      (8, 100 * 1024 + 32), (5, 1 << 20)])
def test_alltoall_tagged(ra, variant, P, chunk):
    send = ra_inputs.tagged_chunks(P, chunk)
    ref = oracle.alltoall(send, P, chunk)
    got, _, _ = _run_alltoall(ra, send, P, chunk, variant=variant)
    _assert_bits_equal(got, ref)


@pytest.mark.parametrize("variant", [0, 1, 2])
def test_alltoall_random_bits_and_involution(ra, variant):
    import torch
    cfg = ra_inputs.CONFIGS[3]
    chunk = 256 * 1024 + 48
    send = ra_inputs.alltoall_payload(cfg, chunk_bytes=chunk)
    ref = oracle.alltoall(send, cfg.P, chunk)
    got, s, r = _run_alltoall(ra, send, cfg.P, chunk, variant=variant)
    _assert_bits_equal(got, ref)
    back = torch.zeros_like(s)
    ra.ra_alltoall_emul_ex(r, back, cfg.P, chunk, variant=variant)
    torch.cuda.synchronize()
    _assert_bits_equal(to_host(back, send.dtype), send)


@pytest.mark.parametrize("smem,ctas,budget", [(16 * 1024, 1, 1), (32 * 1024, 4, 20), (128 * 1024, 1, 148),
                                              (200 * 1024, 1, 74)])
def test_alltoall_knobs_invariant(ra, smem, ctas, budget):
    P, chunk = 4, 300 * 1024 + 16
    send = ra_inputs.bits_u64(P * P * chunk // 8, 4242, ra_inputs.STREAM_A2A)
    ref = oracle.alltoall(send, P, chunk)
    got, _, _ = _run_alltoall(ra, send, P, chunk, sm_budget=budget, smem_bytes_per_cta=smem, ctas_per_sm=ctas)
    _assert_bits_equal(got, ref)


def test_alltoall_errors(ra):
    import torch
    a = torch.zeros(4 * 64, dtype=torch.uint8, device="cuda")
    b = torch.zeros(4 * 64, dtype=torch.uint8, device="cuda")
    with pytest.raises(ra.RaError):
        ra.ra_alltoall_emul(a, a, 2, 64)        # in place not supported
    with pytest.raises(ra.RaError):
        ra.ra_alltoall_emul(a, b, 2, 24)        # chunk not a multiple of 16
    with pytest.raises(ra.RaError):
        ra.ra_alltoall_emul(a, b, 0, 64)
    ra.ra_alltoall_emul(a, b, 2, 0)             # empty


@pytest.mark.parametrize("P", [1, 2, 3, 8, 16])
@pytest.mark.parametrize("count", [1, 3, 4, 1000, 65536 + 36, 2 * 148 * 512 * 4 + 7])
def test_allreduce_copy_engine_fanout_matches_oracle(ra, P, count):
    """variant 2 (ra.h, the DMA-offload mechanism): the kernel reduces into rank 0's buffer only and the copy
    engines put the sum into the others -- every buffer must still equal the oracle bit for bit."""
    bufs = [ra_inputs.uniform_f32(count, 555 + P, ra_inputs.STREAM_AR + r) for r in range(P)]
    ref = [b.copy() for b in bufs]
    oracle.allreduce(ref)
    got = _run_allreduce(ra, bufs, variant=2)
    for r in range(P):
        _assert_bits_equal(got[r], ref[r])


def test_allreduce_copy_engine_fanout_order_and_denormals(ra):
    bufs = [np.full(4099, 16777216.0 if r == 0 else 1.0, dtype=np.float32) for r in range(8)]
    assert np.all(_run_allreduce(ra, bufs, variant=2)[7] == np.float32(16777216.0))   # left to right: 2^24 + 1 stays 2^24
    bufs = [np.full(4099, 2.0 ** -140, dtype=np.float32) for _ in range(2)]
    assert np.all(_run_allreduce(ra, bufs, variant=2, sm_budget=3)[1] == np.float32(2.0 ** -139))
