"""Pins for oracle O2 (allreduce stand-in) and O3 (alltoall stand-in) -- CPU only.

O2: BASELINE.json north_star "fixed rank-order fp32 sum ... written back to all" (pattern PAPER.md:30).
O3: "alltoall chunk transpose (P x P chunks)", chunk (i,j) -> (j,i) (pattern PAPER.md:30, 94).
"""
import struct

import numpy as np
import pytest

import oracle
import ra_inputs as gen


def f32_add(a, b):
    """One IEEE binary32 RNE add, computed exactly in Python: double add of two floats
    is exact-enough (53 >= 2*24+2) so rounding the double sum to float is correctly rounded."""
    return struct.unpack("f", struct.pack("f", float(a) + float(b)))[0]


@pytest.mark.parametrize("P,count", [(1, 5), (2, 33), (3, 7), (5, 33), (4, 1)])
def test_allreduce_brute_force(P, count):
    bufs = [gen.uniform_f32(count, 21, 100 + r) * np.float32(10.0 ** (r - 2)) for r in range(P)]
    want = []
    for e in range(count):
        s = float(bufs[0][e])
        for r in range(1, P):
            s = f32_add(s, bufs[r][e])
        want.append(s)
    want = np.array(want, dtype=np.float32)
    oracle.allreduce(bufs)
    for b in bufs:
        assert np.array_equal(b.view(np.uint32), want.view(np.uint32))


@pytest.mark.parametrize("c", [0.5, 1.0, -3.25, 1.0 / 1024])
def test_allreduce_constant_buffers(c):
    """All ranks = c -> P*c, exact when every partial k*c is representable (c with few significant bits)."""
    P, n = 8, 1000
    bufs = [np.full(n, c, dtype=np.float32) for _ in range(P)]
    oracle.allreduce(bufs)
    for b in bufs:
        assert np.all(b == np.float32(P * c))


def test_allreduce_constant_point_one_is_sequential_not_product():
    """c = 0.1f: the left-to-right sum is 0.80000007 (0x3F4CCCCE), not fl(8*0.1f) = 0.8 (0x3F4CCCCD)."""
    bufs = [np.full(4, 0.1, dtype=np.float32) for _ in range(8)]
    oracle.allreduce(bufs)
    assert bufs[0].view(np.uint32)[0] == 0x3F4CCCCE
    assert np.float32(8) * np.float32(0.1) != bufs[0][0]


def test_allreduce_order_detectors():
    """Hand-computed (binary32, ulp(2^24) = 2):
    [2^24, 1 x7] left-to-right: 2^24 + 1 ties to even 2^24 every time -> 16777216.
       pairwise tree: (2^24+1)+(1+1)+((1+1)+(1+1)) = 2^24 + 2 + 4 = 16777222; right-to-left: 7 + 2^24 -> 16777224.
    [1, 2^-24 x7] left-to-right: 1 + 2^-24 ties to even 1.0 every time -> 1.0 exactly;
       right-to-left: 7*2^-24 + 1 = 1 + 0x0.000007p0 -> rounds to 0x1.000008p+0."""
    bufs = [np.array([16777216.0 if r == 0 else 1.0, 1.0 if r == 0 else 2.0 ** -24], dtype=np.float32) for r in range(8)]
    oracle.allreduce(bufs)
    for b in bufs:
        assert b[0] == np.float32(16777216.0)
        assert b[1] == np.float32(1.0)
    # the other orders really do differ (so a kernel using them fails parity)
    tree = np.float32(np.float32(np.float32(16777216.0) + np.float32(1)) + np.float32(2)) + np.float32(4)
    assert tree == np.float32(16777222.0)
    rl = np.float32(7.0) + np.float32(16777216.0)
    assert rl == np.float32(16777224.0)


def test_allreduce_denormals_kept():
    """2^-140 + 2^-140 = 2^-139 (subnormal); flush-to-zero would give 0."""
    d = np.float32(2.0 ** -140)
    assert d != 0
    bufs = [np.array([d], dtype=np.float32), np.array([d], dtype=np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32)]
    oracle.allreduce(bufs)
    assert bufs[0][0] == np.float32(2.0 ** -139) and bufs[3][0] == np.float32(2.0 ** -139)


def test_allreduce_p1_unchanged_p2_commutative_and_all_equal():
    x = gen.uniform_f32(100, 22, 1)
    keep = x.copy()
    oracle.allreduce([x])
    assert np.array_equal(x, keep)
    a, b = gen.uniform_f32(100, 22, 2), gen.uniform_f32(100, 22, 3)
    want = a + b
    oracle.allreduce([a, b])
    assert np.array_equal(a, want) and np.array_equal(b, want)
    bufs = gen.allreduce_buffers(gen.CONFIGS[0], 4099)
    oracle.allreduce(bufs)
    for b in bufs[1:]:
        assert np.array_equal(b.view(np.uint32), bufs[0].view(np.uint32))


def test_allreduce_against_float64_sum_within_bound():
    """Exact sum within the fp32 error bound: |s - exact| <= (P-1) * 2^-24 * sum|x| (standard)."""
    bufs = gen.allreduce_buffers(gen.CONFIGS[0], 10000)
    exact = np.sum([b.astype(np.float64) for b in bufs], axis=0)
    absum = np.sum([np.abs(b.astype(np.float64)) for b in bufs], axis=0)
    oracle.allreduce(bufs)
    assert np.all(np.abs(bufs[0].astype(np.float64) - exact) <= 3 * 2.0 ** -24 * absum + 1e-30)


# ----------------------------------------------------------------------------- O3
@pytest.mark.parametrize("P,cb", [(1, 16), (2, 16), (3, 48), (4, 32)])
def test_alltoall_brute_force(P, cb):
    send = np.arange(P * P * cb, dtype=np.uint64).astype(np.uint8) ^ np.uint8(0x5A)
    send = (send.astype(np.uint32) * 7 + np.arange(P * P * cb, dtype=np.uint32) // 3).astype(np.uint8)
    want = np.empty_like(send)
    for i in range(P):
        for j in range(P):
            for t in range(cb):
                want[(j * P + i) * cb + t] = send[(i * P + j) * cb + t]
    assert np.array_equal(oracle.alltoall(send, P, cb), want)


def test_alltoall_involution_and_diagonal():
    cfg = gen.CONFIGS[3]
    cb = 4096
    a = gen.alltoall_payload(cfg, cb)
    b = oracle.alltoall(a, cfg.P, cb)
    a2 = oracle.alltoall(b, cfg.P, cb)
    assert np.array_equal(a2, a)           # applied twice = identity
    assert not np.array_equal(b, a)
    w = cb // 8
    A, B = a.reshape(cfg.P, cfg.P, w), b.reshape(cfg.P, cfg.P, w)
    for i in range(cfg.P):
        assert np.array_equal(A[i, i], B[i, i])   # diagonal chunks stay in place
    assert np.array_equal(B, A.transpose(1, 0, 2))  # numpy's own transpose (library routine)


def test_alltoall_tagged_payload_and_checksums():
    P, cb = 5, 256
    t = gen.tagged_chunks(P, cb)
    r = oracle.alltoall(t, P, cb).reshape(P, P, cb // 8)
    for j in range(P):
        for i in range(P):
            words = r[j, i]
            assert np.all((words >> np.uint64(56)) == i) and np.all(((words >> np.uint64(48)) & np.uint64(0xFF)) == j)
            assert np.array_equal(words & np.uint64(0xFFFFFFFFFFFF), np.arange(cb // 8, dtype=np.uint64))
    a = gen.bits_u64(P * P * (cb // 8), 23, 1)
    b = oracle.alltoall(a, P, cb)
    A, B = a.reshape(P, P, -1), b.reshape(P, P, -1)
    assert np.array_equal(np.bitwise_xor.reduce(A, axis=2), np.bitwise_xor.reduce(B, axis=2).T)


def test_alltoall_nan_payload_is_bytewise():
    P, cb = 2, 16
    nanbits = np.array([0x7FC00001, 0xFFC00002, 0x7F800001, 0x80000000] * (P * P), dtype=np.uint32)
    out = oracle.alltoall(nanbits, P, cb)
    assert np.array_equal(out.reshape(P, P, 4), nanbits.reshape(P, P, 4).transpose(1, 0, 2))


# ----------------------------------------------------------------------------- O4
def test_overlap_replay():
    cfg = gen.CONFIGS[0]
    bufs = gen.allreduce_buffers(cfg, 257)
    once = [b.copy() for b in bufs]
    oracle.allreduce(once)
    twice = [b.copy() for b in once]
    oracle.allreduce(twice)           # iteration 2 sums iteration 1's results: s -> P-fold sequential sum of s
    rep = [b.copy() for b in bufs]
    oracle.overlap_replay(2, ar_bufs=rep)
    assert all(np.array_equal(x, y) for x, y in zip(rep, twice))
    a = gen.alltoall_payload(gen.CONFIGS[3], 64)
    ra, rb = oracle.overlap_replay(4, a2a_a=a, P=8, chunk_bytes=64)
    assert np.array_equal(ra, a) and np.array_equal(rb, oracle.alltoall(a, 8, 64))
