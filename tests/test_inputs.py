"""Pins for the seeded input generator (ra_inputs/gen.c) -- CPU only."""
import numpy as np

import ra_inputs as gen

MASK = (1 << 64) - 1
GOLDEN = 0x9E3779B97F4A7C15


def _mix(z):
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
    return z ^ (z >> 31)


def _key(seed, stream):
    return _mix((seed + GOLDEN) & MASK) ^ _mix((stream * GOLDEN + 0x632BE59BD9B4E019) & MASK)


def test_python_mix_is_splitmix64_known_answer():
    # Published SplitMix64 test vector, state seeded with 0: first three outputs.
    out = [_mix(((i + 1) * GOLDEN) & MASK) for i in range(3)]
    assert out == [0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4, 0x06C45D188009454F]


def test_bits_match_python_restatement():
    seed, stream = gen.BASE_SEED + 3, gen.STREAM_A2A
    got = gen.bits_u64(257, seed, stream)
    k = _key(seed, stream)
    want = [_mix((k + (i + 1) * GOLDEN) & MASK) for i in range(257)]
    assert [int(x) for x in got] == want


def test_counter_based_prefix_property():
    a = gen.bits_u64(1000, 7, 9)
    b = gen.bits_u64(10, 7, 9)
    assert np.array_equal(a[:10], b)
    assert not np.array_equal(gen.bits_u64(10, 7, 10), b)   # other stream
    assert not np.array_equal(gen.bits_u64(10, 8, 9), b)    # other seed


def test_uniform_range_and_moments():
    u = gen.uniform_f32(1 << 20, 1, 2)
    assert u.dtype == np.float32 and u.min() >= -1.0 and u.max() < 1.0
    assert abs(float(u.mean())) < 3e-3
    assert abs(float(u.var()) - 1.0 / 3.0) < 3e-3
    # 24-bit grid: u * 2^23 is an integer
    assert np.all(np.mod(u.astype(np.float64) * 8388608.0, 1.0) == 0.0)


def test_normal_moments_and_bf16_grid():
    b = gen.normal_bf16((1 << 20,), 3, 4)
    x = gen.bf16_bits_to_f32(b).astype(np.float64)
    assert abs(x.mean()) < 5e-3 and abs(x.var() - 1.0) < 1e-2
    assert np.isfinite(x).all() and np.abs(x).max() < 7.0
    # 4th moment of N(0,1) is 3 (bf16 rounding perturbs it by < 1e-2 relative)
    assert abs((x ** 4).mean() - 3.0) < 0.1


def test_smallint_values():
    b = gen.smallint_bf16((4096,), 5, 6, -2, 2)
    x = gen.bf16_bits_to_f32(b)
    assert set(np.unique(x).tolist()) == {-2.0, -1.0, 0.0, 1.0, 2.0}


def test_tagged_chunks():
    P, cb = 3, 64
    t = gen.tagged_chunks(P, cb).reshape(P, P, cb // 8)
    for i in range(P):
        for j in range(P):
            for w in range(cb // 8):
                assert int(t[i, j, w]) == (i << 56) | (j << 48) | w


def test_config_table_matches_baseline_json():
    c = gen.CONFIGS
    assert (c[0].M, c[0].N, c[0].K, c[0].P, c[0].ar_count) == (256, 256, 256, 4, 65536)
    assert (c[1].M, c[1].N, c[1].K, c[1].P, c[1].ar_count) == (8192, 8192, 8192, 8, 16 << 20)
    assert (c[2].M, c[2].N, c[2].K) == (64, 16384, 16384)
    assert c[3].coll == "alltoall" and c[3].chunk_bytes == 8 << 20 and c[3].P == 8
    assert c[4].coll == "alltoall" and (c[4].M, c[4].N, c[4].K) == (64, 16384, 16384)
    assert c[1].coll_bytes == 1 << 30 and c[3].coll_bytes == 1 << 30
    assert c[2].gemm_bytes == 2 * (64 * 16384 + 16384 * 16384 + 64 * 16384)


def test_paper_literal_configs():
    """PAPER.md:84-92 (Table 1): GEMM 8192^3 / 8192 x 57344 x 8192, collectives of 896 MB on 4 GPUs."""
    c = {x.name: x for x in gen.CONFIGS}
    for name in ("paper-cb-ar", "paper-mb-ar", "paper-cb-a2a", "paper-mb-a2a"):
        assert c[name].P == 4
    assert (c["paper-mb-ar"].M, c["paper-mb-ar"].N, c["paper-mb-ar"].K) == (8192, 57344, 8192)
    assert c["paper-mb-ar"].ar_count * 4 == 896 << 20 == 8192 * 57344 * 2        # the GEMM's bf16 output
    assert c["paper-mb-a2a"].chunk_bytes * 4 == 896 << 20
    assert c["paper-cb-ar"].coll_bytes == 2 * 4 * (896 << 20)
