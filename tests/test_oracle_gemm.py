"""Pins for oracle O1 (GEMM, PAPER.md:28 `C = alpha*op(A)*op(B) + beta*C`) -- CPU only.

Each pin is something other than the oracle itself: a long-double brute force
typed here, closed forms, exactly-representable special cases, numpy's own
float64 / int64 matmul (independent library routine), torch's bf16 conversion.
"""
import itertools

import numpy as np
import pytest
import torch

import oracle
import ra_inputs as gen


def f32(bits):
    return gen.bf16_bits_to_f32(bits)


def bits_of(x):
    return gen.f32_to_bf16_bits_exact(np.asarray(x, dtype=np.float32))


def brute(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, Cin, ldc):
    """Independent triple loop in long double, straight from PAPER.md:28."""
    Af, Bf = f32(A).astype(np.longdouble), f32(B).astype(np.longdouble)
    Cf = f32(Cin).astype(np.longdouble) if Cin is not None else None
    out = np.zeros((M, N), dtype=np.longdouble)
    for i in range(M):
        for j in range(N):
            acc = np.longdouble(0)
            for k in range(K):
                a = Af[k * lda + i] if transA else Af[i * lda + k]
                b = Bf[j * ldb + k] if transB else Bf[k * ldb + j]
                acc += a * b
            r = np.longdouble(alpha) * acc
            if beta != 0:
                r += np.longdouble(beta) * Cf[i * ldc + j]
            out[i, j] = r
    return out


@pytest.mark.parametrize("transA,transB", list(itertools.product([0, 1], [0, 1])))
@pytest.mark.parametrize("alpha,beta", [(1.0, 0.0), (-0.5, 2.0), (2.0, 1.0), (0.0, -0.5)])
def test_brute_force_all_layouts(transA, transB, alpha, beta):
    M, N, K = 17, 13, 19
    lda = (M if transA else K) + 3       # padded leading dims: catches ld/stride mix-ups
    ldb = (K if transB else N) + 5
    ldc = N + 2
    rowsA = K if transA else M
    rowsB = N if transB else K
    A = gen.normal_bf16((rowsA * lda,), 11, 1)
    B = gen.normal_bf16((rowsB * ldb,), 11, 2)
    Cin = gen.normal_bf16((M * ldc,), 11, 3)
    ref, ref16 = oracle.gemm(transA, transB, M, N, K, alpha, A, B, beta, Cin, lda=lda, ldb=ldb, ldc=ldc)
    want = brute(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, Cin, ldc)
    assert np.max(np.abs(ref.astype(np.longdouble) - want)) <= 1e-13 * max(1.0, float(np.max(np.abs(want))))
    # the rounded copy is torch's fp32->bf16 (independent RNE implementation) of the same values
    t16 = torch.from_numpy(ref.astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(ref16, t16)


def test_identity_left_and_right_bit_exact():
    n = 48
    I = bits_of(np.eye(n))
    X = gen.normal_bf16((n, n), 12, 1)
    # A = I, transB=0: C = B exactly (every product exact, every sum adds zeros)
    _, c16 = oracle.gemm(0, 0, n, n, n, 1.0, I, X)
    assert np.array_equal(c16, X)
    # B = I (transB=1 layout is I^T = I): C = A
    _, c16 = oracle.gemm(0, 1, n, n, n, 1.0, X, I)
    assert np.array_equal(c16, X)
    # transA=1 with A buffer holding X^T: op(A) = X
    _, c16 = oracle.gemm(1, 0, n, n, n, 1.0, np.ascontiguousarray(X.T), I)
    assert np.array_equal(c16, X)
    # transB=1 against I on the left: C(i,j) = op(B)(i,j) = B[j,i]
    _, c16 = oracle.gemm(0, 1, n, n, n, 1.0, I, X)
    assert np.array_equal(c16, X.T)


def test_zero_and_beta_semantics():
    M, N, K = 9, 11, 7
    Z = np.zeros((M, K), dtype=np.uint16)
    B = gen.normal_bf16((N, K), 13, 2)
    A = gen.normal_bf16((M, K), 13, 1)
    Cin = gen.normal_bf16((M, N), 13, 3)
    # A = 0 -> C = beta*Cin exactly (beta = 1: unchanged bits; beta = 2: exact doubling)
    ref, c16 = oracle.gemm(0, 1, M, N, K, 1.0, Z, B, 1.0, Cin)
    assert np.array_equal(c16, Cin)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, Z, B, 2.0, Cin)
    assert np.array_equal(ref, 2.0 * f32(Cin).astype(np.float64))
    # alpha = 0, beta = 1 -> unchanged
    _, c16 = oracle.gemm(0, 1, M, N, K, 0.0, A, B, 1.0, Cin)
    assert np.array_equal(c16, Cin)
    # beta = 0 -> Cin is not read: NaN-filled Cin must not propagate (BLAS, reading A14)
    nan = np.full((M, N), 0x7FC0, dtype=np.uint16)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B, 0.0, nan)
    assert np.isfinite(ref).all()
    ref2, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B, 0.0, None)
    assert np.array_equal(ref, ref2)


@pytest.mark.parametrize("K,want_bf16", [(256, 256.0), (257, 256.0), (259, 260.0), (8192, 8192.0)])
def test_ones_closed_form_and_rne(K, want_bf16):
    """ones x ones = K.  257 and 259 sit exactly between two bf16 values: RNE sends
    257 -> 256 (down, even) and 259 -> 260 (up, even); truncation or round-half-away fail one."""
    M, N = 5, 6
    one = bits_of(np.ones((max(M, N), K)))
    ref, c16 = oracle.gemm(0, 1, M, N, K, 1.0, one[:M].copy(), one[:N].copy())
    assert np.all(ref == float(K))
    assert np.all(f32(c16) == want_bf16)


def test_rank_one_closed_form():
    M, N, K = 12, 10, 33
    u = np.array([(-1) ** i * (i % 5 + 1) for i in range(M)], dtype=np.float32)        # small ints
    v = np.array([2.0 ** ((j % 7) - 3) for j in range(N)], dtype=np.float32)           # powers of two
    A = bits_of(np.repeat(u[:, None], K, axis=1))
    B = bits_of(np.repeat(v[:, None], K, axis=1))     # transB=1 layout: B[j,k] = v_j
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    assert np.array_equal(ref, K * np.outer(u, v).astype(np.float64))


@pytest.mark.parametrize("transA,transB", list(itertools.product([0, 1], [0, 1])))
def test_integer_exact_vs_numpy_int_matmul(transA, transB):
    M, N, K = 37, 29, 301
    A = gen.smallint_bf16((K, M) if transA else (M, K), 14, 1)
    B = gen.smallint_bf16((N, K) if transB else (K, N), 14, 2)
    Ai = f32(A).astype(np.int64)
    Bi = f32(B).astype(np.int64)
    opA = Ai.T if transA else Ai
    opB = Bi.T if transB else Bi
    ref, c16 = oracle.gemm(transA, transB, M, N, K, 1.0, A, B)
    want = opA @ opB
    assert np.array_equal(ref, want.astype(np.float64))
    # |entries| <= 4*301 = 1204 -> not all representable in bf16; compare through torch's rounding
    t16 = torch.from_numpy(want.astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(c16, t16)


def test_against_numpy_float64_matmul():
    M, N, K = 64, 48, 1000
    A = gen.normal_bf16((M, K), 15, 1)
    B = gen.normal_bf16((N, K), 15, 2)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    want = f32(A).astype(np.float64) @ f32(B).astype(np.float64).T
    scale = np.sqrt(K)
    assert np.max(np.abs(ref - want)) <= 1e-12 * scale * 10


def test_linearity_power_of_two_alpha():
    M, N, K = 16, 16, 128
    A = gen.normal_bf16((M, K), 16, 1)
    B = gen.normal_bf16((N, K), 16, 2)
    r1, c1 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    r2, c2 = oracle.gemm(0, 1, M, N, K, 2.0, A, B)
    assert np.array_equal(r2, 2.0 * r1)
    assert np.array_equal(f32(c2), 2.0 * f32(c1))


def test_transposed_buffers_give_identical_results():
    M, N, K = 21, 18, 40
    A = gen.normal_bf16((M, K), 17, 1)
    B = gen.normal_bf16((N, K), 17, 2)
    r_tn, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    r_nn, _ = oracle.gemm(0, 0, M, N, K, 1.0, A, np.ascontiguousarray(B.T))
    r_tt, _ = oracle.gemm(1, 1, M, N, K, 1.0, np.ascontiguousarray(A.T), B)
    r_nt, _ = oracle.gemm(1, 0, M, N, K, 1.0, np.ascontiguousarray(A.T), np.ascontiguousarray(B.T))
    assert np.array_equal(r_tn, r_nn) and np.array_equal(r_tn, r_tt) and np.array_equal(r_tn, r_nt)
    # a genuinely non-symmetric case must differ when the flag is wrong
    r_wrong, _ = oracle.gemm(0, 0, K, K, K, 1.0, gen.normal_bf16((K, K), 17, 5), gen.normal_bf16((K, K), 17, 6))
    r_right, _ = oracle.gemm(0, 1, K, K, K, 1.0, gen.normal_bf16((K, K), 17, 5), gen.normal_bf16((K, K), 17, 6))
    assert not np.array_equal(r_wrong, r_right)


def test_samples_and_norms():
    M, N, K = 33, 27, 65
    A = gen.normal_bf16((M, K), 18, 1)
    B = gen.normal_bf16((N, K), 18, 2)
    Cin = gen.normal_bf16((M, N), 18, 3)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.5, A, B, -0.25, Cin)
    rng = np.random.default_rng(0)
    ii, jj = rng.integers(0, M, 200), rng.integers(0, N, 200)
    s = oracle.gemm_samples(0, 1, M, N, K, 1.5, A, B, ii, jj, -0.25, Cin)
    assert np.array_equal(s, ref[ii, jj])
    ra, cb = oracle.gemm_norms(0, 1, M, N, K, A, B)
    assert np.allclose(ra, np.linalg.norm(f32(A).astype(np.float64), axis=1), rtol=1e-14)
    assert np.allclose(cb, np.linalg.norm(f32(B).astype(np.float64), axis=1), rtol=1e-14)
    # Cauchy-Schwarz: |C_ij| <= ||a_i|| ||b_j|| (the normalisation of the acceptance metric)
    r0, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    assert np.all(np.abs(r0) <= np.outer(ra, cb) * (1 + 1e-12))


def test_bf16_conversion_against_torch():
    rng = np.random.default_rng(1)
    x = rng.standard_normal(100000).astype(np.float32) * np.float32(10.0) ** rng.integers(-30, 30, 100000).astype(np.float32)
    special = np.array([0.0, -0.0, np.inf, -np.inf, 1.0, 257.0, 259.0, 3.3895314e38, 1e-45, 65504.0], dtype=np.float32)
    x = np.concatenate([x, special])
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(oracle.f32_to_bf16(x), want)
    assert np.isnan(f32(oracle.f32_to_bf16(np.array([np.nan], dtype=np.float32)))).all()
    # widening is exact: matches torch
    b = rng.integers(0, 1 << 16, 70000).astype(np.uint16)
    w = torch.from_numpy(b.view(np.int16)).view(torch.bfloat16).to(torch.float32).numpy()
    got = oracle.bf16_to_f32(b)
    assert np.array_equal(got.view(np.uint32), w.view(np.uint32))
