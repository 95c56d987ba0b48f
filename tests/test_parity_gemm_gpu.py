"""GPU parity: K1 tcgen05 GEMM vs the CPU oracle, through the C ABI.

Acceptance (BASELINE.json north_star): max |gpu - ref| / (|alpha| ||opA(i,:)|| ||opB(:,j)|| + |beta||Cin|) <= 1e-2;
bit-exact where the arithmetic is exact (identity, integer-valued inputs, power-of-two alpha).
"""
import numpy as np
import pytest

import oracle
import ra_inputs
from helpers import GEMM_TOL, gemm_norm_err, to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ra():
    import paper_2606_09200_b200 as m
    return m


def run_gemm(ra, M, N, K, A, B, alpha=1.0, beta=0.0, Cin=None, occ=None, lda=None, ldb=None, ldc=None, fill=None,
             transA=0, transB=1):
    """A, B: bit arrays in the storage the trans flags describe.  Returns C bits [M, N] and the full [M, ldc] buffer."""
    import torch
    lda = lda or (M if transA else K)
    ldb = ldb or (K if transB else N)
    ldc = ldc or N
    dA, dB = to_dev(A), to_dev(B)
    if Cin is not None:
        dC = to_dev(Cin)
    else:
        dC = torch.full((M, ldc), 0x7FC0 if fill is None else fill, dtype=torch.int16, device="cuda")  # NaN-filled
    ws_bytes = ra.ra_gemm_workspace_bytes(transA, transB, M, N, K, occ)
    ws = torch.empty(max(ws_bytes, 16), dtype=torch.uint8, device="cuda")
    ra.ra_gemm(transA, transB, M, N, K, alpha, dA, lda, dB, ldb, beta, dC, ldc, occ=occ, workspace=ws)
    torch.cuda.synchronize()
    out = to_host(dC, np.uint16).reshape(M, ldc)
    return out[:, :N].copy(), out


def _up8(x):
    return (x + 7) // 8 * 8


def check(ra, M, N, K, seed, alpha=1.0, beta=0.0, occ=None, transA=0, transB=1):
    # leading dimensions rounded up to the 8-element pitch TMA needs; the pad columns hold data too
    # (so a kernel that ignored ld would read/write the wrong elements)
    def pad(x):
        return _up8(x) + (8 if x % 16 else 0)
    lda = pad(M) if transA else pad(K)
    ldb = pad(K) if transB else pad(N)
    ldc = _up8(N)
    A = ra_inputs.normal_bf16((K if transA else M, lda), seed, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N if transB else K, ldb), seed, ra_inputs.STREAM_B)
    Cin = ra_inputs.normal_bf16((M, ldc), seed, ra_inputs.STREAM_C) if beta != 0.0 else None
    ref, _ = oracle.gemm(transA, transB, M, N, K, alpha, A, B, beta, Cin, lda=lda, ldb=ldb, ldc=ldc)
    rowA, colB = oracle.gemm_norms(transA, transB, M, N, K, A, B, lda=lda, ldb=ldb)
    got, full = run_gemm(ra, M, N, K, A, B, alpha, beta, Cin, occ, lda=lda, ldb=ldb, ldc=ldc, transA=transA, transB=transB)
    cin_view = Cin[:, :N] if Cin is not None else None
    err = gemm_norm_err(got, ref, rowA, colB, alpha, beta, cin_view)
    assert err <= GEMM_TOL, (f"normalised error {err} for {M}x{N}x{K} trans {transA}{transB} "
                             f"plan {ra.ra_gemm_plan_query(transA, transB, M, N, K, occ)}")
    if Cin is not None and ldc > N:
        assert np.array_equal(full[:, N:], Cin[:, N:]), "pad columns of C were modified"
    return err


@pytest.mark.parametrize("transA,transB", [(0, 0), (1, 0), (1, 1)])
@pytest.mark.parametrize("M,N,K,occ", [
    (128, 256, 64, None), (200, 136, 72, None), (130, 260, 200, None), (384, 768, 2048, None),     # single-CTA tiles
    (64, 1024, 2048, None), (17, 640, 1536, None),                                                  # operand swap (+ stream-K)
    (512, 512, 256, dict(cta_group=2)), (1000, 520, 200, dict(cta_group=2)), (2048, 2048, 512, dict(cta_group=2)),  # CTA pairs
    (200, 200, 4096, None), (200, 10000, 1024, None),                                               # one narrow wave / stream-K
    (257, 131, 75, None), (1030, 259, 333, dict(cta_group=2)), (61, 643, 1027, None),               # odd M, N, K (padded ld)
])
def test_all_trans_combinations(ra, transA, transB, M, N, K, occ):
    """op(A), op(B) of PAPER.md:28: every storage order of both operands (MN-major UMMA descriptors + TMA boxes)."""
    check(ra, M, N, K, seed=7000 + M + N + K, occ=occ, transA=transA, transB=transB)


@pytest.mark.parametrize("transA,transB", [(0, 0), (1, 0), (1, 1)])
def test_trans_integer_exact(ra, transA, transB):
    M, N, K = 384, 520, 1024
    A = ra_inputs.smallint_bf16((K, M) if transA else (M, K), 51, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K) if transB else (K, N), 51, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(transA, transB, M, N, K, 1.0, A, B)
    got, _ = run_gemm(ra, M, N, K, A, B, transA=transA, transB=transB)
    assert np.array_equal(got, ref16)


def test_tiny_config(ra):
    cfg = ra_inputs.CONFIGS[0]
    A, B = ra_inputs.gemm_operands(cfg)
    ref, _ = oracle.gemm(0, 1, cfg.M, cfg.N, cfg.K, 1.0, A, B)
    rowA, colB = oracle.gemm_norms(0, 1, cfg.M, cfg.N, cfg.K, A, B)
    got, _ = run_gemm(ra, cfg.M, cfg.N, cfg.K, A, B)
    assert gemm_norm_err(got, ref, rowA, colB) <= GEMM_TOL


@pytest.mark.parametrize("M,N,K", [
    (128, 256, 64), (128, 64, 128), (256, 512, 256),          # whole tiles, each BN
    (200, 136, 72), (1, 8, 8), (130, 260, 200), (77, 40, 1000),  # ragged M, N, K tails
    (384, 768, 4096),                                          # several tiles per CTA? (6 tiles)
    (64, 1024, 2048), (17, 640, 1536), (64, 128, 512),         # skinny-M: operand swap (+ stream-K)
    (200, 200, 8192), (300, 200, 8192), (200, 10000, 1024),   # one narrow wave; stream-K on the non-swapped path
    (129, 67, 75), (5, 3, 1), (257, 1001, 333), (1030, 259, 1027),   # nothing a multiple of 8 (ld padded): OOB fill in K,
                                                               # element-granular edges in M and N
])
def test_shapes(ra, M, N, K):
    check(ra, M, N, K, seed=1000 + M + N + K)


@pytest.mark.parametrize("alpha,beta", [(1.0, 1.0), (-0.5, 2.0), (2.0, -0.5), (0.0, 1.0), (0.0, 0.0), (1.0, 0.0)])
@pytest.mark.parametrize("M,N,K", [(200, 136, 72), (64, 1024, 2048)])
def test_alpha_beta(ra, alpha, beta, M, N, K):
    check(ra, M, N, K, seed=5, alpha=alpha, beta=beta)


def test_identity_bit_exact(ra):
    # A = I  =>  C == B^T exactly (every product exact, every sum adds zeros).
    n = 256
    eye = ra_inputs.f32_to_bf16_bits_exact(np.eye(n, dtype=np.float32))
    Bm = ra_inputs.normal_bf16((384, n), 11, ra_inputs.STREAM_B)        # B is N x K
    got, _ = run_gemm(ra, n, 384, n, eye, Bm)
    assert np.array_equal(got, Bm.T)
    got, _ = run_gemm(ra, 384, n, n, Bm, eye)                           # B = I  =>  C == A
    assert np.array_equal(got, Bm)


@pytest.mark.parametrize("M,N,K", [(256, 256, 256), (200, 520, 4096), (64, 2048, 16384), (128, 256, 16384)])
def test_integer_exact(ra, M, N, K):
    # entries in {-2..2}: all partial sums are integers < 2^24 -> fp32 accumulation is exact in any order,
    # so the bf16 result must equal the oracle's bf16 rounding bit for bit (strongest layout/index pin).
    A = ra_inputs.smallint_bf16((M, K), 31, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 31, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got, _ = run_gemm(ra, M, N, K, A, B)
    assert np.array_equal(got, ref16)


@pytest.mark.parametrize("M,N,K", [(256, 256, 64), (512, 512, 256), (1000, 520, 200), (384, 768, 4096), (2048, 2048, 512),
                                   (257, 264, 72), (4096, 1024, 1024)])
@pytest.mark.parametrize("occ", [dict(cta_group=2, m_blocks=1), dict(cta_group=2, m_blocks=1, sm_budget=9, smem_reserve_bytes=96 * 1024),
                                 dict(cta_group=2, tiles_per_cta=1)])
def test_cta_pairs(ra, M, N, K, occ):
    """tcgen05 cta_group::2 path (2-CTA clusters, 256 x 256 tiles), forced on shapes the planner would not pick it for."""
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cta_group"] == 2 and plan["tile_m"] == 256 and plan["grid"] % 2 == 0, plan
    check(ra, M, N, K, seed=4000 + M + N + K, occ=occ)


@pytest.mark.parametrize("M,N,K", [(512, 256, 64), (1000, 520, 200), (2048, 2048, 512), (700, 264, 4096), (4096, 1024, 1024),
                                   (513, 264, 72), (1024, 512, 448), (520, 256, 8192)])   # K: skew on/off, empty middle
@pytest.mark.parametrize("occ", [dict(cta_group=2, m_blocks=2), dict(cta_group=2, m_blocks=2, sm_budget=10, smem_reserve_bytes=64 * 1024)])
def test_big_tiles(ra, M, N, K, occ):
    """m_blocks = 2: two 128-row MMA blocks per CTA share one B stage (512 x 256 tiles per CTA pair, single accumulator set)."""
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cta_group"] == 2 and plan["m_blocks"] == 2 and plan["tile_m"] == 512 and plan["stages"] >= 3, plan
    check(ra, M, N, K, seed=4500 + M + N + K, occ=occ)


@pytest.mark.parametrize("transA,transB", [(0, 0), (1, 0), (1, 1)])
def test_big_tiles_trans(ra, transA, transB):
    check(ra, 1032, 520, 328, seed=4600 + 2 * transA + transB, occ=dict(cta_group=2, m_blocks=2), transA=transA, transB=transB)
    check(ra, 1024, 512, 256, seed=4610 + 2 * transA + transB, alpha=-0.5, beta=2.0, occ=dict(cta_group=2, m_blocks=2),
          transA=transA, transB=transB)


def test_big_tiles_integer_exact_and_bit_identical(ra):
    M, N, K = 2048, 768, 2048
    A = ra_inputs.smallint_bf16((M, K), 43, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 43, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got2, _ = run_gemm(ra, M, N, K, A, B, occ=dict(cta_group=2, m_blocks=2))
    assert np.array_equal(got2, ref16)
    # same per-element K order => big tiles, pair tiles and single-CTA tiles agree bit for bit (A12)
    An = ra_inputs.normal_bf16((M, K), 44, ra_inputs.STREAM_A)
    Bn = ra_inputs.normal_bf16((N, K), 44, ra_inputs.STREAM_B)
    c4, _ = run_gemm(ra, M, N, K, An, Bn, occ=dict(cta_group=2, m_blocks=2))
    c2, _ = run_gemm(ra, M, N, K, An, Bn, occ=dict(cta_group=2, m_blocks=1, cluster_k=1))   # (no K split: same association)
    c1, _ = run_gemm(ra, M, N, K, An, Bn, occ=dict(cta_group=1, sm_budget=24, cluster_k=1))
    assert np.array_equal(c4, c2) and np.array_equal(c4, c1)


def test_cta_pairs_integer_exact_and_bit_identical_to_single(ra):
    M, N, K = 1024, 768, 2048
    A = ra_inputs.smallint_bf16((M, K), 41, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 41, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got2, _ = run_gemm(ra, M, N, K, A, B, occ=dict(cta_group=2))
    assert np.array_equal(got2, ref16)
    # same per-element K order (k-blocks ascending, one accumulator) => pairs and single CTAs agree bit for bit
    An = ra_inputs.normal_bf16((M, K), 42, ra_inputs.STREAM_A)
    Bn = ra_inputs.normal_bf16((N, K), 42, ra_inputs.STREAM_B)
    c2, _ = run_gemm(ra, M, N, K, An, Bn, occ=dict(cta_group=2, sm_budget=148, cluster_k=1))
    c1, _ = run_gemm(ra, M, N, K, An, Bn, occ=dict(cta_group=1, sm_budget=24, cluster_k=1))
    assert ra.ra_gemm_plan_query(0, 1, M, N, K, dict(cta_group=1, sm_budget=24))["split_k"] == 1
    assert np.array_equal(c1, c2)


def test_ones_closed_form(ra):
    for K in (256, 8192):
        one = ra_inputs.f32_to_bf16_bits_exact(np.ones((136, K), np.float32))
        got, _ = run_gemm(ra, 130, 136, K, one, one)
        assert np.all(ra_inputs.bf16_bits_to_f32(got) == np.float32(K))


def test_beta0_ignores_nan_in_c_and_respects_ldc(ra):
    M, N, K, ldc = 100, 72, 256, 96
    A = ra_inputs.normal_bf16((M, K), 3, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 3, ra_inputs.STREAM_B)
    got, full = run_gemm(ra, M, N, K, A, B, ldc=ldc)
    assert not np.any((got & 0x7FFF) > 0x7F80)              # no NaN leaked from the NaN-filled C
    assert np.all(full[:, N:] == 0x7FC0)                    # padding columns untouched
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B)
    assert gemm_norm_err(got, ref, rowA, colB) <= GEMM_TOL


def test_alpha_power_of_two_linearity(ra):
    M, N, K = 192, 320, 512
    A = ra_inputs.normal_bf16((M, K), 9, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 9, ra_inputs.STREAM_B)
    c1, _ = run_gemm(ra, M, N, K, A, B, alpha=1.0)
    c2, _ = run_gemm(ra, M, N, K, A, B, alpha=2.0)
    assert np.array_equal(ra_inputs.bf16_bits_to_f32(c2), 2.0 * ra_inputs.bf16_bits_to_f32(c1))


@pytest.mark.parametrize("occ", [
    dict(smem_reserve_bytes=0, sm_budget=74), dict(smem_reserve_bytes=64 * 1024, sm_budget=148),
    dict(smem_reserve_bytes=128 * 1024, sm_budget=110), dict(smem_reserve_bytes=160 * 1024, sm_budget=92),
    dict(smem_reserve_bytes=200 * 1024, sm_budget=148), dict(tiles_per_cta=1), dict(tiles_per_cta=3, smem_reserve_bytes=32 * 1024),
    dict(sm_budget=1), dict(sm_budget=7),
])
@pytest.mark.parametrize("M,N,K", [(512, 768, 1024), (64, 2048, 4096)])
def test_knobs_do_not_change_results(ra, occ, M, N, K):
    # PAPER.md:47 "without modifying kernel logic": occupancy shaping must not change what is computed.
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["smem_left_per_sm"] >= occ.get("smem_reserve_bytes", 0) or plan["clamped"]
    check(ra, M, N, K, seed=77, occ=occ)


def test_run_to_run_reproducible_stream_k(ra):
    M, N, K = 64, 4096, 8192
    sk = dict(cluster_k=1)                                   # without cluster split-K this shape is a stream-K plan
    assert ra.ra_gemm_plan_query(0, 1, M, N, K, sk)["split_k"] > 1
    A = ra_inputs.normal_bf16((M, K), 21, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 21, ra_inputs.STREAM_B)
    first, _ = run_gemm(ra, M, N, K, A, B, occ=sk)
    for _ in range(5):
        again, _ = run_gemm(ra, M, N, K, A, B, occ=sk)
        assert np.array_equal(first, again)


def test_budget_bit_identical_data_parallel(ra):
    # sm_budget / tiles_per_cta only change which CTA computes a tile.
    M, N, K = 1024, 1024, 512
    A = ra_inputs.normal_bf16((M, K), 22, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 22, ra_inputs.STREAM_B)
    base, _ = run_gemm(ra, M, N, K, A, B, occ=dict(sm_budget=32))
    for occ in (dict(sm_budget=16), dict(sm_budget=8, smem_reserve_bytes=100 * 1024), dict(tiles_per_cta=2)):
        plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
        if plan["split_k"] > 1 or plan["tile_n"] != 256:
            continue
        got, _ = run_gemm(ra, M, N, K, A, B, occ=occ)
        assert np.array_equal(base, got)


def test_errors(ra):
    import torch
    a = torch.zeros(64 * 64, dtype=torch.int16, device="cuda")
    b = torch.zeros(64 * 64, dtype=torch.int16, device="cuda")
    c = torch.zeros(64 * 64, dtype=torch.int16, device="cuda")
    for kw, st in [
        (dict(transA=1, lda=24), ra.RA_ERR_INVALID_ARG), (dict(lda=60), ra.RA_ERR_INVALID_ARG), (dict(lda=68), ra.RA_ERR_UNSUPPORTED),
        (dict(M=-1), ra.RA_ERR_INVALID_ARG), (dict(C=a), ra.RA_ERR_INVALID_ARG),
    ]:
        args = dict(transA=0, transB=1, M=32, N=32, K=64, alpha=1.0, A=a, lda=64, B=b, ldb=64, beta=0.0, C=c, ldc=64)
        args.update(kw)
        with pytest.raises(ra.RaError) as e:
            ra.ra_gemm(**args)
        assert e.value.status == st, kw
    ra.ra_gemm(0, 1, 0, 32, 64, 1.0, a, 64, b, 64, 0.0, c, 64)     # M == 0: nothing to do
    # K == 0: C = beta*C
    c.fill_(0x3F80)  # 1.0
    ra.ra_gemm(0, 1, 32, 32, 0, 1.0, a, 8, b, 8, 2.0, c, 64)
    torch.cuda.synchronize()
    out = to_host(c, np.uint16).reshape(64, 64)
    assert np.all(out[:32, :32] == 0x4000) and np.all(out[:32, 32:] == 0x3F80)


# ---- cluster split-K: 2-CTA clusters split one tile's K range, reduction through distributed shared memory ---------
@pytest.mark.parametrize("M,N,K", [(200, 200, 8192), (130, 100, 1000), (128, 64, 128), (64, 1024, 2048), (17, 640, 1536),
                                   (300, 128, 4096), (257, 131, 333), (1000, 64, 320), (8192, 128, 1024)])
def test_cluster_split_k(ra, M, N, K):
    occ = dict(cluster_k=2, cta_group=1)
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cluster_k"] == 2 and plan["split_k"] == 1 and plan["grid"] == 2 * plan["n_tiles"], plan
    assert ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ) == 0
    check(ra, M, N, K, seed=8000 + M + N + K, occ=occ)
    check(ra, M, N, K, seed=8100 + M + N + K, alpha=-0.5, beta=2.0, occ=occ)


@pytest.mark.parametrize("transA,transB", [(0, 0), (1, 0), (1, 1)])
def test_cluster_split_k_trans(ra, transA, transB):
    check(ra, 264, 200, 1032, seed=8200 + 2 * transA + transB, occ=dict(cluster_k=2, cta_group=1), transA=transA, transB=transB)
    check(ra, 40, 648, 520, seed=8210 + 2 * transA + transB, occ=dict(cluster_k=2), transA=transA, transB=transB)   # swapped


def test_cluster_split_k_auto_exact_and_reproducible(ra):
    M, N, K = 8192, 64, 2048                                   # 64 tiles x 32 k-blocks: the planner picks it on its own
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K)
    assert plan["cluster_k"] == 2 and plan["grid"] == 128, plan
    A = ra_inputs.smallint_bf16((M, K), 51, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 51, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got, _ = run_gemm(ra, M, N, K, A, B)
    assert np.array_equal(got, ref16)                          # integer inputs: exact in any summation order
    An = ra_inputs.normal_bf16((M, K), 52, ra_inputs.STREAM_A)
    Bn = ra_inputs.normal_bf16((N, K), 52, ra_inputs.STREAM_B)
    first, _ = run_gemm(ra, M, N, K, An, Bn)
    for _ in range(3):
        again, _ = run_gemm(ra, M, N, K, An, Bn)
        assert np.array_equal(first, again)                    # fixed order (low half + high half): run-to-run identical
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, An, Bn)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, An, Bn)
    assert gemm_norm_err(first, ref, rowA, colB) <= GEMM_TOL


# ---- fp32 output (ra_gemm_ex, RA_DTYPE_F32) -------------------------------------------------------------------------
def run_gemm_f32(ra, M, N, K, A, B, alpha=1.0, beta=0.0, Cin=None, occ=None, ldc=None, transA=0, transB=1):
    import torch
    lda = M if transA else K
    ldb = K if transB else N
    ldc = ldc or (N + 3) // 4 * 4
    dC = torch.full((M, ldc), float("nan"), dtype=torch.float32, device="cuda")
    if Cin is not None:
        dC.copy_(torch.from_numpy(Cin))
    ws = torch.empty(max(ra.ra_gemm_workspace_bytes(transA, transB, M, N, K, occ), 16), dtype=torch.uint8, device="cuda")
    ra.ra_gemm_ex(transA, transB, M, N, K, alpha, to_dev(A), lda, to_dev(B), ldb, beta, dC, ldc, ra.RA_DTYPE_F32, occ=occ, workspace=ws)
    torch.cuda.synchronize()
    return dC.cpu().numpy()


@pytest.mark.parametrize("M,N,K,occ", [
    (1024, 512, 512, None), (700, 264, 1024, dict(cta_group=2, m_blocks=2)), (200, 136, 72, None), (64, 1024, 2048, None),
    (200, 10000, 1024, None), (8192, 64, 2048, None), (129, 67, 72, None), (40, 648, 520, None)])
def test_f32_output(ra, M, N, K, occ):
    """C in fp32: same accumulator, no bf16 rounding.  Error bound: fp32 accumulation only (<= K * 2^-24 of the norm
    bound, far below it in practice); rounding the fp32 result to bf16 reproduces ra_gemm bit for bit."""
    A = ra_inputs.normal_bf16((M, K), 61, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 61, ra_inputs.STREAM_B)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B)
    ldc = (N + 3) // 4 * 4 + 4
    full = run_gemm_f32(ra, M, N, K, A, B, occ=occ, ldc=ldc)
    got = full[:, :N]
    assert np.all(np.isfinite(got)) and np.all(np.isnan(full[:, N:])), "unwritten C or pad columns touched"
    err = float(np.max(np.abs(got.astype(np.float64) - ref) / (np.outer(rowA, colB) + 1e-30)))
    assert err <= 2e-5, err
    bf, _ = run_gemm(ra, M, N, K, A, B, occ=occ, ldc=(N + 7) // 8 * 8)
    assert np.array_equal(oracle.f32_to_bf16(np.ascontiguousarray(got)), bf)
    # alpha / beta with an fp32 C_in
    rng = np.random.default_rng(M + N + K)
    Cin = rng.standard_normal((M, ldc)).astype(np.float32)
    out = run_gemm_f32(ra, M, N, K, A, B, alpha=-0.5, beta=2.0, Cin=Cin, occ=occ, ldc=ldc)
    want = -0.5 * ref + 2.0 * Cin[:, :N].astype(np.float64)
    den = 0.5 * np.outer(rowA, colB) + 2.0 * np.abs(Cin[:, :N]) + 1e-30
    assert float(np.max(np.abs(out[:, :N] - want) / den)) <= 2e-5
    assert np.array_equal(out[:, N:], Cin[:, N:])


def test_f32_output_integer_exact_and_errors(ra):
    import torch
    M, N, K = 512, 384, 4096
    A = ra_inputs.smallint_bf16((M, K), 62, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 62, ra_inputs.STREAM_B)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got = run_gemm_f32(ra, M, N, K, A, B)
    assert np.array_equal(got.astype(np.float64), ref)          # integers below 2^24: exact in fp32
    dC = torch.full((M, N), 3.0, dtype=torch.float32, device="cuda")
    ra.ra_gemm_ex(0, 1, M, N, K, 0.0, to_dev(A), K, to_dev(B), K, 0.5, dC, N, ra.RA_DTYPE_F32)   # alpha = 0: C = beta*C
    torch.cuda.synchronize()
    assert torch.all(dC == 1.5)
    with pytest.raises(ra.RaError) as e:
        ra.ra_gemm_ex(0, 1, M, N, K, 1.0, to_dev(A), K, to_dev(B), K, 0.0, dC, N, 7)
    assert e.value.status == ra.RA_ERR_INVALID_ARG
    with pytest.raises(ra.RaError) as e:
        ra.ra_gemm_ex(0, 1, M, N, K, 1.0, to_dev(A), K, to_dev(B), K, 0.0, dC, N + 2, ra.RA_DTYPE_F32)   # ldc % 4 != 0
    assert e.value.status == ra.RA_ERR_UNSUPPORTED


# ---- cluster split-K on CTA pairs: 4-CTA clusters, two pairs split one 256 x 256 tile's K range ----------------------
@pytest.mark.parametrize("M,N,K", [(512, 512, 4096), (300, 264, 2048), (1000, 520, 1032), (256, 256, 128), (257, 1001, 333)])
def test_pair_cluster_split_k(ra, M, N, K):
    occ = dict(cluster_k=2, cta_group=2, m_blocks=1)
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cluster_k"] == 2 and plan["cta_group"] == 2 and plan["grid"] == 4 * plan["n_tiles"], plan
    check(ra, M, N, K, seed=8300 + M + N + K, occ=occ)
    check(ra, M, N, K, seed=8400 + M + N + K, alpha=2.0, beta=-0.5, occ=occ)
    for transA, transB in ((0, 0), (1, 0), (1, 1)):
        check(ra, M, N, K, seed=8500 + M + 2 * transA + transB, occ=occ, transA=transA, transB=transB)


def test_pair_cluster_split_k_auto_exact_and_reproducible(ra):
    M, N, K = 384, 4096, 4096                                   # 32 pair tiles, 64 k-blocks: picked by the planner
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K)
    assert plan["cluster_k"] == 2 and plan["cta_group"] == 2 and plan["grid"] == 128, plan
    A = ra_inputs.smallint_bf16((M, K), 71, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 71, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got, _ = run_gemm(ra, M, N, K, A, B)
    assert np.array_equal(got, ref16)
    An = ra_inputs.normal_bf16((M, K), 72, ra_inputs.STREAM_A)
    Bn = ra_inputs.normal_bf16((N, K), 72, ra_inputs.STREAM_B)
    first, _ = run_gemm(ra, M, N, K, An, Bn)
    for _ in range(3):
        again, _ = run_gemm(ra, M, N, K, An, Bn)
        assert np.array_equal(first, again)
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, An, Bn)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, An, Bn)
    assert gemm_norm_err(first, ref, rowA, colB) <= GEMM_TOL


@pytest.mark.parametrize("M,N,K", [(200, 128, 8192), (130, 100, 1000), (128, 64, 256), (64, 1024, 2048), (17, 640, 1536),
                                   (257, 120, 336), (128, 1024, 4096)])
def test_cluster_split_k_four_parts(ra, M, N, K):
    occ = dict(cluster_k=4, cta_group=1)
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cluster_k"] == 4 and plan["split_k"] == 1 and plan["grid"] == 4 * plan["n_tiles"], plan
    assert ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ) == 0
    check(ra, M, N, K, seed=8600 + M + N + K, occ=occ)
    check(ra, M, N, K, seed=8700 + M + N + K, alpha=-0.5, beta=2.0, occ=occ, transA=1, transB=0)
    A = ra_inputs.smallint_bf16((M, K), 81, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, K), 81, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    got, _ = run_gemm(ra, M, N, K, A, B, occ=occ, ldc=(N + 7) // 8 * 8)
    assert np.array_equal(got, ref16)                          # integer inputs: exact whatever the association
    again, _ = run_gemm(ra, M, N, K, A, B, occ=occ, ldc=(N + 7) // 8 * 8)
    assert np.array_equal(got, again)


def _persisting_l2_limit():
    """The device's current cudaLimitPersistingL2CacheSize, read through cuda-python (independent of the library)."""
    cudart = pytest.importorskip("cuda.bindings.runtime")
    err, val = cudart.cudaDeviceGetLimit(cudart.cudaLimit.cudaLimitPersistingL2CacheSize)
    assert int(err) == 0, err
    return int(val)


def test_l2_persist_same_bits_and_state(ra):
    """occ.l2_persist_bytes (ra.h): a resource knob -- raster group + evict_last loads -- that must not change one bit of
    C (per-element k order is untouched), sets the device carve-out for ra_gemm and leaves it, and ra_l2_persist(0) /
    ra_overlap_run take it back."""
    M, N, K = 4096, 4096, 2048                      # 128 tiles of 512 x 256 over 74 CTA pairs: two waves, groups matter
    A = ra_inputs.normal_bf16((M, K), 71, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 71, ra_inputs.STREAM_B)
    base, _ = run_gemm(ra, M, N, K, A, B)
    occ = dict(l2_persist_bytes=24 << 20)
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["l2_persist_bytes"] == 24 << 20 and plan["group_x"] == 8, plan     # 2 MiB per tile row: all 8 rows of X stay resident
    got, _ = run_gemm(ra, M, N, K, A, B, occ=occ)
    assert got.tobytes() == base.tobytes()
    set_to = _persisting_l2_limit()                 # ra_gemm leaves the carve-out set (the next GEMM wants it too);
    assert 24 << 20 <= set_to < 40 << 20            # the driver rounds up to sixteenths of the L2 (7.9 MiB on B200)
    assert ra.ra_l2_persist(0) == 0
    assert _persisting_l2_limit() == 0
    # a knob-free GEMM after a persisting one takes the carve-out back by itself
    run_gemm(ra, M, N, K, A, B, occ=occ)
    assert _persisting_l2_limit() == set_to
    again, _ = run_gemm(ra, M, N, K, A, B)
    assert _persisting_l2_limit() == 0 and again.tobytes() == base.tobytes()
    # more than the device has: clamped, reported
    granted = ra.ra_l2_persist(1 << 40)
    assert 0 < granted <= 126 << 20 and _persisting_l2_limit() == granted
    assert ra.ra_l2_persist(0) == 0
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B)
    assert gemm_norm_err(got, ref, rowA, colB) <= GEMM_TOL


@pytest.mark.parametrize("M,N,K,occ", [
    (256, 256, 256, {}),                                     # Tiny
    (1024, 768, 2048, dict(cta_group=2, m_blocks=2)),        # big tiles, skewed issue over 64 k-blocks of 32
    (2048, 1024, 1024, dict(cta_group=2, m_blocks=1)),       # pair tiles
    (64, 2048, 4096, {}),                                    # skinny (operands swapped)
    (200, 136, 72, {}),                                      # ragged everywhere: K = 72 -> 3 k-blocks, the last 8 wide
    (129, 67, 40, {}),
    (1000, 3000, 520, dict(cluster_k=1)),                    # ragged K (520 = 16 units of 32 + 8) on a data-parallel pair-tile plan
    (512, 512, 8192, dict(sm_budget=37)),
])
def test_tile_k_32_same_bits_as_64(ra, M, N, K, occ):
    """occ.tile_k = 32 (ra.h; the tile-k axis of PAPER.md:140-144): half-size stages in 64-byte swizzle rows.  A
    data-parallel tile accumulates the same products in the same ascending-k order whatever the stage size, so C is
    bit-identical to tile_k = 64; stream-K plans cut K at different unit boundaries (tolerance there).  Oracle-exact on
    integer operands in any case."""
    occ = dict(occ, cluster_k=1)         # tile_k = 32 has no cluster split-K: compare like with like (same fp32 association)
    lda, ldb, ldc = _up8(K), _up8(K), _up8(N)
    A = ra_inputs.normal_bf16((M, lda), 90, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, ldb), 90, ra_inputs.STREAM_B)
    p64 = ra.ra_gemm_plan_query(0, 1, M, N, K, dict(occ, tile_k=64))
    p32 = ra.ra_gemm_plan_query(0, 1, M, N, K, dict(occ, tile_k=32))
    assert p32["tile_k"] == 32 and p64["tile_k"] == 64 and p32["clamped"] == 0, p32
    c64, _ = run_gemm(ra, M, N, K, A, B, occ=dict(occ, tile_k=64), lda=lda, ldb=ldb, ldc=ldc)
    c32, full = run_gemm(ra, M, N, K, A, B, occ=dict(occ, tile_k=32), lda=lda, ldb=ldb, ldc=ldc)
    assert np.all(full[:, N:] == 0x7FC0)                                    # pad columns of C untouched
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B, lda=lda, ldb=ldb)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B, lda=lda, ldb=ldb)
    assert gemm_norm_err(c32, ref, rowA, colB) <= GEMM_TOL
    if p32["split_k"] == 1 and p64["split_k"] == 1:
        assert c32.tobytes() == c64.tobytes()
    Ai = ra_inputs.smallint_bf16((M, lda), 91, ra_inputs.STREAM_A)
    Bi = ra_inputs.smallint_bf16((N, ldb), 91, ra_inputs.STREAM_B)
    ci, _ = run_gemm(ra, M, N, K, Ai, Bi, occ=dict(occ, tile_k=32), lda=lda, ldb=ldb, ldc=ldc)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, Ai, Bi, lda=lda, ldb=ldb)
    assert ci.tobytes() == ref16.tobytes()


@pytest.mark.parametrize("tile_k", [64, 32])
@pytest.mark.parametrize("M,N,K,occ", [
    (64, 4096, 8192, dict(cluster_k=1)),                          # swapped skinny path, 32 tiles over 148 CTAs
    (64, 4096, 8192, dict(cluster_k=1, sm_budget=74, smem_reserve_bytes=128 * 1024)),   # shallow pipeline
    (48, 2048, 4104, dict(cluster_k=1, sm_budget=40)),            # ragged M and K (4104 = 64 * 64 + 8)
    (200, 10000, 1024, dict()),                                   # non-swapped: 80 tiles of 128 x 256 over 148 CTAs
    (1000, 2000, 1032, dict(cta_group=1, cluster_k=1, sm_budget=37)),   # ragged everywhere, fix-up stores at the C edge
])
def test_stream_k_integer_exact(ra, M, N, K, occ, tile_k):
    """The stream-K fix-up (the last part to arrive sums all parts' fp32 partials in ascending-k order) against the
    oracle, bit for bit: with operands in {-2..2} every partial sum is an exact integer, so a lost, doubled or misplaced
    k-range shows in the bits.  The plan is asserted to BE stream-K (split_k > 1) at the tile_k asked for -- the cases
    that used to carry this label planned data-parallel.  PAPER.md:28 (the definition), PAPER.md:47 (occupancy shaping
    leaves the kernel's result alone)."""
    occ = dict(occ, tile_k=tile_k)
    if tile_k == 32 and not ra.ra_gemm_plan_query(0, 1, M, N, K, occ)["split_k"] > 1:
        pytest.skip("tile_k = 32 turns this shape into a data-parallel plan")
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["split_k"] > 1 and plan["tile_k"] == tile_k and plan["cluster_k"] == 1, plan
    assert ra.ra_gemm_workspace_bytes(0, 1, M, N, K, occ) > 0
    lda, ldb, ldc = _up8(K), _up8(K), _up8(N)
    A = ra_inputs.smallint_bf16((M, lda), 95, ra_inputs.STREAM_A)
    B = ra_inputs.smallint_bf16((N, ldb), 95, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, A, B, lda=lda, ldb=ldb)
    got, full = run_gemm(ra, M, N, K, A, B, occ=occ, lda=lda, ldb=ldb, ldc=ldc)
    assert np.all(full[:, N:] == 0x7FC0)
    bad = np.argwhere(got != ref16)
    assert bad.size == 0, (f"{len(bad)} of {M * N} entries differ, first at {bad[0].tolist()}", plan)
    # alpha / beta through the same fix-up path: C = 2 * acc - Cin is still exact in fp32 and mostly exact in bf16 (RNE otherwise)
    Cin = ra_inputs.smallint_bf16((M, ldc), 96, ra_inputs.STREAM_C)
    _, ref16b = oracle.gemm(0, 1, M, N, K, 2.0, A, B, -1.0, Cin, lda=lda, ldb=ldb, ldc=ldc)
    got2, _ = run_gemm(ra, M, N, K, A, B, alpha=2.0, beta=-1.0, Cin=Cin, occ=occ, lda=lda, ldb=ldb, ldc=ldc)
    assert got2.tobytes() == ref16b.tobytes()


def test_tile_k_32_is_clamped_where_it_cannot_apply(ra):
    p = ra.ra_gemm_plan_query(1, 1, 1024, 1024, 1024, dict(tile_k=32))        # MN-major A
    assert p["tile_k"] == 64 and p["clamped"] == 1
    with pytest.raises(ra.RaError):
        ra.ra_gemm_plan_query(1, 1, 1024, 1024, 1024, dict(tile_k=32, allow_clamp=0))
    with pytest.raises(ra.RaError):
        ra.ra_gemm_plan_query(0, 1, 1024, 1024, 1024, dict(tile_k=48))


@pytest.mark.parametrize("M,N,K,occ", [
    (4096, 4096, 2048, {}),                                    # 128 big tiles over 74 CTA pairs
    (4096, 4096, 1024, dict(sm_budget=20)),                    # 13 tiles per pair: many claims per worker, ring wraps
    (2048, 3000, 512, dict(cta_group=1, cluster_k=1, sm_budget=16)),   # single-CTA tiles, ragged N: always static (the knob is a no-op)
    (3000, 1000, 96, dict(cta_group=2, m_blocks=1, sm_budget=8)),      # 2 k-blocks per tile: the claim happens on the first one
    (1536, 1536, 64, dict(cta_group=2, m_blocks=1, sm_budget=4)),      # ONE k-block per tile
])
def test_dynamic_tile_order_same_bits_as_static(ra, M, N, K, occ):
    """occ.tile_order (ra.h): which worker computes a tile must not change one bit of it.  Dynamic (default) and static runs
    are compared byte for byte, the dynamic one twice (its assignment differs from run to run), and against the oracle."""
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["split_k"] == 1 and plan["cluster_k"] == 1 and plan["n_tiles"] > plan["grid"] // plan["cta_group"], plan
    A = ra_inputs.normal_bf16((M, K), 95, ra_inputs.STREAM_A)
    B = ra_inputs.normal_bf16((N, K), 95, ra_inputs.STREAM_B)
    stat, _ = run_gemm(ra, M, N, K, A, B, occ=dict(occ, tile_order=1))
    dyn1, _ = run_gemm(ra, M, N, K, A, B, occ=occ)
    dyn2, _ = run_gemm(ra, M, N, K, A, B, occ=dict(occ, tile_order=0))
    assert dyn1.tobytes() == stat.tobytes() and dyn2.tobytes() == stat.tobytes()
    ref, _ = oracle.gemm(0, 1, M, N, K, 1.0, A, B)
    rowA, colB = oracle.gemm_norms(0, 1, M, N, K, A, B)
    assert gemm_norm_err(dyn1, ref, rowA, colB) <= GEMM_TOL


def test_dynamic_tile_order_back_to_back_and_concurrent_streams(ra):
    """The claim counter and the ring live in a launch slot that re-arms itself (the last CTA out zeroes the counters and
    bumps the generation the ring tags carry; no memset in front of the kernel): 50 launches back to back on one stream,
    and two different GEMMs on two streams at once, all exact on integer operands."""
    import torch
    M, N, K = 2048, 2048, 512
    occ = dict(sm_budget=12)
    Ai = ra_inputs.smallint_bf16((M, K), 96, ra_inputs.STREAM_A)
    Bi = ra_inputs.smallint_bf16((N, K), 96, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, Ai, Bi)
    dA, dB = to_dev(Ai), to_dev(Bi)
    c1 = torch.zeros((M, N), dtype=torch.int16, device="cuda")
    c2 = torch.zeros((M, N), dtype=torch.int16, device="cuda")
    ws = torch.empty(16, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for i in range(50):
        ra.ra_gemm(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, c1, N, occ=occ, workspace=ws, stream=s1)
        if i % 5 == 0:
            ra.ra_gemm(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, c2, N, occ=dict(sm_budget=20), workspace=ws, stream=s2)
    torch.cuda.synchronize()
    assert to_host(c1, np.uint16).reshape(M, N).tobytes() == ref16.tobytes()
    assert to_host(c2, np.uint16).reshape(M, N).tobytes() == ref16.tobytes()


def test_dynamic_tile_order_same_key_on_two_streams(ra):
    """include/ra.h, tile_order: every launch in flight has a claim counter of its own.  The SAME call (pointers, shape,
    knobs -- one launch-cache entry) 50 times on each of two streams at once: with one shared counter each kernel would
    skip the tiles the other claimed and leave the poison in C.  Both streams write the same values to the same C, so
    any interleaving of correct launches gives the oracle's bits (integer operands: exact)."""
    import torch
    M, N, K = 2048, 2048, 512
    occ = dict(sm_budget=24)                       # 12 workers x 512 x 256 tiles, 32 tiles: dynamic order, room for both kernels
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cta_group"] == 2 and plan["split_k"] == 1 and plan["n_tiles"] > plan["grid"] // 2, plan
    Ai = ra_inputs.smallint_bf16((M, K), 97, ra_inputs.STREAM_A)
    Bi = ra_inputs.smallint_bf16((N, K), 97, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, Ai, Bi)
    dA, dB = to_dev(Ai), to_dev(Bi)
    ws = torch.empty(16, dtype=torch.uint8, device="cuda")
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    for rep in range(3):
        dC = torch.full((M, N), 0x7FC0, dtype=torch.int16, device="cuda")
        torch.cuda.synchronize()
        for i in range(50):
            ra.ra_gemm(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, dC, N, occ=occ, workspace=ws, stream=s1)
            ra.ra_gemm(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, dC, N, occ=occ, workspace=ws, stream=s2)
        torch.cuda.synchronize()
        assert to_host(dC, np.uint16).reshape(M, N).tobytes() == ref16.tobytes(), rep


def test_dynamic_tile_order_more_keys_in_flight_than_cache_entries(ra):
    """40 distinct calls (40 output buffers -> 40 launch-cache keys) cycled three times through the 32-entry cache over
    four streams without a synchronisation in between: evictions happen while earlier launches are still running.  A
    launch slot is handed out only once its previous launch has completed (else the launch takes the static order), so
    every C must equal the oracle's bits."""
    import torch
    M, N, K = 1536, 2048, 512
    occ = dict(sm_budget=16)
    plan = ra.ra_gemm_plan_query(0, 1, M, N, K, occ)
    assert plan["cta_group"] == 2 and plan["n_tiles"] > plan["grid"] // 2, plan
    Ai = ra_inputs.smallint_bf16((M, K), 98, ra_inputs.STREAM_A)
    Bi = ra_inputs.smallint_bf16((N, K), 98, ra_inputs.STREAM_B)
    _, ref16 = oracle.gemm(0, 1, M, N, K, 1.0, Ai, Bi)
    dA, dB = to_dev(Ai), to_dev(Bi)
    ws = torch.empty(16, dtype=torch.uint8, device="cuda")
    cs = [torch.full((M, N), 0x7FC0, dtype=torch.int16, device="cuda") for _ in range(40)]
    streams = [torch.cuda.Stream() for _ in range(4)]
    torch.cuda.synchronize()
    for rnd in range(3):
        for i, c in enumerate(cs):
            ra.ra_gemm(0, 1, M, N, K, 1.0, dA, K, dB, K, 0.0, c, N, occ=occ, workspace=ws, stream=streams[(i + rnd) % 4])
    torch.cuda.synchronize()
    for i, c in enumerate(cs):
        assert to_host(c, np.uint16).reshape(M, N).tobytes() == ref16.tobytes(), i
