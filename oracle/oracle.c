/*
 * oracle/oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of what the hot path of
 * arxiv/paper_2606_09200 computes.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library; the
 * product (paper_2606_09200_b200/) never does.  It shares no code with the CUDA
 * path: no common header, helper, table or constant.
 *
 * Every function is the DEFINITION of its result written out (the kernels reach
 * exactly that result, the GEMM up to floating-point summation order), so there
 * is no blocking, fusion or reordering here -- only an OpenMP split of the
 * outermost loop over independent outputs.
 *
 *   oracle_gemm*      PAPER.md:28  (section 2.1)  C = alpha*op(A)*op(B) + beta*C,
 *                     A in R^{MxK}, B in R^{KxN}, C in R^{MxN}.  dtype reading A1
 *                     (DESIGN.md): bf16 inputs, result kept in fp64 (+ bf16 RNE copy).
 *   oracle_allreduce  PAPER.md:30  (section 2.2) allreduce "aggregated across all
 *                     GPUs"; BASELINE.json north_star fixes the single-device
 *                     stand-in: fixed rank-order fp32 sum, written back to all P.
 *   oracle_alltoall   PAPER.md:30, 94 alltoall "route tokens between devices";
 *                     stand-in: chunk (i,j) -> (j,i), bytewise.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): long-double brute force
 * written in the test, identity/zero/ones closed forms, rank-1 closed form,
 * integer-exact inputs, numpy float64 matmul (independent library), order
 * detectors 2^24+1+..+1, denormal pin, involution, tagged payload, checksums.
 * No function here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -fno-fast-math -ffp-contract=off -fopenmp (oracle/__init__.py).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

/* ---- bf16 <-> fp32 ------------------------------------------------------- */
/* bf16 is the upper 16 bits of an IEEE-754 binary32: widening is exact. */
static inline float bf16_to_f32(uint16_t b) {
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, 4);
    return f;
}

/* round-to-nearest-even on the 16 dropped bits; NaN stays NaN (quiet). */
static inline uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x0040u);
    uint32_t lsb = (u >> 16) & 1u;
    u += 0x7FFFu + lsb;
    return (uint16_t)(u >> 16);
}

void oracle_bf16_to_f32(const uint16_t* in, float* out, size_t n) {
    for (size_t i = 0; i < n; ++i) out[i] = bf16_to_f32(in[i]);
}
void oracle_f32_to_bf16(const float* in, uint16_t* out, size_t n) {
    for (size_t i = 0; i < n; ++i) out[i] = f32_to_bf16_rne(in[i]);
}

/* ---- O1: GEMM ----------------------------------------------
 * Row-major buffers.  transA=0: A is M x K (lda >= K), op(A)(i,k) = A[i*lda+k];
 * transA=1: A is K x M (lda >= M), op(A)(i,k) = A[k*lda+i].
 * transB=0: B is K x N (ldb >= N), op(B)(k,j) = B[k*ldb+j];
 * transB=1: B is N x K (ldb >= K), op(B)(k,j) = B[j*ldb+k].
 * beta == 0 => C_in is not read (BLAS semantics, reading A14). */
static inline double opA(const uint16_t* A, int lda, int transA, long i, long k) {
    return (double)bf16_to_f32(transA ? A[k * (long)lda + i] : A[i * (long)lda + k]);
}
static inline double opB(const uint16_t* B, int ldb, int transB, long k, long j) {
    return (double)bf16_to_f32(transB ? B[j * (long)ldb + k] : B[k * (long)ldb + j]);
}

static inline double gemm_entry(int transA, int transB, int K, double alpha, const uint16_t* A, int lda,
                                const uint16_t* B, int ldb, double beta, const uint16_t* Cin, int ldc,
                                long i, long j) {
    double acc = 0.0;
    for (long k = 0; k < K; ++k) acc += opA(A, lda, transA, i, k) * opB(B, ldb, transB, k, j);
    double r = alpha * acc;
    if (beta != 0.0) r += beta * (double)bf16_to_f32(Cin[i * (long)ldc + j]);
    return r;
}

/* Full result.  ref: M x N doubles (ld = N).  ref_bf16 (optional, may be NULL):
 * the same values rounded fp64 -> fp32 -> bf16 RNE, M x N (ld = N). */
void oracle_gemm(int transA, int transB, int M, int N, int K, float alpha, const uint16_t* A, int lda,
                 const uint16_t* B, int ldb, float beta, const uint16_t* Cin, int ldc, double* ref,
                 uint16_t* ref_bf16) {
#pragma omp parallel for schedule(dynamic, 1)
    for (long i = 0; i < M; ++i)
        for (long j = 0; j < N; ++j) {
            double r = gemm_entry(transA, transB, K, (double)alpha, A, lda, B, ldb, (double)beta, Cin, ldc, i, j);
            ref[i * (long)N + j] = r;
            if (ref_bf16) ref_bf16[i * (long)N + j] = f32_to_bf16_rne((float)r);
        }
}

/* Sampled entries: ref[s] = C(ii[s], jj[s]) -- lets the full-size configs be
 * checked entry by entry without computing all M*N entries. */
void oracle_gemm_samples(int transA, int transB, int M, int N, int K, float alpha, const uint16_t* A, int lda,
                         const uint16_t* B, int ldb, float beta, const uint16_t* Cin, int ldc,
                         const int64_t* ii, const int64_t* jj, size_t n_samples, double* ref) {
    (void)M; (void)N;
#pragma omp parallel for schedule(dynamic, 16)
    for (long s = 0; s < (long)n_samples; ++s)
        ref[s] = gemm_entry(transA, transB, K, (double)alpha, A, lda, B, ldb, (double)beta, Cin, ldc, ii[s], jj[s]);
}

/* 2-norms used by the acceptance metric (BASELINE.json: "max-abs normalised by
 * |A||B| row/column norms"): rowA[i] = ||op(A)(i,:)||_2, colB[j] = ||op(B)(:,j)||_2. */
void oracle_gemm_norms(int transA, int transB, int M, int N, int K, const uint16_t* A, int lda,
                       const uint16_t* B, int ldb, double* rowA, double* colB) {
#pragma omp parallel for schedule(static)
    for (long i = 0; i < M; ++i) {
        double s = 0.0;
        for (long k = 0; k < K; ++k) { double v = opA(A, lda, transA, i, k); s += v * v; }
        rowA[i] = sqrt(s);
    }
#pragma omp parallel for schedule(static)
    for (long j = 0; j < N; ++j) {
        double s = 0.0;
        for (long k = 0; k < K; ++k) { double v = opB(B, ldb, transB, k, j); s += v * v; }
        colB[j] = sqrt(s);
    }
}

/* ---- O2: allreduce stand-in (BASELINE.json north_star) --------
 * for every element e: s = b0[e]; s = s + b1[e]; ...; s = s + b_{P-1}[e]  (each +
 * one IEEE-754 binary32 RNE add, this order), then b_r[e] = s for all r.
 * `volatile` pins each partial sum to a binary32 store so no wider intermediate
 * or reassociation can be introduced by the compiler. */
void oracle_allreduce(float* const* bufs, int P, size_t count) {
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < (long long)count; ++e) {
        volatile float s = bufs[0][e];
        for (int r = 1; r < P; ++r) s = s + bufs[r][e];
        for (int r = 0; r < P; ++r) bufs[r][e] = s;
    }
}

/* ---- O3: alltoall stand-in (BASELINE.json) -----------------
 * recv[(j*P+i)] <- send[(i*P+j)] for all chunks, bytewise. */
void oracle_alltoall(const void* send, void* recv, int P, size_t chunk_bytes) {
#pragma omp parallel for schedule(static) collapse(2)
    for (int i = 0; i < P; ++i)
        for (int j = 0; j < P; ++j)
            memcpy((char*)recv + ((size_t)j * P + i) * chunk_bytes,
                   (const char*)send + ((size_t)i * P + j) * chunk_bytes, chunk_bytes);
}

int oracle_num_threads(void);
#ifdef _OPENMP
#include <omp.h>
int oracle_num_threads(void) { return omp_get_max_threads(); }
void oracle_set_threads(int n) { omp_set_num_threads(n); }
#else
int oracle_num_threads(void) { return 1; }
void oracle_set_threads(int n) { (void)n; }
#endif
