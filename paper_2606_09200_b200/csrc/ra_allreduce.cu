// ra_allreduce.cu -- K2: single-device allreduce stand-in (S4, BASELINE.json north_star).
//
//   bufs[r][e] <- ((bufs[0][e] + bufs[1][e]) + ...) + bufs[P-1][e]      for all r, e   (fp32, RNE, this order)
//
// HBM-bound: per element index 4P bytes read + 4P bytes written, P-1 adds.  One thread owns one
// 16-byte vector index per grid-stride step: P independent 128-bit streaming loads are issued
// before the first add (P*16 B in flight per thread), four independent left-to-right chains (one
// per vector lane), then P 128-bit streaming stores.  No shared memory, no TMEM: the kernel can
// co-reside with a GEMM CTA on any SM that has thread/register room (the property the paper
// relies on: "communication kernels are intentionally lightweight and low-occupancy").
// Compiled without fast-math: add.rn.f32 keeps denormals (oracle pin "denormal").
#include "ra_common.cuh"

namespace ra {

struct ArPtrs {
    float* p[RA_MAX_RANKS];
};

// 256 threads x <= 64 registers: 2 warps x 2048 registers per SM sub-partition.  The register file is
// split four ways (16 K registers per sub-partition), and a resident tcgen05 GEMM CTA (6 warps x 160
// registers) leaves only 6 K free in two of them -- a 512-thread CTA (8 K per sub-partition) measured
// 0.03 % co-residency with the GEMM (bench.py residency map), a 256-thread CTA fits.
constexpr int kArThreads = 256;
constexpr int kArCtasPerSm = 4;          // launch bound (registers); the default grid uses kArDefaultCtasPerSm
constexpr int kArDefaultCtasPerSm = 2;

__device__ __forceinline__ float4 ld_stream(const float4* p) {
    float4 v;
    // .cs = cache-streaming (evict-first): the buffers are touched once and must not displace the
    // GEMM's operand tiles in L2.  Not .nc: the same kernel writes these addresses.
    asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(float4* p, float4 v) {
    asm volatile("st.global.cs.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
                 : "memory");
}

template <int P>
__global__ void __launch_bounds__(kArThreads, kArCtasPerSm)
allreduce_kernel(const __grid_constant__ ArPtrs ptrs, size_t count, Trace tr) {
    uint64_t* rec = (threadIdx.x == 0) ? trace_begin(tr, KID_ALLREDUCE) : nullptr;

    const size_t nvec = count >> 2;
    const size_t stride = (size_t)gridDim.x * kArThreads;
    for (size_t v = (size_t)blockIdx.x * kArThreads + threadIdx.x; v < nvec; v += stride) {
        // loads are issued in batches of <= 8 ranks (128 B in flight per thread per batch) so that
        // P = 16 does not spill; the running sum crosses batches in rank order.
        float4 s;
#pragma unroll
        for (int b = 0; b < P; b += 8) {
            constexpr int kB = 8;
            float4 x[kB];
#pragma unroll
            for (int r = 0; r < kB; ++r)
                if (b + r < P) x[r] = ld_stream(reinterpret_cast<const float4*>(ptrs.p[b + r]) + v);
#pragma unroll
            for (int r = 0; r < kB; ++r) {
                if (b + r >= P) continue;
                if (b + r == 0) {
                    s = x[0];
                } else {
                    s.x = __fadd_rn(s.x, x[r].x);
                    s.y = __fadd_rn(s.y, x[r].y);
                    s.z = __fadd_rn(s.z, x[r].z);
                    s.w = __fadd_rn(s.w, x[r].w);
                }
            }
        }
#pragma unroll
        for (int r = 0; r < P; ++r) st_stream(reinterpret_cast<float4*>(ptrs.p[r]) + v, s);
    }
    // ragged tail: count % 4 scalars
    if (blockIdx.x == 0) {
        const size_t e = (nvec << 2) + threadIdx.x;
        if (threadIdx.x < 4 && e < count) {
            float s = ptrs.p[0][e];
#pragma unroll
            for (int r = 1; r < P; ++r) s = __fadd_rn(s, ptrs.p[r][e]);
#pragma unroll
            for (int r = 0; r < P; ++r) ptrs.p[r][e] = s;
        }
    }
    if (threadIdx.x == 0) trace_end(rec);
}

template <int P>
static cudaError_t launch_ar(const ArPtrs& ptrs, size_t count, int grid, cudaStream_t stream) {
    allreduce_kernel<P><<<grid, kArThreads, 0, stream>>>(ptrs, count, g_trace);
    return cudaGetLastError();
}

ra_status allreduce_launch(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, cudaStream_t stream) {
    if (bufs == nullptr || P < 1 || P > RA_MAX_RANKS) return RA_ERR_INVALID_ARG;
    if (sm_budget < 0 || ctas_per_sm < 0 || ctas_per_sm > kArCtasPerSm) return RA_ERR_INVALID_ARG;
    ArPtrs ptrs{};
    for (int r = 0; r < P; ++r) {
        if (bufs[r] == nullptr || (reinterpret_cast<uintptr_t>(bufs[r]) & 15u)) return RA_ERR_INVALID_ARG;
        ptrs.p[r] = bufs[r];
    }
    const size_t bytes = count * sizeof(float);
    for (int a = 0; a < P; ++a)
        for (int b = a + 1; b < P; ++b) {
            const uintptr_t pa = reinterpret_cast<uintptr_t>(bufs[a]), pb = reinterpret_cast<uintptr_t>(bufs[b]);
            if (pa < pb + bytes && pb < pa + bytes && bytes > 0) return RA_ERR_INVALID_ARG;
            if (pa == pb) return RA_ERR_INVALID_ARG;
        }
    if (count == 0) return RA_OK;

    DeviceInfo di;
    RA_TRY(device_info(&di));
    RA_TRY(require_sm100(di));
    int sms = (sm_budget == 0 || sm_budget > di.sm_count) ? di.sm_count : sm_budget;
    const size_t nvec = count >> 2;
    size_t want = (nvec + kArThreads - 1) / kArThreads;
    if (want == 0) want = 1;
    size_t grid = (size_t)sms * (ctas_per_sm ? ctas_per_sm : kArDefaultCtasPerSm);
    if (grid > want) grid = want;

    cudaError_t e;
    switch (P) {
#define RA_AR_CASE(n) case n: e = launch_ar<n>(ptrs, count, (int)grid, stream); break;
        RA_AR_CASE(1) RA_AR_CASE(2) RA_AR_CASE(3) RA_AR_CASE(4) RA_AR_CASE(5) RA_AR_CASE(6) RA_AR_CASE(7) RA_AR_CASE(8)
        RA_AR_CASE(9) RA_AR_CASE(10) RA_AR_CASE(11) RA_AR_CASE(12) RA_AR_CASE(13) RA_AR_CASE(14) RA_AR_CASE(15)
        RA_AR_CASE(16)
#undef RA_AR_CASE
        default: return RA_ERR_INVALID_ARG;
    }
    RA_CUDA(e);
    return RA_OK;
}

}  // namespace ra

extern "C" {
ra_status ra_allreduce_emul(float* const* bufs, int P, size_t count, int sm_budget, void* stream) {
    return ra::allreduce_launch(bufs, P, count, sm_budget, 0, static_cast<cudaStream_t>(stream));
}
ra_status ra_allreduce_emul_ex(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, void* stream) {
    return ra::allreduce_launch(bufs, P, count, sm_budget, ctas_per_sm, static_cast<cudaStream_t>(stream));
}
}
