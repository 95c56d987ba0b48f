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

// ALL = true: the sum goes back to every rank buffer.  ALL = false (variant 2): to buffer 0 only, the copy engines fan it
// out afterwards.  A template parameter: as a run-time store predicate it cost the all-buffers kernel 4 % (171 -> 178 us).
template <int P, bool ALL>
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
        for (int r = 0; r < (ALL ? P : 1); ++r) st_stream(reinterpret_cast<float4*>(ptrs.p[r]) + v, s);
    }
    // ragged tail: count % 4 scalars
    if (blockIdx.x == 0) {
        const size_t e = (nvec << 2) + threadIdx.x;
        if (threadIdx.x < 4 && e < count) {
            float s = ptrs.p[0][e];
#pragma unroll
            for (int r = 1; r < P; ++r) s = __fadd_rn(s, ptrs.p[r][e]);
#pragma unroll
            for (int r = 0; r < (ALL ? P : 1); ++r) ptrs.p[r][e] = s;
        }
    }
    if (threadIdx.x == 0) trace_end(rec);
}

// ---- variant 1: TMA-ring allreduce ------------------------------------------------------------------------------
// The same arithmetic with the data path of the alltoall stand-in: per work unit (one slice of `slice` floats) a single
// thread bulk-loads the P rank slices into a shared-memory slot (cp.async.bulk, mbarrier complete_tx), the CTA's threads
// sum them from shared memory in rank order -- 128-bit ld.shared, the same left-to-right fp32 chain per element, so the
// result is bit-identical to variant 0 and to the oracle -- into the slot's first slice, and the thread bulk-stores that
// slice to all P buffers.  Two slots: the loads of unit t+1 are in flight while unit t is summed.  The kernel needs few
// threads and registers but P * slice * 4 bytes of shared memory per slot: a collective whose co-residency with the GEMM
// IS decided by smem_reserve_bytes, and one that saturates HBM from few SMs.
constexpr int kArTmaThreads = 128;
constexpr int kArTmaSlots = 2;

__device__ __forceinline__ void ar_bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void ar_bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes, uint64_t policy) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst),
                 "r"(src_smem), "r"(bytes), "l"(policy)
                 : "memory");
}

struct ArTmaParams {
    ArPtrs ptrs;
    int P;
    uint32_t slice;          // floats per slice (multiple of 4)
    uint64_t nvec_floats;    // count rounded down to a multiple of 4: the part moved in 16-byte pieces
    uint64_t count;
    uint64_t n_units;        // ceil(nvec_floats / slice)
};

__global__ void __launch_bounds__(kArTmaThreads)
allreduce_tma_kernel(const __grid_constant__ ArTmaParams p, Trace tr) {
    extern __shared__ __align__(128) uint8_t ar_smem[];
    __shared__ __align__(8) uint64_t full_bar[kArTmaSlots];
    uint64_t* rec = (threadIdx.x == 0) ? trace_begin(tr, KID_ALLREDUCE) : nullptr;
    const uint32_t slot_bytes = (uint32_t)p.P * p.slice * 4u;
    const uint32_t smem_base = smem_u32(ar_smem);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kArTmaSlots; ++s) mbar_init(smem_u32(&full_bar[s]), 1);
        mbar_fence_init();
    }
    __syncthreads();
    const uint64_t policy = policy_evict_first();
    const uint64_t G = gridDim.x, first = blockIdx.x;
    const uint64_t n_my = first < p.n_units ? (p.n_units - first + G - 1) / G : 0;
    auto unit_floats = [&](uint64_t u) -> uint32_t {
        const uint64_t off = u * p.slice, left = p.nvec_floats - off;
        return left < p.slice ? (uint32_t)left : p.slice;
    };
    auto issue_loads = [&](uint64_t t) {                 // thread 0 only
        const uint32_t slot = (uint32_t)(t % kArTmaSlots);
        const uint64_t u = first + t * G;
        const uint32_t nf = unit_floats(u);
        const uint32_t bar = smem_u32(&full_bar[slot]);
        mbar_expect_tx(bar, (uint32_t)p.P * nf * 4u);
        for (int r = 0; r < p.P; ++r)
            ar_bulk_g2s(smem_base + slot * slot_bytes + (uint32_t)r * p.slice * 4u, p.ptrs.p[r] + u * p.slice, nf * 4u, bar, policy);
    };
    if (threadIdx.x == 0 && n_my > 0) issue_loads(0);
    for (uint64_t t = 0; t < n_my; ++t) {
        const uint32_t slot = (uint32_t)(t % kArTmaSlots);
        const uint64_t u = first + t * G;
        const uint32_t nf = unit_floats(u);
        if (threadIdx.x == 0 && t + 1 < n_my) {
            // the other slot was last read by the stores of unit t-1: they must have drained it before it is refilled
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            issue_loads(t + 1);
        }
        mbar_wait(smem_u32(&full_bar[slot]), (uint32_t)((t / kArTmaSlots) & 1));
        const uint32_t base = smem_base + slot * slot_bytes;
        for (uint32_t v = threadIdx.x; v < nf / 4; v += kArTmaThreads) {
            float4 s;
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(s.x), "=f"(s.y), "=f"(s.z), "=f"(s.w) : "r"(base + v * 16u));
            for (int r = 1; r < p.P; ++r) {
                float4 x;
                asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w)
                             : "r"(base + (uint32_t)r * p.slice * 4u + v * 16u));
                s.x = __fadd_rn(s.x, x.x);
                s.y = __fadd_rn(s.y, x.y);
                s.z = __fadd_rn(s.z, x.z);
                s.w = __fadd_rn(s.w, x.w);
            }
            asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(base + v * 16u), "f"(s.x), "f"(s.y), "f"(s.z), "f"(s.w) : "memory");
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int r = 0; r < p.P; ++r) ar_bulk_s2g(p.ptrs.p[r] + u * p.slice, base, nf * 4u, policy);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    // ragged tail: count % 4 scalars
    if (blockIdx.x == 0 && threadIdx.x < 4) {
        const uint64_t e = p.nvec_floats + threadIdx.x;
        if (e < p.count) {
            float s = p.ptrs.p[0][e];
            for (int r = 1; r < p.P; ++r) s = __fadd_rn(s, p.ptrs.p[r][e]);
            for (int r = 0; r < p.P; ++r) p.ptrs.p[r][e] = s;
        }
    }
    if (threadIdx.x == 0) trace_end(rec);
}

template <int P>
static cudaError_t launch_ar(const ArPtrs& ptrs, size_t count, bool all, int grid, cudaStream_t stream) {
    if (all) allreduce_kernel<P, true><<<grid, kArThreads, 0, stream>>>(ptrs, count, g_trace);
    else allreduce_kernel<P, false><<<grid, kArThreads, 0, stream>>>(ptrs, count, g_trace);
    return cudaGetLastError();
}

// Argument rules of ra_allreduce_emul(_ex); also called by the overlap driver BEFORE it enqueues anything.
ra_status allreduce_validate(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, int smem_bytes_per_cta,
                             int variant) {
    if (bufs == nullptr || P < 1 || P > RA_MAX_RANKS) return RA_ERR_INVALID_ARG;
    if (sm_budget < 0 || ctas_per_sm < 0 || ctas_per_sm > kArCtasPerSm) return RA_ERR_INVALID_ARG;
    if (smem_bytes_per_cta < 0 || variant < 0 || variant > 2) return RA_ERR_INVALID_ARG;
    for (int r = 0; r < P; ++r)
        if (bufs[r] == nullptr || (reinterpret_cast<uintptr_t>(bufs[r]) & 15u)) return RA_ERR_INVALID_ARG;
    const size_t bytes = count * sizeof(float);
    for (int a = 0; a < P; ++a)
        for (int b = a + 1; b < P; ++b) {
            const uintptr_t pa = reinterpret_cast<uintptr_t>(bufs[a]), pb = reinterpret_cast<uintptr_t>(bufs[b]);
            if (pa < pb + bytes && pb < pa + bytes && bytes > 0) return RA_ERR_INVALID_ARG;
            if (pa == pb) return RA_ERR_INVALID_ARG;
        }
    if (variant == 1 && count > 0) {          // the TMA ring needs at least one 128-byte slice per rank and slot
        const int smem = smem_bytes_per_cta ? smem_bytes_per_cta : 64 * 1024;
        if ((((uint32_t)smem / (uint32_t)(kArTmaSlots * P * 4)) & ~31u) < 32) return RA_ERR_INVALID_ARG;
    }
    return RA_OK;
}

ra_status allreduce_launch(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, int smem_bytes_per_cta,
                           int variant, cudaStream_t stream) {
    RA_TRY(allreduce_validate(bufs, P, count, sm_budget, ctas_per_sm, smem_bytes_per_cta, variant));
    ArPtrs ptrs{};
    for (int r = 0; r < P; ++r) ptrs.p[r] = bufs[r];
    if (count == 0) return RA_OK;

    DeviceInfo di;
    RA_TRY(device_info(&di));
    RA_TRY(require_sm100(di));
    RA_TRY(l2_persist_first_use(stream));
    int sms = (sm_budget == 0 || sm_budget > di.sm_count) ? di.sm_count : sm_budget;
    if (variant == 1) {
        int smem = smem_bytes_per_cta ? smem_bytes_per_cta : 64 * 1024;
        const int max_dyn = di.smem_per_block_optin - 256;
        if (smem > max_dyn) smem = max_dyn;
        // slice: floats per rank per slot, a multiple of 32 floats (128 bytes)
        uint32_t slice = ((uint32_t)smem / (uint32_t)(kArTmaSlots * P * 4)) & ~31u;
        if (slice < 32) return RA_ERR_INVALID_ARG;
        ArTmaParams tp{};
        tp.ptrs = ptrs;
        tp.P = P;
        tp.count = count;
        tp.nvec_floats = count & ~(size_t)3;
        if (tp.nvec_floats < slice) slice = (uint32_t)((tp.nvec_floats + 31) & ~(size_t)31);
        if (slice == 0) slice = 32;
        tp.slice = slice;
        tp.n_units = (tp.nvec_floats + slice - 1) / slice;
        const int dyn = (int)(kArTmaSlots * P * slice * 4);
        uint64_t grid = (uint64_t)sms * (ctas_per_sm ? ctas_per_sm : 2);
        if (grid > tp.n_units) grid = tp.n_units;
        if (grid == 0) grid = 1;                                   // count < 4: only the scalar tail
        if (dyn > 48 * 1024)
            RA_CUDA(cudaFuncSetAttribute(allreduce_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn));
            // same split as the GEMM asks for, so that either kernel can join the other on an SM (see prepare_kernel in ra_gemm.cu)
            RA_CUDA(cudaFuncSetAttribute(allreduce_tma_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        allreduce_tma_kernel<<<(unsigned)grid, kArTmaThreads, dyn, stream>>>(tp, g_trace);
        RA_CUDA(cudaGetLastError());
        return RA_OK;
    }
    const size_t nvec = count >> 2;
    size_t want = (nvec + kArThreads - 1) / kArThreads;
    if (want == 0) want = 1;
    size_t grid = (size_t)sms * (ctas_per_sm ? ctas_per_sm : kArDefaultCtasPerSm);
    if (grid > want) grid = want;

    cudaError_t e;
    switch (P) {
#define RA_AR_CASE(n) case n: e = launch_ar<n>(ptrs, count, variant != 2, (int)grid, stream); break;
        RA_AR_CASE(1) RA_AR_CASE(2) RA_AR_CASE(3) RA_AR_CASE(4) RA_AR_CASE(5) RA_AR_CASE(6) RA_AR_CASE(7) RA_AR_CASE(8)
        RA_AR_CASE(9) RA_AR_CASE(10) RA_AR_CASE(11) RA_AR_CASE(12) RA_AR_CASE(13) RA_AR_CASE(14) RA_AR_CASE(15)
        RA_AR_CASE(16)
#undef RA_AR_CASE
        default: return RA_ERR_INVALID_ARG;
    }
    RA_CUDA(e);
    if (variant == 2) {
        // the all-gather half on the copy engines (the mechanism of ConCCL's DMA offload): the kernel above
        // wrote the sum to buffer 0 only -- 4P + 4 bytes per element through the SMs instead of 8P -- and P-1
        // device-to-device copies, ordered after it on the same stream, put it into the other rank buffers without a
        // resident CTA.  Same bits; 12P - 4 bytes of HBM traffic per element instead of 8P.
        for (int r = 1; r < P; ++r)
            RA_CUDA(cudaMemcpyAsync(bufs[r], bufs[0], count * sizeof(float), cudaMemcpyDeviceToDevice, stream));
    }
    return RA_OK;
}

}  // namespace ra

extern "C" {
ra_status ra_allreduce_emul(float* const* bufs, int P, size_t count, int sm_budget, void* stream) {
    return ra::allreduce_launch(bufs, P, count, sm_budget, 0, 0, 0, static_cast<cudaStream_t>(stream));
}
ra_status ra_allreduce_emul_ex(float* const* bufs, int P, size_t count, int sm_budget, int smem_bytes_per_cta, int ctas_per_sm,
                               int variant, void* stream) {
    return ra::allreduce_launch(bufs, P, count, sm_budget, ctas_per_sm, smem_bytes_per_cta, variant,
                                static_cast<cudaStream_t>(stream));
}
}
