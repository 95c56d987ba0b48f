// ra_alltoall.cu -- K3: single-device alltoall stand-in (S5; BASELINE.json).
//
//   recv[(j*P + i)*chunk_bytes + b] = send[(i*P + j)*chunk_bytes + b]
//
// Pure byte movement, HBM-bound (2*chunk_bytes per chunk).  Variant 0 moves the data with TMA
// bulk copies: one elected thread per CTA drives a ring of R shared-memory slots,
//   cp.async.bulk global->shared (mbarrier complete_tx)  ->  cp.async.bulk shared->global (bulk group),
// so the SM's LSU and register file stay idle -- the only SM resource the kernel holds is its
// shared-memory ring, which is exactly what the GEMM's smem_reserve_bytes knob makes room for.
// Variant 1 is a plain 128-bit LDG/STG copy with no shared memory.  Neither touches TMEM.
// Variant 2 uses no SM at all: one cudaMemcpyAsync (copy engine) per chunk.
#include "ra_common.cuh"

namespace ra {

constexpr int kA2aThreads = 32;       // variant 0: one warp, one issuing lane
constexpr int kA2aSlots = 4;          // ring depth R
constexpr int kA2aDefaultSmem = 64 * 1024;
constexpr int kA2aDefaultCtasPerSm = 2;
constexpr int kCopyThreads = 256;     // variant 1
constexpr int kCopyUnroll = 4;
constexpr int kCopyCtasPerSm = 4;

__device__ __forceinline__ void bulk_g2s(uint32_t dst_smem, const void* src, uint32_t bytes, uint32_t bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst_smem), "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src_smem, uint32_t bytes, uint64_t policy) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst),
                 "r"(src_smem), "r"(bytes), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
template <int N>
__device__ __forceinline__ void bulk_wait_all() {
    asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory");
}

struct A2aParams {
    const uint8_t* send;
    uint8_t* recv;
    uint8_t* peer_recv[RA_MAX_RANKS];   // peer mode (ra_alltoall_peer): rank j's receive buffer; `send` is this rank's row
    int32_t peer_rank;                  // -1: single-device emulation (send / recv hold all P x P chunks)
    uint32_t P;
    uint32_t slice_bytes;        // S: bytes per ring slot
    uint64_t chunk_bytes;
    uint32_t slices_per_chunk;   // ceil(chunk_bytes / S)
    uint64_t n_units;            // P*P*slices_per_chunk
};

__device__ __forceinline__ void a2a_unit(const A2aParams& p, uint64_t u, const uint8_t*& src, uint8_t*& dst,
                                         uint32_t& bytes) {
    const uint64_t c = u / p.slices_per_chunk;
    const uint32_t s = (uint32_t)(u - c * p.slices_per_chunk);
    const uint64_t off = (uint64_t)s * p.slice_bytes;
    const uint64_t left = p.chunk_bytes - off;
    bytes = left < p.slice_bytes ? (uint32_t)left : p.slice_bytes;
    if (p.peer_rank >= 0) {                   // chunk c of this rank's row goes to slot `rank` of rank c's buffer
        src = p.send + c * p.chunk_bytes + off;
        dst = p.peer_recv[c] + (uint64_t)p.peer_rank * p.chunk_bytes + off;
        return;
    }
    const uint32_t i = (uint32_t)(c / p.P), j = (uint32_t)(c - (uint64_t)i * p.P);
    src = p.send + ((uint64_t)i * p.P + j) * p.chunk_bytes + off;
    dst = p.recv + ((uint64_t)j * p.P + i) * p.chunk_bytes + off;
}

__global__ void __launch_bounds__(kA2aThreads)
alltoall_tma_kernel(const A2aParams p, Trace tr) {
    extern __shared__ __align__(128) uint8_t smem[];
    __shared__ __align__(8) uint64_t full_bar[kA2aSlots];

    if (threadIdx.x != 0) return;  // one issuing thread; the rest of the warp only exists to fill the launch
    uint64_t* rec = trace_begin(tr, KID_ALLTOALL);

#pragma unroll
    for (int s = 0; s < kA2aSlots; ++s) mbar_init(smem_u32(&full_bar[s]), 1);
    mbar_fence_init();

    const uint64_t policy = policy_evict_first();  // payload is touched once: keep it out of the GEMM's L2 set
    const uint64_t G = gridDim.x;
    const uint64_t first = blockIdx.x;
    const uint64_t n_my = first < p.n_units ? (p.n_units - first + G - 1) / G : 0;
    const uint32_t smem_base = smem_u32(smem);

    auto issue_load = [&](uint64_t t) {
        const uint32_t slot = (uint32_t)(t % kA2aSlots);
        const uint8_t* src;
        uint8_t* dst;
        uint32_t bytes;
        a2a_unit(p, first + t * G, src, dst, bytes);
        const uint32_t bar = smem_u32(&full_bar[slot]);
        mbar_expect_tx(bar, bytes);
        bulk_g2s(smem_base + slot * p.slice_bytes, src, bytes, bar, policy);
    };

    const uint64_t pro = n_my < (uint64_t)(kA2aSlots - 1) ? n_my : (uint64_t)(kA2aSlots - 1);
    for (uint64_t t = 0; t < pro; ++t) issue_load(t);

    for (uint64_t t = 0; t < n_my; ++t) {
        const uint32_t slot = (uint32_t)(t % kA2aSlots);
        mbar_wait(smem_u32(&full_bar[slot]), (uint32_t)((t / kA2aSlots) & 1));
        const uint8_t* src;
        uint8_t* dst;
        uint32_t bytes;
        a2a_unit(p, first + t * G, src, dst, bytes);
        bulk_s2g(dst, smem_base + slot * p.slice_bytes, bytes, policy);
        bulk_commit();
        const uint64_t nt = t + kA2aSlots - 1;
        if (nt < n_my) {
            // slot of unit nt was last read by the store of unit t-1: all groups but the newest must
            // have finished READING shared memory before the slot is overwritten.
            bulk_wait_read<1>();
            issue_load(nt);
        }
    }
    bulk_wait_all<0>();
    trace_end(rec);
}

// variant 1: LDG/STG.  Unit = (chunk, 64 KiB block of it); threads copy 16 B each, 4 in flight.
__global__ void __launch_bounds__(kCopyThreads)
alltoall_ldg_kernel(const A2aParams p, Trace tr) {
    uint64_t* rec = (threadIdx.x == 0) ? trace_begin(tr, KID_ALLTOALL) : nullptr;
    for (uint64_t u = blockIdx.x; u < p.n_units; u += gridDim.x) {
        const uint8_t* src;
        uint8_t* dst;
        uint32_t bytes;
        a2a_unit(p, u, src, dst, bytes);
        const uint32_t nvec = bytes >> 4;
        const int4* s4 = reinterpret_cast<const int4*>(src);
        int4* d4 = reinterpret_cast<int4*>(dst);
        for (uint32_t v = threadIdx.x; v < nvec; v += kCopyThreads * kCopyUnroll) {
            int4 x[kCopyUnroll];
#pragma unroll
            for (int k = 0; k < kCopyUnroll; ++k)
                if (v + k * kCopyThreads < nvec) x[k] = __ldcs(s4 + v + k * kCopyThreads);
#pragma unroll
            for (int k = 0; k < kCopyUnroll; ++k)
                if (v + k * kCopyThreads < nvec) __stcs(d4 + v + k * kCopyThreads, x[k]);
        }
    }
    if (threadIdx.x == 0) trace_end(rec);
}

// Argument rules of ra_alltoall_emul(_ex); also called by the overlap driver BEFORE it enqueues anything.
ra_status alltoall_validate(const void* send, const void* recv, int P, size_t chunk_bytes, int sm_budget, int smem_bytes_per_cta,
                            int ctas_per_sm, int variant) {
    if (send == nullptr || recv == nullptr || P < 1 || P > 256) return RA_ERR_INVALID_ARG;
    if (sm_budget < 0 || smem_bytes_per_cta < 0 || ctas_per_sm < 0 || (variant < 0 || variant > 2))
        return RA_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(send) & 15u) || (reinterpret_cast<uintptr_t>(recv) & 15u)) return RA_ERR_INVALID_ARG;
    if (chunk_bytes % 16 != 0) return RA_ERR_INVALID_ARG;
    const size_t total = (size_t)P * P * chunk_bytes;
    const uintptr_t a = reinterpret_cast<uintptr_t>(send), b = reinterpret_cast<uintptr_t>(recv);
    if (a == b || (total > 0 && a < b + total && b < a + total)) return RA_ERR_INVALID_ARG;
    if (variant == 0 && chunk_bytes > 0) {    // ring slots of at least 1 KiB
        const int smem = smem_bytes_per_cta ? smem_bytes_per_cta : kA2aDefaultSmem;
        if ((((uint32_t)smem / kA2aSlots) & ~127u) < 1024) return RA_ERR_INVALID_ARG;
    }
    return RA_OK;
}

static ra_status launch_kernels(A2aParams p, uint64_t n_chunks, const DeviceInfo& di, int sm_budget, int smem_bytes_per_cta,
                                int ctas_per_sm, int variant, cudaStream_t stream);

ra_status alltoall_launch(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget,
                          int smem_bytes_per_cta, int ctas_per_sm, int variant, cudaStream_t stream) {
    RA_TRY(alltoall_validate(send, recv, P, chunk_bytes, sm_budget, smem_bytes_per_cta, ctas_per_sm, variant));
    if (chunk_bytes == 0) return RA_OK;

    DeviceInfo di;
    RA_TRY(device_info(&di));
    RA_TRY(require_sm100(di));
    RA_TRY(l2_persist_first_use(stream));
    if (variant == 2) {
        // SM-free variant (the mechanism of ConCCL): the device's copy engines move the chunks;
        // no CTA is ever resident, so the GEMM's occupancy knobs are irrelevant to it.  One plain
        // cudaMemcpyAsync per chunk (i,j) -> (j,i), P*P copies enqueued on `stream`.
        const char* s8 = static_cast<const char*>(send);
        char* r8 = static_cast<char*>(recv);
        for (int i = 0; i < P; ++i) {
            for (int j = 0; j < P; ++j)
                RA_CUDA(cudaMemcpyAsync(r8 + ((size_t)j * P + i) * chunk_bytes, s8 + ((size_t)i * P + j) * chunk_bytes,
                                        chunk_bytes, cudaMemcpyDeviceToDevice, stream));
        }
        return RA_OK;
    }
    A2aParams p{};
    p.send = static_cast<const uint8_t*>(send);
    p.recv = static_cast<uint8_t*>(recv);
    p.peer_rank = -1;
    p.P = (uint32_t)P;
    p.chunk_bytes = chunk_bytes;
    return launch_kernels(p, (uint64_t)P * P, di, sm_budget, smem_bytes_per_cta, ctas_per_sm, variant, stream);
}

// N4 (ra_peer.cu): rank `rank` pushes its P chunks into slot `rank` of the P receive buffers (its own included).
ra_status alltoall_peer_launch(const void* send, void* const* recv, int P, int rank, size_t chunk_bytes, int sm_budget,
                               int smem_bytes_per_cta, int ctas_per_sm, int variant, cudaStream_t stream) {
    if (send == nullptr || recv == nullptr || P < 1 || P > RA_MAX_RANKS || rank < 0 || rank >= P) return RA_ERR_INVALID_ARG;
    if (sm_budget < 0 || smem_bytes_per_cta < 0 || ctas_per_sm < 0 || variant < 0 || variant > 2) return RA_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(send) & 15u) || chunk_bytes % 16 != 0) return RA_ERR_INVALID_ARG;
    const uintptr_t s0 = reinterpret_cast<uintptr_t>(send), s1 = s0 + (size_t)P * chunk_bytes;
    for (int j = 0; j < P; ++j) {
        if (recv[j] == nullptr || (reinterpret_cast<uintptr_t>(recv[j]) & 15u)) return RA_ERR_INVALID_ARG;
        const uintptr_t r0 = reinterpret_cast<uintptr_t>(recv[j]), r1 = r0 + (size_t)P * chunk_bytes;
        if (chunk_bytes > 0 && s0 < r1 && r0 < s1) return RA_ERR_INVALID_ARG;            // send must not alias a receive buffer
        for (int i = 0; i < j; ++i) {                                                     // nor two ranks share one
            const uintptr_t q0 = reinterpret_cast<uintptr_t>(recv[i]), q1 = q0 + (size_t)P * chunk_bytes;
            if (chunk_bytes > 0 && q0 < r1 && r0 < q1) return RA_ERR_INVALID_ARG;
        }
    }
    if (variant == 0 && chunk_bytes > 0) {
        const int smem = smem_bytes_per_cta ? smem_bytes_per_cta : kA2aDefaultSmem;
        if ((((uint32_t)smem / kA2aSlots) & ~127u) < 1024) return RA_ERR_INVALID_ARG;
    }
    if (chunk_bytes == 0) return RA_OK;
    DeviceInfo di;
    RA_TRY(device_info(&di));
    RA_TRY(require_sm100(di));
    RA_TRY(l2_persist_first_use(stream));
    if (variant == 2) {                       // copy engines: one peer-to-peer cudaMemcpyAsync per destination
        for (int j = 0; j < P; ++j)
            RA_CUDA(cudaMemcpyAsync(static_cast<char*>(recv[j]) + (size_t)rank * chunk_bytes,
                                    static_cast<const char*>(send) + (size_t)j * chunk_bytes, chunk_bytes, cudaMemcpyDefault, stream));
        return RA_OK;
    }
    A2aParams p{};
    p.send = static_cast<const uint8_t*>(send);
    p.recv = nullptr;
    for (int j = 0; j < P; ++j) p.peer_recv[j] = static_cast<uint8_t*>(recv[j]);
    p.peer_rank = rank;
    p.P = (uint32_t)P;
    p.chunk_bytes = chunk_bytes;
    return launch_kernels(p, (uint64_t)P, di, sm_budget, smem_bytes_per_cta, ctas_per_sm, variant, stream);
}

static ra_status launch_kernels(A2aParams p, uint64_t n_chunks, const DeviceInfo& di, int sm_budget, int smem_bytes_per_cta,
                                int ctas_per_sm, int variant, cudaStream_t stream) {
    const size_t chunk_bytes = p.chunk_bytes;
    const int sms = (sm_budget == 0 || sm_budget > di.sm_count) ? di.sm_count : sm_budget;

    if (variant == 0) {
        int smem = smem_bytes_per_cta ? smem_bytes_per_cta : kA2aDefaultSmem;
        const int max_dyn = di.smem_per_block_optin - 256;
        if (smem > max_dyn) smem = max_dyn;
        uint32_t slice = ((uint32_t)smem / kA2aSlots) & ~127u;  // keep slots 128-B aligned
        if (slice < 1024) return RA_ERR_INVALID_ARG;
        if (slice > chunk_bytes) slice = (uint32_t)((chunk_bytes + 127) & ~(size_t)127);
        p.slice_bytes = slice;
        p.slices_per_chunk = (uint32_t)((chunk_bytes + slice - 1) / slice);
        p.n_units = n_chunks * p.slices_per_chunk;
        const int dyn = (int)(slice * kA2aSlots);
        int cps = ctas_per_sm ? ctas_per_sm : kA2aDefaultCtasPerSm;
        uint64_t grid = (uint64_t)sms * cps;
        if (grid > p.n_units) grid = p.n_units;
        if (dyn > 48 * 1024)
            RA_CUDA(cudaFuncSetAttribute(alltoall_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn));
            // same split as the GEMM asks for, so that either kernel can join the other on an SM (see prepare_kernel in ra_gemm.cu)
            RA_CUDA(cudaFuncSetAttribute(alltoall_tma_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        alltoall_tma_kernel<<<(unsigned)grid, kA2aThreads, dyn, stream>>>(p, g_trace);
    } else {
        p.slice_bytes = 64 * 1024;
        p.slices_per_chunk = (uint32_t)((chunk_bytes + p.slice_bytes - 1) / p.slice_bytes);
        p.n_units = n_chunks * p.slices_per_chunk;
        int cps = ctas_per_sm ? ctas_per_sm : kCopyCtasPerSm;
        uint64_t grid = (uint64_t)sms * cps;
        if (grid > p.n_units) grid = p.n_units;
        alltoall_ldg_kernel<<<(unsigned)grid, kCopyThreads, 0, stream>>>(p, g_trace);
    }
    RA_CUDA(cudaGetLastError());
    return RA_OK;
}

}  // namespace ra

extern "C" {
ra_status ra_alltoall_emul(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget, void* stream) {
    return ra::alltoall_launch(send, recv, P, chunk_bytes, sm_budget, 0, 0, 0, static_cast<cudaStream_t>(stream));
}
ra_status ra_alltoall_emul_ex(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget,
                              int smem_bytes_per_cta, int ctas_per_sm, int variant, void* stream) {
    return ra::alltoall_launch(send, recv, P, chunk_bytes, sm_budget, smem_bytes_per_cta, ctas_per_sm, variant,
                               static_cast<cudaStream_t>(stream));
}
}
