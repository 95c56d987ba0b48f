// ra_common.cuh -- shared host/device helpers of libra.so (product code; never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "ra.h"

namespace ra {

// ---- host: error plumbing -------------------------------------------------------------------
extern thread_local int g_last_cuda_error;

inline ra_status cuda_fail(cudaError_t e) {
    g_last_cuda_error = (int)e;
    return RA_ERR_CUDA;
}
#define RA_CUDA(expr)                                      \
    do {                                                   \
        cudaError_t _e = (expr);                           \
        if (_e != cudaSuccess) return ::ra::cuda_fail(_e); \
    } while (0)
#define RA_TRY(expr)                     \
    do {                                 \
        ra_status _s = (expr);           \
        if (_s != RA_OK) return _s;      \
    } while (0)

struct DeviceInfo {
    int device = -1;
    int cc_major = 0, cc_minor = 0;
    int sm_count = 0;
    int smem_per_sm = 0;
    int smem_per_block_optin = 0;
    int smem_reserved_per_block = 0;
    int prio_least = 0, prio_greatest = 0;
};
// Queries (and caches per device) the attributes above.  RA_ERR_CUDA without a device.
ra_status device_info(DeviceInfo* out);
// RA_ERR_ARCH unless the current device is sm_100-family.
ra_status require_sm100(const DeviceInfo& di);
// Sets the current device's persisting-L2 carve-out to min(bytes, device maximum) unless that is what this library
// last set (then no driver call is made); bytes = 0 also resets the persisting lines.  Must not be called while a
// stream of the device is being captured unless it is a no-op.
ra_status l2_persist_ensure(long long bytes, long long* granted = nullptr);
// The same for a launch on `stream`: skipped (RA_OK) while that stream is being captured; no driver call when nothing changes.
ra_status l2_persist_ensure_on(long long bytes, cudaStream_t stream);
// Gives the current device's carve-out back as the library found it and forgets the device (ra_shutdown).
void l2_persist_restore();
// Collectives call this before their first launch on a device: takes back a carve-out the context came up with.
ra_status l2_persist_first_use(cudaStream_t stream);

// Planner constants used when no device is present (plan queries on a CPU-only box): B200 values.
constexpr int kDefaultSmCount = 148;
constexpr int kDefaultSmemPerSm = 233472;       // 228 KiB
constexpr int kDefaultSmemPerBlockOptin = 232448; // 227 KiB
constexpr int kDefaultSmemReservedPerBlock = 1024;

// ---- trace --------------------------------------------------------------------------------
struct Trace {
    uint64_t* buf;   // buf[0] = counter, then 4 words per record
    uint64_t cap;
};
extern Trace g_trace;

enum : uint32_t { KID_GEMM = 1, KID_ALLREDUCE = 2, KID_ALLTOALL = 3 };

#ifdef __CUDACC__
// ---- device: small PTX wrappers ---------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t globaltimer() {
    uint64_t t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ uint32_t smid() {
    uint32_t s;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(s));
    return s;
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
    return pred != 0;
}

// trace: one thread per CTA calls begin() at entry and end() at exit.
__device__ __forceinline__ uint64_t* trace_begin(Trace tr, uint32_t kid) {
    if (tr.buf == nullptr) return nullptr;
    unsigned long long idx = atomicAdd((unsigned long long*)tr.buf, 1ull);
    if (idx >= tr.cap) return nullptr;
    uint64_t* rec = tr.buf + 1 + 4 * idx;
    rec[0] = ((uint64_t)kid << 32) | smid();
    rec[1] = blockIdx.x;
    rec[2] = globaltimer();
    return rec;
}
__device__ __forceinline__ void trace_end(uint64_t* rec) {
    if (rec) rec[3] = globaltimer();
}

// mbarrier
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// try_wait suspends the thread until the phase completes or a time limit passes.  With the suspend-time hint (ns) the
// limit is long, so a warp that waits for most of a tile (the epilogue warps: ~100 us per accumulator) sleeps instead of
// re-issuing the probe every few hundred cycles -- the un-hinted loop executed 5.7x the instructions of the whole rest of
// the kernel (ncu inst_executed 118 M vs cuBLAS's 21 M on 8192^3), and on a power-capped chip those are joules.
constexpr uint32_t kMbarSuspendNs = 1000000u;   // 1 ms; completion of the phase wakes the thread at once
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred P;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity), "r"(kMbarSuspendNs)
        : "memory");
    return ok != 0;
}
// Bounded wait: a protocol bug (wrong phase, lost arrive) must surface as a trapped launch
// (cudaErrorLaunchFailure -> RA_ERR_CUDA), never as a hung GPU.  A suspended waiter is woken by every mbarrier event of
// its CTA (ncu: the epilogue warps re-probe ~7 k times per kernel), so the loop body is kept to the probe itself and the
// clock is read once per 256 failed probes.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    if (mbar_try_wait(bar, parity)) return;
    uint64_t t0 = 0;
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 255u) == 0) {
            const uint64_t now = globaltimer();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 5000000000ull) __trap();   // 5 s
        }
    }
}

// L2 eviction policies for TMA / bulk copies
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_normal() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
#endif  // __CUDACC__

}  // namespace ra
