// ra_api.cu -- status strings, device facts, trace registration (host side of libra.so).
#include <mutex>

#include "ra_common.cuh"

namespace ra {

thread_local int g_last_cuda_error = 0;
Trace g_trace = {nullptr, 0};

static std::mutex g_di_mutex;
static DeviceInfo g_di_cache[64];
static bool g_di_valid[64] = {};

ra_status device_info(DeviceInfo* out) {
    int dev = -1;
    RA_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_di_mutex);
    if (dev >= 0 && dev < 64 && g_di_valid[dev]) {
        *out = g_di_cache[dev];
        return RA_OK;
    }
    DeviceInfo di;
    di.device = dev;
    RA_CUDA(cudaDeviceGetAttribute(&di.cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    RA_CUDA(cudaDeviceGetAttribute(&di.cc_minor, cudaDevAttrComputeCapabilityMinor, dev));
    RA_CUDA(cudaDeviceGetAttribute(&di.sm_count, cudaDevAttrMultiProcessorCount, dev));
    RA_CUDA(cudaDeviceGetAttribute(&di.smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    RA_CUDA(cudaDeviceGetAttribute(&di.smem_per_block_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    RA_CUDA(cudaDeviceGetAttribute(&di.smem_reserved_per_block, cudaDevAttrReservedSharedMemoryPerBlock, dev));
    RA_CUDA(cudaDeviceGetStreamPriorityRange(&di.prio_least, &di.prio_greatest));
    if (dev >= 0 && dev < 64) {
        g_di_cache[dev] = di;
        g_di_valid[dev] = true;
    }
    *out = di;
    return RA_OK;
}

ra_status require_sm100(const DeviceInfo& di) { return di.cc_major == 10 ? RA_OK : RA_ERR_ARCH; }

// ---- persisting-L2 carve-out (cudaLimitPersistingL2CacheSize) -------------------------------------------------------
// evict_last TMA loads only stick when the device has a persisting carve-out (measured: without it the policy changes
// nothing), and the carve-out is taken away from every other kernel's L2 (measured: the streaming collectives lose
// 10 % at 24 MiB, 35 % at 32-56 MiB, 2.3x at 64+ MiB; the driver grants sixteenths of the L2, rounded up).  It is therefore a per-setting resource like the shared-memory
// reserve: the library tracks what it last set per device and only calls the driver on a change.
static std::mutex g_l2_mutex;
static long long g_l2_state[64];     // what was asked for (after clamping to the device maximum)
static long long g_l2_granted[64];   // what the driver made of it (it rounds up to sixteenths of the L2: 7.9 MiB steps on B200)
static bool g_l2_known[64] = {};
static long long g_l2_found[64];     // what the context had when the library first looked (given back by l2_persist_restore)

ra_status l2_persist_ensure(long long bytes, long long* granted) {
    if (bytes < 0) return RA_ERR_INVALID_ARG;
    int dev = -1;
    RA_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return RA_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_l2_mutex);
    if (!g_l2_known[dev]) {
        // A fresh context does not always start at 0: boxes of this pool were seen to come up with 3/16 of the L2
        // (24870912 bytes) set aside, which costs the streaming collectives ~4 % (6.23 -> 5.96 TB/s).  Whatever is found
        // counts as foreign state and is replaced by what the caller asks for -- 0 unless a setting wants a carve-out.
        size_t cur = 0;
        RA_CUDA(cudaDeviceGetLimit(&cur, cudaLimitPersistingL2CacheSize));
        g_l2_granted[dev] = (long long)cur;
        g_l2_found[dev] = (long long)cur;
        g_l2_state[dev] = cur == 0 ? 0 : -1;
        g_l2_known[dev] = true;
    }
    int max_bytes = 0;
    RA_CUDA(cudaDeviceGetAttribute(&max_bytes, cudaDevAttrMaxPersistingL2CacheSize, dev));
    const long long want = bytes < (long long)max_bytes ? bytes : (long long)max_bytes;
    if (want != g_l2_state[dev]) {
        // Shrinking: persisting lines are given up FIRST -- the driver was seen to leave the limit at what is still in use
        // (3/16 of the L2 after a 24 MiB panel) when asked to go to 0 with lines resident.
        const auto apply = [&](size_t* got) -> cudaError_t {
            cudaError_t e = cudaSuccess;
            if (want < g_l2_state[dev] || g_l2_state[dev] < 0) e = cudaCtxResetPersistingL2Cache();
            if (e == cudaSuccess) e = cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)want);
            if (e == cudaSuccess) e = cudaDeviceGetLimit(got, cudaLimitPersistingL2CacheSize);
            if (e == cudaSuccess && want == 0 && *got != 0) {  // in-flight work re-marked lines in between: drain and retry once
                e = cudaDeviceSynchronize();
                if (e == cudaSuccess) e = cudaCtxResetPersistingL2Cache();
                if (e == cudaSuccess) e = cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, 0);
                if (e == cudaSuccess) e = cudaDeviceGetLimit(got, cudaLimitPersistingL2CacheSize);
            }
            return e;
        };
        size_t got = (size_t)g_l2_granted[dev];
        const cudaError_t e = apply(&got);
        if (e != cudaSuccess) {
            if (want > 0) RA_CUDA(e);          // the caller asked for a carve-out and cannot have it: that is an error
            // want == 0 is housekeeping with the feature OFF (every collective and every plain GEMM passes through here): where
            // the driver will not let this process change the limit (a set-aside fixed from outside, MPS) nothing the caller
            // asked for has failed.  Best effort: forget the error, remember that it was tried, carry on.
            (void)cudaGetLastError();
            got = (size_t)g_l2_granted[dev];
        }
        g_l2_state[dev] = want;
        g_l2_granted[dev] = (long long)got;
    }
    if (granted) *granted = g_l2_granted[dev];
    return RA_OK;
}

// ra_gemm's form: the same, except that nothing happens while `stream` is being captured (cudaDeviceSetLimit cannot be
// captured; the GEMM then runs with whatever carve-out is in place -- same results, the evict_last hints just do not stick)
// and that the common case -- the state already is what is asked for -- costs one mutex and no driver call.
ra_status l2_persist_ensure_on(long long bytes, cudaStream_t stream) {
    if (bytes < 0) return RA_ERR_INVALID_ARG;
    int dev = -1;
    RA_CUDA(cudaGetDevice(&dev));
    if (dev >= 0 && dev < 64) {
        std::lock_guard<std::mutex> lk(g_l2_mutex);
        if (g_l2_known[dev] && g_l2_state[dev] == bytes) return RA_OK;
    }
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();
        return RA_OK;
    }
    return l2_persist_ensure(bytes);
}

// ra_shutdown: the current device's carve-out goes back to what the context had before the library first touched it (an
// application that set one for its own access-policy windows gets it back), and the library forgets the device's state.
void l2_persist_restore() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) {
        (void)cudaGetLastError();
        return;
    }
    std::lock_guard<std::mutex> lk(g_l2_mutex);
    if (!g_l2_known[dev]) return;
    if (g_l2_granted[dev] != g_l2_found[dev]) {
        bool ok = cudaCtxResetPersistingL2Cache() == cudaSuccess;
        ok = ok && cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, (size_t)g_l2_found[dev]) == cudaSuccess;
        if (!ok) (void)cudaGetLastError();
    }
    g_l2_known[dev] = false;
}

// First use of a collective on a device: take back a carve-out the context came up with (see above).  A no-op once the
// library knows the device's state, and skipped while `stream` is being captured (cudaDeviceSetLimit is not capturable).
ra_status l2_persist_first_use(cudaStream_t stream) {
    int dev = -1;
    RA_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return RA_OK;
    {
        std::lock_guard<std::mutex> lk(g_l2_mutex);
        if (g_l2_known[dev]) return RA_OK;
    }
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) {
        (void)cudaGetLastError();
        return RA_OK;
    }
    return l2_persist_ensure(0);
}

}  // namespace ra

extern "C" {

const char* ra_status_str(ra_status s) {
    switch (s) {
        case RA_OK: return "RA_OK";
        case RA_ERR_INVALID_ARG: return "RA_ERR_INVALID_ARG";
        case RA_ERR_UNSUPPORTED: return "RA_ERR_UNSUPPORTED";
        case RA_ERR_INFEASIBLE_KNOB: return "RA_ERR_INFEASIBLE_KNOB";
        case RA_ERR_CUDA: return "RA_ERR_CUDA";
        case RA_ERR_ARCH: return "RA_ERR_ARCH";
        case RA_ERR_SCRATCH_LIMIT: return "RA_ERR_SCRATCH_LIMIT";
    }
    return "RA_ERR_UNKNOWN";
}

int ra_last_cuda_error(void) { return ra::g_last_cuda_error; }

ra_status ra_device_info(int* sm_count, int* smem_per_sm, int* smem_per_block_optin, int* smem_reserved_per_block,
                         int* prio_least, int* prio_greatest) {
    ra::DeviceInfo di;
    RA_TRY(ra::device_info(&di));
    if (sm_count) *sm_count = di.sm_count;
    if (smem_per_sm) *smem_per_sm = di.smem_per_sm;
    if (smem_per_block_optin) *smem_per_block_optin = di.smem_per_block_optin;
    if (smem_reserved_per_block) *smem_reserved_per_block = di.smem_reserved_per_block;
    if (prio_least) *prio_least = di.prio_least;
    if (prio_greatest) *prio_greatest = di.prio_greatest;
    return RA_OK;
}

ra_status ra_l2_persist(int64_t bytes, int64_t* granted) {
    long long g = 0;
    RA_TRY(ra::l2_persist_ensure((long long)bytes, &g));
    if (granted) *granted = (int64_t)g;
    return RA_OK;
}

ra_status ra_set_trace(uint64_t* buf, size_t capacity) {
    if (buf != nullptr && capacity == 0) return RA_ERR_INVALID_ARG;
    ra::g_trace.buf = buf;
    ra::g_trace.cap = buf ? (uint64_t)capacity : 0;
    return RA_OK;
}

}  // extern "C"
