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

ra_status ra_set_trace(uint64_t* buf, size_t capacity) {
    if (buf != nullptr && capacity == 0) return RA_ERR_INVALID_ARG;
    ra::g_trace.buf = buf;
    ra::g_trace.cap = buf ? (uint64_t)capacity : 0;
    return RA_OK;
}

}  // extern "C"
