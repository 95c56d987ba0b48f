// ra_peer.cu -- N4: the collective stand-ins as REAL exchanges over peer memory ("aggregated across all
// GPUs using allreduce ... alltoall to route tokens between devices", 4 / 8 GPUs per node).
//
// One process per GPU.  Every rank owns one buffer; the others reach it through a CUDA IPC mapping (NVLink / NVSwitch
// peer memory), so each rank holds P device pointers in RANK ORDER, its own among them.  The kernels are K2 and K3
// unchanged -- they only ever saw P pointers:
//
//   allreduce   rank r reduces ITS slice [b_r, e_r) of all P buffers in the fixed order 0, 1, ..., P-1 (one RNE binary32
//               add per rank, as the emulation and the oracle do) and writes the sum back to that slice of all P buffers:
//               reduce-scatter and all-gather fused in one pass over peer memory, (P-1)/P of the slice's reads and
//               writes crossing NVLink.  The slices partition [0, count), so after every rank has run, every buffer
//               holds the oracle's result bit for bit -- the per-element association never depends on who reduces it.
//   alltoall    rank r pushes chunk j of its send buffer into slot r of rank j's receive buffer (P bulk-copy streams,
//               the diagonal one local): recv_j[r] = send_r[j], the emulation's (i,j) -> (j,i) with row i living on rank i.
//
// Ordering between ranks is the caller's (a barrier of the process group before -- inputs ready -- and after -- every slice
// / chunk written); the kernels never wait on another rank.  With one GPU at hand this path is exercised by P sequential
// "ranks" on one device and by two processes sharing one device through real IPC handles; it is unmeasured on NVLink.
#include <cuda.h>

#include <cstring>
#include <mutex>
#include <unordered_map>

#include "ra_common.cuh"

namespace ra {

ra_status allreduce_launch(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, int smem_bytes_per_cta,
                           int variant, cudaStream_t stream);
ra_status alltoall_peer_launch(const void* send, void* const* recv, int P, int rank, size_t chunk_bytes, int sm_budget,
                               int smem_bytes_per_cta, int ctas_per_sm, int variant, cudaStream_t stream);

// slice r of P over `count` floats: boundaries rounded down to 4 floats (the kernels' 16-byte vectors), the last ends at count
static void slice_of(size_t count, int P, int rank, size_t* begin, size_t* end) {
    auto cut = [&](int r) -> size_t {
        if (r >= P) return count;
        return (size_t)(((unsigned __int128)count * (unsigned)r) / (unsigned)P) & ~(size_t)3;
    };
    *begin = cut(rank);
    *end = cut(rank + 1);
}

typedef CUresult (*GetAddressRangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);
static ra_status address_range(const void* p, uintptr_t* base, size_t* size) {
    static std::once_flag once;
    static GetAddressRangeFn fn = nullptr;
    static cudaError_t err = cudaSuccess;
    std::call_once(once, [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        err = cudaGetDriverEntryPoint("cuMemGetAddressRange", &f, cudaEnableDefault, &q);
        if (err == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = reinterpret_cast<GetAddressRangeFn>(f);
    });
    if (fn == nullptr) return cuda_fail(err != cudaSuccess ? err : cudaErrorSymbolNotFound);
    CUdeviceptr b = 0;
    size_t s = 0;
    if (fn(&b, &s, (CUdeviceptr)(uintptr_t)p) != CUDA_SUCCESS) return cuda_fail(cudaErrorInvalidValue);
    *base = (uintptr_t)b;
    *size = s;
    return RA_OK;
}

static std::mutex g_ipc_mu;
// pointer handed out -> {mapping base (what cudaIpcCloseMemHandle wants), how many ra_ipc_open calls returned it}.  Opening one
// handle twice gives the same pointer and takes a second reference inside the driver: every open is paired with one close.
struct IpcOpen { uintptr_t base; int count; };
static std::unordered_map<uintptr_t, IpcOpen> g_ipc_open;

// ra_shutdown: unmap whatever the caller left open
void peer_close_all() {
    std::lock_guard<std::mutex> lk(g_ipc_mu);
    for (auto& kv : g_ipc_open)
        for (int i = 0; i < kv.second.count; ++i) (void)cudaIpcCloseMemHandle(reinterpret_cast<void*>(kv.second.base));
    g_ipc_open.clear();
    (void)cudaGetLastError();
}

}  // namespace ra

extern "C" {

ra_status ra_peer_slice(size_t count, int P, int rank, size_t* begin, size_t* end) {
    if (P < 1 || P > RA_MAX_RANKS || rank < 0 || rank >= P || begin == nullptr || end == nullptr) return RA_ERR_INVALID_ARG;
    ra::slice_of(count, P, rank, begin, end);
    return RA_OK;
}

ra_status ra_ipc_export(const void* dev_ptr, ra_ipc_handle* out) {
    if (dev_ptr == nullptr || out == nullptr) return RA_ERR_INVALID_ARG;
    uintptr_t base = 0;
    size_t size = 0;
    RA_TRY(ra::address_range(dev_ptr, &base, &size));
    cudaIpcMemHandle_t h;
    RA_CUDA(cudaIpcGetMemHandle(&h, reinterpret_cast<void*>(base)));
    static_assert(sizeof(h) == sizeof(out->opaque), "ra_ipc_handle mirrors cudaIpcMemHandle_t");
    memcpy(out->opaque, &h, sizeof(h));
    out->offset = (uint64_t)(reinterpret_cast<uintptr_t>(dev_ptr) - base);
    out->bytes = (uint64_t)(size - (size_t)out->offset);
    return RA_OK;
}

ra_status ra_ipc_open(const ra_ipc_handle* h, void** dev_ptr) {
    if (h == nullptr || dev_ptr == nullptr) return RA_ERR_INVALID_ARG;
    cudaIpcMemHandle_t ch;
    memcpy(&ch, h->opaque, sizeof(ch));
    void* base = nullptr;
    RA_CUDA(cudaIpcOpenMemHandle(&base, ch, cudaIpcMemLazyEnablePeerAccess));
    void* p = static_cast<uint8_t*>(base) + h->offset;
    {
        std::lock_guard<std::mutex> lk(ra::g_ipc_mu);
        ra::IpcOpen& e = ra::g_ipc_open[reinterpret_cast<uintptr_t>(p)];      // value-initialised {0, 0} when new
        e.base = reinterpret_cast<uintptr_t>(base);
        e.count += 1;
    }
    *dev_ptr = p;
    return RA_OK;
}

ra_status ra_ipc_close(void* dev_ptr) {
    uintptr_t base = 0;
    {
        std::lock_guard<std::mutex> lk(ra::g_ipc_mu);
        auto it = ra::g_ipc_open.find(reinterpret_cast<uintptr_t>(dev_ptr));
        if (it == ra::g_ipc_open.end()) return RA_ERR_INVALID_ARG;
        base = it->second.base;
        if (--it->second.count <= 0) ra::g_ipc_open.erase(it);
    }
    RA_CUDA(cudaIpcCloseMemHandle(reinterpret_cast<void*>(base)));
    return RA_OK;
}

ra_status ra_allreduce_peer(float* const* bufs, int P, int rank, size_t count, int sm_budget, int variant, void* stream) {
    if (bufs == nullptr || P < 1 || P > RA_MAX_RANKS || rank < 0 || rank >= P) return RA_ERR_INVALID_ARG;
    size_t b = 0, e = 0;
    ra::slice_of(count, P, rank, &b, &e);
    float* sl[RA_MAX_RANKS];
    for (int r = 0; r < P; ++r) {
        if (bufs[r] == nullptr) return RA_ERR_INVALID_ARG;
        sl[r] = bufs[r] + b;
    }
    return ra::allreduce_launch(sl, P, e - b, sm_budget, 0, 0, variant, static_cast<cudaStream_t>(stream));
}

ra_status ra_alltoall_peer(const void* send, void* const* recv, int P, int rank, size_t chunk_bytes, int sm_budget, int variant,
                           void* stream) {
    return ra::alltoall_peer_launch(send, recv, P, rank, chunk_bytes, sm_budget, 0, 0, variant, static_cast<cudaStream_t>(stream));
}

}  // extern "C"
