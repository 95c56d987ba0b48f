// ra_gemm.cu -- K1: bf16 GEMM on the tcgen05 tensor cores (S1, S2, S3).
//
//   C[M,N] = alpha * op(A) * op(B) + beta * C          (section 2.1)
//
// Kernel coordinates.  The kernel multiplies two K-contiguous ("K-major") operands
//     X : RX x K  (rows -> TMEM lanes, 128 per CTA tile, the UMMA "M" side)
//     Y : RY x K  (rows -> TMEM columns, BN per CTA tile, the UMMA "N" side)
// into acc[x][y] = sum_k X[x][k]*Y[y][k].  transA=0,transB=1 maps A->X, B->Y (C[x][y]); the
// skinny-M path swaps them (B->X, A->Y, C[y][x]) so that the 128-row side is the long weight
// dimension and tiny M costs BN = 64 columns instead of a padded 128-row tile.
//
// Per CTA (192 threads):
//   warp 0   TMA producer      one elected lane: cp.async.bulk.tensor.2d into a ring of `stages`
//                              128B-swizzled shared-memory stages, mbarrier complete_tx
//   warp 1   MMA issuer        allocates TMEM; one elected lane issues tcgen05.mma (128 x BN x 16,
//                              kind::f16, bf16 in / fp32 accumulate in TMEM), tcgen05.commit frees
//                              the smem stage / publishes the accumulator
//   warps 2-5 epilogue         tcgen05.ld (32 lanes x 32 columns per instruction) -> alpha/beta ->
//                              cvt.rn.bf16x2.f32 -> swizzled shared-memory staging -> TMA stores (direct
//                              stores on the swapped path, for fp32 C, stream-K fix-ups and ragged-N boxes).
//                              Two TMEM accumulators (2 x BN columns) so the epilogue of tile i overlaps
//                              the main loop of tile i+1.
//
// Tile forms (template <BN, CG, XH>, picked by make_plan):
//   <BN,1,1>   single-CTA tiles 128 x BN, BN in {64,128,256}: small / skinny problems, stream-K, split-K
//   <256,2,1>  CTA pairs (2-CTA cluster, tcgen05 cta_group::2): 256 x 256 per pair, half the Y traffic per CTA
//   <256,2,2>  big tiles: two 128-row X blocks per CTA share one Y stage, 512 x 256 per pair, all 512 TMEM
//              columns hold ONE tile; the two blocks are issued skewed so the drain of one hides behind the
//              MMAs of the other at both ends of a tile (large problems; the tile cuBLAS uses too)
//
// Scheduling (S3: occupancy shaping).  grid = sm_budget persistent CTAs, one
// per SM; pipeline depth (and, when squeezed, the tile) follows from smem_reserve_bytes; tile_k = 32 halves the
// stages; l2_persist_bytes keeps one raster group's X panel in a persisting L2 carve-out.  Work
// decompositions (no floating-point atomics anywhere; integer atomics only hand out work):
//   data-parallel   grouped rasterisation for L2 reuse.  Multi-wave persistent plans hand tiles out DYNAMICALLY (next unclaimed
//                   tile of the raster, one integer atomic per tile: see g_dyn) so that workers which finish together run
//                   neighbouring tiles in step and their loads coalesce in L2; otherwise worker c owns tiles c, c+G, c+2G, ...
//                   Either way one worker accumulates a C element in ascending k: the assignment never changes a result.
//   cluster split-K a 2-CTA cluster takes one tile's k-blocks half each; CTA 1 hands its accumulator to CTA 0
//                   through distributed shared memory (no workspace; low + high half, fixed order)
//   stream-K        the n_tiles*KB k-block units are cut into G equal contiguous ranges; a tile
//                   whose units span several CTAs is finished by the LAST of them to arrive
//                   (threadfence + one integer atomic per part): it sums the fp32 partials of all
//                   parts from the workspace in ascending-k order, so the result does not depend
//                   on arrival order and is bit-reproducible.
#include <cuda.h>
#include <cuda_bf16.h>

#include <cstring>
#include <mutex>
#include <vector>

#include "ra_common.cuh"

namespace ra {

constexpr int kBM = 128;        // tile rows on the X side (UMMA M)
constexpr int kBK = 64;         // 64 bf16 = 128 B = one swizzle-128B atom row
constexpr int kUmmaK = 16;
constexpr int kGemmThreads = 192;
constexpr int kEpiThreads = 128;
constexpr int kMaxStages = 8;
constexpr int kBarrierBytes = 256;
constexpr int kAlignSlack = 1024;
// epilogue staging for TMA stores: per epilogue warp two buffers of 32 rows x 64 bf16 (128-byte swizzled rows)
constexpr int kEpiBoxCols = 64;
constexpr int kEpiBufBytes = 32 * kEpiBoxCols * 2;          // 4 KiB
constexpr int kEpiStageBytes = 4 * 2 * kEpiBufBytes;        // 32 KiB

// bytes of one pipeline stage in ONE CTA: 128*xh rows of X + bn/cg rows of Y, 64 bf16 each
__host__ __device__ constexpr int stage_bytes(int bn, int cg, int xh) { return (kBM * xh + bn / cg) * kBK * 2; }

struct GemmParams {
    int RX, RY, K;
    int tiles_x, tiles_y, n_tiles, kb_per_tile;
    int swap;          // 0: C[x*ldc + y]   1: C[y*ldc + x]
    int stream_k;
    int stages;
    int bk;            // k extent of one pipeline stage: 64 (128-byte swizzle rows) or 32 (64-byte rows; K-major operands only)
    float alpha, beta;
    __nv_bfloat16* C;
    int ldc;
    float* partials;   // stream-K: [2*grid][BN][128] fp32
    int* counters;     // stream-K: [n_tiles]
    int hintX, hintY;  // L2 policy per operand: 0 normal, 1 evict_first, 2 evict_last
    int hintC;         // L2 policy of the TMA stores of C (written once, never re-read by this kernel)
    int group_x;       // rasterisation: X-tiles per group
    int dyn;           // 1: dynamic tile order (data-parallel multi-wave plans): a worker's next tile is the next unclaimed one
    unsigned long long* dyn_ring;   // [workers][kDynRing] tagged entries ((generation << 12 | step) << 32 | tile), written by the worker's scheduler thread
    unsigned int* dyn_ctr;          // [0] tiles claimed beyond the first `workers`, [1] CTAs that left the kernel, [2] generation
    int xmn, ymn;      // operand storage: 0 = K-contiguous rows (K-major), 1 = row index contiguous (MN-major)
    int epi_tma;       // 1: whole tiles leave through shared memory + TMA stores (non-swapped C only)
    int skew;          // XH == 2: k-blocks by which X block 0 leads block 1 at both ends of a tile (<= stages)
    int c_f32;         // 1: C is fp32 (ldc in floats): alpha*acc + beta*C without the bf16 rounding, direct stores only
    int ks;            // 2: cluster split-K -- the two CTAs of a cluster take one tile's k-blocks half each and CTA 1
                       //    hands its accumulator to CTA 0 through distributed shared memory (CG == 1, XH == 1 only)
};

// ---- residency counters (S3 by measurement) -----------------------------------------------------
// Every GEMM CTA counts itself in on its SM (%smid) at entry and out at exit; the running maximum of GEMM CTAs seen
// on one SM at the same time is what ra_gemm_residency() reports.  One atomic pair per CTA, issued by an epilogue
// lane that is idle at both moments.  Module-scope device memory: nothing is allocated.
__device__ int g_gemm_resident[1024];
__device__ int g_gemm_max_resident;

// ---- dynamic tile order -------------------------------------------------------------------------------------------
// Workers that finish a tile at the same moment claim CONSECUTIVE tiles (one integer atomic per tile) -- neighbours in the
// raster, which share an operand panel -- and so start them in step: their TMA loads of the shared rows reach the L2 request
// coalescer together and are served by one slice read.  A static assignment (worker w owns tiles w, w + W, ...) keeps handing
// adjacent tiles to workers that drifted apart waves ago: ncu on 8192^3 shows 1.07 GPC deliveries per L2-slice read with
// the static order (1.25 in a one-wave problem, where everybody starts together) against cuBLAS's 1.37.
// One launch slot per launch in flight (see dyn_slot_acquire): [kDynWorkers][kDynRing] ring entries + {claim counter, exit counter, generation}.
// The slot re-arms ITSELF: ring tags carry the slot's generation, and the last CTA to leave the kernel zeroes the two
// counters and bumps the generation, so the next launch finds a clean slot without a memset node in front of it.  (A
// memset node was tried first and cost the overlapped step 6 %: it delays K_g^(i+1) by a few microseconds, the waiting
// collective K_c^i takes the SMs first, and an SM that runs shared-memory-free CTAs has to drain before it can give a
// GEMM CTA its 225 KiB carve-out -- the two kernels serialised.)  The ring needs no acknowledgements: the scheduler thread (the TMA producer) is never more than `stages`
// (<= kMaxStages = 8) k-blocks -- hence at most 8 tiles, when a tile is a single k-block -- ahead of the MMA issuer, which is
// never more than two tiles (two accumulators) ahead of the epilogue, and it publishes one step ahead: 11 steps of history
// at most, so kDynRing = 16 cannot be overrun.
constexpr int kDynWorkers = 160;
constexpr int kDynRing = 16;
static_assert(kDynRing >= kMaxStages + 4 && (kDynRing & (kDynRing - 1)) == 0, "ring depth");
constexpr int kDynSlots = 32;
constexpr int kDynSlotWords = kDynWorkers * kDynRing + 8;     // u64 words per slot; u32 {claims, exits, generation} start at word kDynWorkers * kDynRing
constexpr int kDynMaxSteps = 4000;                            // steps per worker that fit the tag's 12-bit step field
__device__ unsigned long long g_dyn[kDynSlots * kDynSlotWords];

// ---- device helpers ---------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- cluster (CTA pair) helpers ------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of the same shared-memory offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
// arrive (+ expect_tx) on a barrier given by its shared::cluster address (may live in the peer CTA)
__device__ __forceinline__ void mbar_expect_tx_cluster(uint32_t bar_cluster, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cluster.b64 _, [%0], %1;" ::"r"(bar_cluster), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t bar_cluster) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}

// TMA tile load.  CG == 2: the .cta_group::2 form, whose mbarrier may live in the peer (leader) CTA.
template <int CG>
__device__ __forceinline__ void tma_load_2d(uint32_t dst_smem, const CUtensorMap* map, int c0, int c1, uint32_t bar,
                                            uint64_t policy) {
    if (policy == 0) {
        // no cache hint: the default L2 behaviour (a createpolicy evict_normal hint is NOT the same thing -- ncu
        // shows such lines as "evict_normal_demote" and 2.4x the cross-die L2 fabric traffic)
        if constexpr (CG == 1) {
            asm volatile(
                "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
                " [%0], [%1, {%3, %4}], [%2];"
                ::"r"(dst_smem), "l"(map), "r"(bar), "r"(c0), "r"(c1)
                : "memory");
        } else {
            asm volatile(
                "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes"
                " [%0], [%1, {%3, %4}], [%2];"
                ::"r"(dst_smem), "l"(map), "r"(bar), "r"(c0), "r"(c1)
                : "memory");
        }
        return;
    }
    if constexpr (CG == 1) {
        asm volatile(
            "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
            " [%0], [%1, {%3, %4}], [%2], %5;"
            ::"r"(dst_smem), "l"(map), "r"(bar), "r"(c0), "r"(c1), "l"(policy)
            : "memory");
    } else {
        asm volatile(
            "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
            " [%0], [%1, {%3, %4}], [%2], %5;"
            ::"r"(dst_smem), "l"(map), "r"(bar), "r"(c0), "r"(c1), "l"(policy)
            : "memory");
    }
}

// K-major, 128-byte swizzle: rows of 128 B, 8-row groups 1024 B apart (SBO), LBO unused (=1),
// descriptor version 1 (sm_100), layout type 2 = SWIZZLE_128B.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// K-major, 64-byte swizzle (tile_k = 32): rows of 64 B, 8-row groups 512 B apart (SBO), layout type 4 = SWIZZLE_64B.
__device__ __forceinline__ uint64_t umma_desc_sw64(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)(512 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)4 << 61;
    return d;
}
// MN-major, 128-byte swizzle.  The stage holds one 8 KiB box per 64 rows (TMA box = 64 rows x 64 k, the 64 rows
// contiguous = one 128-byte line per k): canonical layout ((8,8,m),(8,k)) : ((1,8,LBO),(64,SBO)) elements, i.e.
// 8 k-lines of 128 B form a 1024-B swizzle atom; SBO = 1024 B between 8-k groups, LBO = 8192 B between 64-row boxes.
// One UMMA (K = 16) spans two k groups, so the k step advances the start address by 2048 B.
__device__ __forceinline__ uint64_t umma_desc_sw128_mn(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)(8192 >> 4) << 16;
    d |= (uint64_t)(1024 >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// kind::f16 instruction descriptor: D = fp32, A = B = bf16, M x N; bit 15 / 16 = A / B is MN-major.
__host__ __device__ constexpr uint32_t umma_idesc_bf16(int m, int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(m >> 4) << 24);
}
// D[tmem] (+)= X[smem] * Y[smem]^T.  CG == 2: one instruction drives the tensor cores of both SMs of the
// pair (M = 256: rows 0-127 from the leader's X stage, 128-255 from the peer's; Y split N/2 + N/2).
template <int CG>
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
    if constexpr (CG == 1) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
            "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
            ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
            : "memory");
    } else {
        asm volatile(
            "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
            "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
            ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
            : "memory");
    }
}
// mbarrier arrive when all MMAs issued so far have retired.  CG == 2: multicast to the same barrier
// offset in both CTAs of the pair.
template <int CG>
__device__ __forceinline__ void umma_commit(uint32_t bar, uint16_t pair_mask) {
    if constexpr (CG == 1) {
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
    } else {
        asm volatile(
            "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
            ::"r"(bar), "h"(pair_mask)
            : "memory");
    }
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void epi_bar_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kEpiThreads) : "memory"); }

// TMA store of one (64 cols x 32 rows) box, shared -> global, clipped at the tensor's bounds
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src_smem, int c0, int c1, uint64_t policy) {
    if (policy == 0) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
                     ::"l"(map), "r"(src_smem), "r"(c0), "r"(c1) : "memory");
    } else {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3}], [%1], %4;"
                     ::"l"(map), "r"(src_smem), "r"(c0), "r"(c1), "l"(policy) : "memory");
    }
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ---- cluster split-K: accumulator hand-over through distributed shared memory ---------------------------------
__device__ __forceinline__ void st_cluster_v4(uint32_t addr_cluster, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr_cluster), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void ld_shared_v4(uint32_t addr, uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) {
    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(addr) : "memory");
}
// bulk copy local shared memory -> another CTA's shared memory, completing `bytes` on that CTA's mbarrier
__device__ __forceinline__ void dsmem_bulk_copy(uint32_t dst_cluster, uint32_t src_cta, uint32_t bytes, uint32_t bar_cluster) {
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_cluster), "r"(src_cta), "r"(bytes), "r"(bar_cluster) : "memory");
}
// arrive on a barrier of another CTA of the cluster, releasing this thread's prior (distributed) shared-memory writes
__device__ __forceinline__ void mbar_arrive_release_cluster(uint32_t bar_cluster) {
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(bar_cluster) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait_acquire_cluster(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred P;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait_acquire_cluster(uint32_t bar, uint32_t parity) {
    uint64_t t0 = 0;
    uint32_t spins = 0;
    while (!mbar_try_wait_acquire_cluster(bar, parity)) {
        if ((++spins & 4095u) == 0) {
            const uint64_t now = globaltimer();
            if (t0 == 0) t0 = now;
            else if (now - t0 > 5000000000ull) __trap();   // 5 s: a protocol bug is a failed launch, not a hang
        }
    }
}

__device__ __forceinline__ uint64_t make_policy(int kind) {
    return kind == 1 ? policy_evict_first() : (kind == 2 ? policy_evict_last() : 0ull);   // 0 = no hint
}

// ---- static schedule: every role walks the same sequence of (tile, kb0, kb1) segments ----------
struct Seg {
    int tile, kb0, kb1;
    long long start_unit;   // stream-K: first unit of this segment
};
template <bool DYN>
struct Sched {
    const GemmParams& p;
    long long u0, u1, cur;  // stream-K unit range of this worker
    int it;
    int wid, nw;            // worker (CTA, CTA pair, or split-K cluster) index and count
    int krank;              // cluster split-K: which half of a tile's k-blocks this CTA takes (else 0)
    int role;               // dynamic order: 0 = this worker's scheduler thread, 1 = a single consumer thread, 2 = a consumer warp
    int pending;            // scheduler: the tile claimed for the next step
    unsigned gen;           // dynamic order: the slot's generation during this launch (constant until the last CTA leaves)
    __device__ Sched(const GemmParams& p_, int wid_, int nw_, int krank_ = 0, int role_ = 1)
        : p(p_), it(0), wid(wid_), nw(nw_), krank(krank_), role(role_), pending(-1), gen(0) {
        if constexpr (DYN) asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(gen) : "l"(p.dyn_ctr + 2) : "memory");
        if (p.stream_k) {
            const long long U = (long long)p.n_tiles * p.kb_per_tile;
            u0 = (long long)wid * U / nw;
            u1 = (long long)(wid + 1) * U / nw;
            cur = u0;
        } else {
            u0 = u1 = cur = 0;
        }
    }
    __device__ bool next(Seg& s) {
        if (p.stream_k) {
            if (cur >= u1) return false;
            s.tile = (int)(cur / p.kb_per_tile);
            s.kb0 = (int)(cur - (long long)s.tile * p.kb_per_tile);
            const long long left = u1 - cur;
            const int room = p.kb_per_tile - s.kb0;
            s.kb1 = s.kb0 + (int)(left < room ? left : room);
            s.start_unit = cur;
            cur += s.kb1 - s.kb0;
            return true;
        }
        long long t = (long long)wid + (long long)it * nw;
        if constexpr (DYN) if (it > 0) {
            if (role == 0) {
                t = pending;                   // claim_next() ran during the previous tile
            } else {
                unsigned long long v = 0;
                if (role == 1 || (threadIdx.x & 31) == 0) {
                    const unsigned long long* e = p.dyn_ring + (size_t)wid * kDynRing + (it & (kDynRing - 1));
                    uint64_t t0 = 0;
                    for (;;) {
                        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(e) : "memory");
                        if ((unsigned)(v >> 32) == ((gen << 12) | (unsigned)it)) break;
                        __nanosleep(64);
                        const uint64_t now = globaltimer();
                        if (t0 == 0) t0 = now;
                        else if (now - t0 > 5000000000ull) __trap();
                    }
                }
                if (role == 2) v = __shfl_sync(0xffffffffu, v, 0);
                t = (long long)(unsigned)(v & 0xffffffffu);
            }
        }
        if (t >= p.n_tiles) return false;
        ++it;
        s.tile = (int)t;
        s.kb0 = 0;
        s.kb1 = p.kb_per_tile;
        if (p.ks > 1) {                        // part r of ks takes k-blocks [KB*r/ks, KB*(r+1)/ks)
            s.kb0 = p.kb_per_tile * krank / p.ks;
            s.kb1 = p.kb_per_tile * (krank + 1) / p.ks;
        }
        s.start_unit = 0;
        return true;
    }
    // scheduler thread, once per tile (after the tile's first loads are in flight): claim the tile of the NEXT step and
    // publish it to this worker's other threads.  A claim at or past n_tiles is the stop mark.
    __device__ void claim_next() {
        const unsigned c = atomicAdd(p.dyn_ctr, 1u);
        const long long t = (long long)nw + (long long)c;
        pending = t < (long long)p.n_tiles ? (int)t : p.n_tiles;
        const unsigned long long v = ((unsigned long long)((gen << 12) | (unsigned)it) << 32) | (unsigned)pending;
        unsigned long long* e = p.dyn_ring + (size_t)wid * kDynRing + (it & (kDynRing - 1));
        asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(e), "l"(v) : "memory");
    }
};
// grouped rasterisation: group_x X-tiles form a group; inside a group x runs fastest.
__device__ __forceinline__ void tile_xy(const GemmParams& p, int tile, int& tx, int& ty) {
    const int per_group = p.group_x * p.tiles_y;
    const int g = tile / per_group;
    const int first_x = g * p.group_x;
    const int gsize = min(p.group_x, p.tiles_x - first_x);
    const int r = tile - g * per_group;
    tx = first_x + r % gsize;
    ty = r / gsize;
}

// ---- epilogue pieces ---------------------------------------------------------------------------
// 32 accumulator values acc[x][y0 .. y0+31] of row x -> C.
// fp32 C (ra_gemm_ex, c_dtype = RA_DTYPE_F32): same addressing, 4-byte elements, no rounding step
__device__ __forceinline__ void store_out_f32(const GemmParams& p, const float (&acc)[32], int x, int y0) {
    const float alpha = p.alpha, beta = p.beta;
    float* C = reinterpret_cast<float*>(p.C);
    if (!p.swap) {
        float* row = C + (size_t)x * p.ldc + y0;
        if (y0 + 32 <= p.RY) {
#pragma unroll
            for (int v = 0; v < 8; ++v) {
                float4 o = make_float4(alpha * acc[4 * v], alpha * acc[4 * v + 1], alpha * acc[4 * v + 2], alpha * acc[4 * v + 3]);
                if (beta != 0.f) {
                    const float4 c = *reinterpret_cast<const float4*>(row + 4 * v);
                    o.x = fmaf(beta, c.x, o.x); o.y = fmaf(beta, c.y, o.y); o.z = fmaf(beta, c.z, o.z); o.w = fmaf(beta, c.w, o.w);
                }
                *reinterpret_cast<float4*>(row + 4 * v) = o;
            }
        } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                if (y0 + j < p.RY) {
                    float r = alpha * acc[j];
                    if (beta != 0.f) r = fmaf(beta, row[j], r);
                    row[j] = r;
                }
            }
        }
    } else {
        float* ptr = C + (size_t)y0 * p.ldc + x;
        const size_t ld = (size_t)p.ldc;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            if (y0 + j < p.RY) {
                float r = alpha * acc[j];
                if (beta != 0.f) r = fmaf(beta, ptr[j * ld], r);
                ptr[j * ld] = r;
            }
        }
    }
}

__device__ __forceinline__ void store_out(const GemmParams& p, const float (&acc)[32], int x, int y0) {
    if (x >= p.RX || y0 >= p.RY) return;
    if (p.c_f32) {
        store_out_f32(p, acc, x, y0);
        return;
    }
    const float alpha = p.alpha, beta = p.beta;
    if (!p.swap) {
        __nv_bfloat16* row = p.C + (size_t)x * p.ldc + y0;
        if (y0 + 32 <= p.RY) {
            uint4 out[4];
            uint32_t* o = reinterpret_cast<uint32_t*>(out);
            if (beta != 0.f) {
                uint4 cin[4];
#pragma unroll
                for (int v = 0; v < 4; ++v) cin[v] = *reinterpret_cast<const uint4*>(row + 8 * v);
                const __nv_bfloat162* ci = reinterpret_cast<const __nv_bfloat162*>(cin);
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const float2 c = __bfloat1622float2(ci[j]);
                    const __nv_bfloat162 r = __floats2bfloat162_rn(fmaf(beta, c.x, alpha * acc[2 * j]),
                                                                   fmaf(beta, c.y, alpha * acc[2 * j + 1]));
                    o[j] = *reinterpret_cast<const uint32_t*>(&r);
                }
            } else {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const __nv_bfloat162 r = __floats2bfloat162_rn(alpha * acc[2 * j], alpha * acc[2 * j + 1]);
                    o[j] = *reinterpret_cast<const uint32_t*>(&r);
                }
            }
#pragma unroll
            for (int v = 0; v < 4; ++v) *reinterpret_cast<uint4*>(row + 8 * v) = out[v];
        } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                if (y0 + j < p.RY) {
                    float r = alpha * acc[j];
                    if (beta != 0.f) r = fmaf(beta, __bfloat162float(row[j]), r);
                    row[j] = __float2bfloat16_rn(r);
                }
            }
        }
    } else {
        // transposed store: lanes of a warp hold consecutive x -> each j is one coalesced 64-byte row piece.
        // Whole chunks take branch-free code (the guarded loop costs ~70 cycles per element in BSSY/BRA overhead:
        // 2.7 us of a 64 x 16384 x K GEMM's fixed time went there).
        __nv_bfloat16* ptr = p.C + (size_t)y0 * p.ldc + x;
        const size_t ld = (size_t)p.ldc;
        if (y0 + 32 <= p.RY && beta == 0.f) {
#pragma unroll
            for (int j = 0; j < 32; ++j) ptr[j * ld] = __float2bfloat16_rn(alpha * acc[j]);
        } else if (y0 + 32 <= p.RY) {
#pragma unroll
            for (int j = 0; j < 32; ++j)
                ptr[j * ld] = __float2bfloat16_rn(fmaf(beta, __bfloat162float(ptr[j * ld]), alpha * acc[j]));
        } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                if (y0 + j < p.RY) {
                    float r = alpha * acc[j];
                    if (beta != 0.f) r = fmaf(beta, __bfloat162float(ptr[j * ld]), r);
                    ptr[j * ld] = __float2bfloat16_rn(r);
                }
            }
        }
    }
}

// 32 accumulator values of row x, columns y0.. -> alpha/beta -> 16 packed bf16x2 (same arithmetic as store_out)
__device__ __forceinline__ void pack_out(const GemmParams& p, const uint32_t (&v)[32], int x, int y0, uint32_t (&o)[16]) {
    const float alpha = p.alpha, beta = p.beta;
    if (beta == 0.f) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const __nv_bfloat162 r = __floats2bfloat162_rn(alpha * __uint_as_float(v[2 * j]), alpha * __uint_as_float(v[2 * j + 1]));
            o[j] = *reinterpret_cast<const uint32_t*>(&r);
        }
        return;
    }
    const __nv_bfloat16* row = p.C + (size_t)x * p.ldc + y0;
    uint32_t cin[16];
    if (x < p.RX && y0 + 32 <= p.RY) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint4 t = *reinterpret_cast<const uint4*>(row + 8 * q);
            cin[4 * q] = t.x; cin[4 * q + 1] = t.y; cin[4 * q + 2] = t.z; cin[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const uint32_t lo = (x < p.RX && y0 + 2 * j < p.RY) ? (uint32_t)__bfloat16_as_ushort(row[2 * j]) : 0u;
            const uint32_t hi = (x < p.RX && y0 + 2 * j + 1 < p.RY) ? (uint32_t)__bfloat16_as_ushort(row[2 * j + 1]) : 0u;
            cin[j] = lo | (hi << 16);
        }
    }
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const float2 c = __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162*>(&cin[j]));
        const __nv_bfloat162 r = __floats2bfloat162_rn(fmaf(beta, c.x, alpha * __uint_as_float(v[2 * j])),
                                                       fmaf(beta, c.y, alpha * __uint_as_float(v[2 * j + 1])));
        o[j] = *reinterpret_cast<const uint32_t*>(&r);
    }
}

// DYN = dynamic tile order (see g_dyn).  A template parameter: compiled into every instantiation as a run-time branch it cost
// the single-wave shapes, which never take it, 5-10 % (2048^3: 18.5 -> 20.5 us).  Instantiated for CTA-pair tiles only.
template <int BN, int CG, int XH, int KBK, bool DYN>
__global__ void __launch_bounds__(256, 2)
gemm_kernel(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapY,
            const __grid_constant__ CUtensorMap mapC, const GemmParams p, Trace tr) {
    // CG == 2: the CTA pair of a 2-cluster works on one 256 x BN tile.  Each CTA stages its own 128 rows of X
    // and its own BN/2 rows of Y; the leader (cluster rank 0) issues tcgen05.mma.cta_group::2, which reads both
    // CTAs' stages and writes rows [128*rank, 128*rank+128) of the accumulator into each CTA's TMEM.
    //
    // XH == 2 ("big" tiles): every CTA owns 256 rows of X as two 128-row blocks that share one Y stage, i.e. two
    // MMAs per k-step into two accumulators (TMEM columns [0,BN) and [BN,2BN)).  A pair then covers 512 x 256 and
    // stages 256 + 128 rows per k-block instead of 2 x (128 + 128): 25 % less L2->SM traffic per flop, which is
    // what bounds the 256 x 256 pair tile (64 B/clk/SM).  The price: both accumulators belong to the current
    // tile, so the epilogue overlaps only the first k-blocks of the next tile (see the MMA issuer).
    constexpr int kYRows = BN / CG;
    // KBK = k extent of one pipeline stage: 64 (128-byte swizzle rows) or 32 (64-byte rows; K-major operands only).  A template
    // parameter, not a run-time one: as a run-time value it cost the weight-streaming GEMM 5 % (87.4 -> 92.0 us), whose
    // producer thread has no slack for the extra address arithmetic per k-block.
    static_assert(KBK == 64 || KBK == 32, "KBK");
    constexpr int kXHalfBytes = kBM * KBK * 2;
    constexpr int kXBytes = XH * kXHalfBytes;
    constexpr int kStageBytes = kXBytes + kYRows * KBK * 2;
    constexpr int kTmemCols = 2 * BN;   // XH == 1: two accumulators (double buffer); XH == 2: the two X blocks of one tile
    constexpr int kTileX = kBM * XH * CG;
    constexpr uint32_t kIdesc = umma_idesc_bf16(kBM * CG, BN);
    static_assert(BN == 64 || BN == 128 || BN == 256, "BN");
    static_assert(CG == 1 || CG == 2, "CG");
    static_assert(XH == 1 || XH == 2, "XH");
    static_assert(kStageBytes == stage_bytes(BN, CG, XH) * KBK / kBK, "stage size");

    extern __shared__ uint8_t smem_raw[];
    // 1024-byte alignment for the 128B swizzle; the barrier block sits after the stages.  Both CTAs of a pair
    // compute identical offsets (same kernel, same dynamic-smem base), which cta_group::2 relies on.
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t epi_base = smem_base + p.stages * kStageBytes;     // staging for TMA stores (epi_tma only)
    const uint32_t bar_base = epi_base + (p.epi_tma ? kEpiStageBytes : 0);
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (kMaxStages + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * kMaxStages + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * kMaxStages + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * kMaxStages + 4);
    const uint32_t flag_slot = tmem_slot + 8;
    const uint32_t ks_ready_bar = tmem_slot + 16;   // in CTA 1: CTA 0's stages are free to receive the accumulator
    const uint32_t ks_data_bar = tmem_slot + 24;    // in CTA 0: CTA 1's accumulator has landed
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));   // generic view of smem_base

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    // cluster layout: [k-half (cluster split-K)][pair rank (CG == 2)] -- a CTA pair is two consecutive cluster ranks
    const uint32_t crank = (CG == 2 || p.ks > 1) ? cluster_ctarank() : 0u;
    const uint32_t rank = (CG == 2) ? (crank & 1u) : 0u;               // rank inside the CTA pair, 0 = leader
    const uint32_t lead = (CG == 2) ? (crank & ~1u) : crank;           // cluster rank of this CTA's pair leader
    const uint16_t pair_mask = (uint16_t)(3u << lead);                 // both CTAs of the pair (CG == 2 commits)
    const int kdiv = CG * p.ks;                                        // CTAs per worker
    const int wid = (int)(blockIdx.x / kdiv), nw = (int)(gridDim.x / kdiv);
    const int krank = (p.ks > 1) ? (int)(crank / CG) : 0;
    uint64_t* rec = (threadIdx.x == 0) ? trace_begin(tr, KID_GEMM) : nullptr;
    const uint32_t my_sm = smid();

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapX) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapY) : "memory");
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(full_bar(s), CG);           // one arrive.expect_tx per producer of the pair
            mbar_init(empty_bar(s), 1);           // one tcgen05.commit (multicast to both CTAs when CG == 2)
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(tfull_bar(b), 1);
            mbar_init(tempty_bar(b), 4 * CG);     // one arrive per epilogue warp of the pair
        }
        mbar_init(ks_ready_bar, 4);               // one arrive per epilogue warp of CTA 0
        mbar_init(ks_data_bar, 1);                // one arrive.expect_tx by part 0; the senders' bulk copies complete the bytes
        mbar_fence_init();
    }
    if (warp == 1) {
        if constexpr (CG == 1) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot),
                         "r"((uint32_t)kTmemCols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot),
                         "r"((uint32_t)kTmemCols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    if (CG == 2 || p.ks > 1) cluster_sync_all();  // the peer's barriers exist before anything remote touches them
    else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t*>(smem_gen + (tmem_slot - smem_base));

    if (warp == 0) {
        // ================= TMA producer (one per CTA) =================
        if (lane == 0) {
            const uint64_t polX = make_policy(p.hintX), polY = make_policy(p.hintY);
            Sched<DYN> sched(p, wid, nw, krank, rank == 0 ? 0 : 1);      // the pair leader's producer is the worker's scheduler thread
            Seg sg;
            int stage = 0;
            uint32_t phase = 0;
            while (sched.next(sg)) {
                int tx, ty;
                tile_xy(p, sg.tile, tx, ty);
                const int x0 = tx * kTileX + (int)rank * (kBM * XH);
                const int y0 = ty * BN + (int)rank * kYRows;
                const int claim_at = sg.kb0 + min(p.stages, sg.kb1 - sg.kb0 - 1);   // pipeline full: the claim's round trip is hidden
                for (int kb = sg.kb0; kb < sg.kb1; ++kb) {
                    if constexpr (DYN) if (rank == 0 && kb == claim_at) sched.claim_next();
                    mbar_wait(empty_bar(stage), phase ^ 1u);           // local: MMAs reading this stage retired
                    const uint32_t sx = smem_base + stage * kStageBytes;
                    uint32_t bar;
                    if constexpr (CG == 1) {
                        bar = full_bar(stage);
                        mbar_expect_tx(bar, kStageBytes);
                    } else {
                        bar = mapa(full_bar(stage), lead);            // the leader's barrier collects both halves
                        mbar_expect_tx_cluster(bar, kStageBytes);
                    }
                    // K-major operand: one box (64 k x rows).  MN-major operand: one box (64 rows x 64 k) per 64 rows.
                    if (!p.xmn) {
                        tma_load_2d<CG>(sx, &mapX, kb * KBK, x0, bar, polX);
                    } else {
#pragma unroll
                        for (int b = 0; b < kBM * XH / 64; ++b) tma_load_2d<CG>(sx + b * 8192, &mapX, x0 + 64 * b, kb * kBK, bar, polX);
                    }
                    if (!p.ymn) {
                        tma_load_2d<CG>(sx + kXBytes, &mapY, kb * KBK, y0, bar, polY);
                    } else {
#pragma unroll
                        for (int b = 0; b < kYRows / 64; ++b)
                            tma_load_2d<CG>(sx + kXBytes + b * 8192, &mapY, y0 + 64 * b, kb * kBK, bar, polY);
                    }
                    if (++stage == p.stages) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================= MMA issuer (leader CTA only) =================
        if (lane == 0 && rank == 0) {
            Sched<DYN> sched(p, wid, nw, krank);
            Seg sg;
            int stage = 0;
            uint32_t phase = 0;
            int acc_it = 0;
            const uint32_t idesc = kIdesc | ((uint32_t)p.xmn << 15) | ((uint32_t)p.ymn << 16);
            const int kx_step = p.xmn ? (2048 >> 4) : (32 >> 4), ky_step = p.ymn ? (2048 >> 4) : (32 >> 4);
            // the four UMMA_K steps of X block h against the Y rows of one stage, into accumulator column acc_col
            auto issue_block = [&](int st, int h, uint32_t acc_col, bool first) {
                const uint32_t sx = smem_base + st * kStageBytes;
                const uint32_t sxh = sx + h * kXHalfBytes;
                if constexpr (KBK == 32) {         // two UMMA_K steps per stage, 64-byte swizzle (K-major operands only)
                    const uint64_t dx = umma_desc_sw64(sxh), dy = umma_desc_sw64(sx + kXBytes);
#pragma unroll
                    for (int k = 0; k < 2; ++k)
                        umma_bf16<CG>(tmem_base + acc_col, dx + (uint64_t)(2 * k), dy + (uint64_t)(2 * k), idesc, (!first || k > 0) ? 1u : 0u);
                    return;
                }
                const uint64_t dx = p.xmn ? umma_desc_sw128_mn(sxh) : umma_desc_sw128(sxh);
                const uint64_t dy = p.ymn ? umma_desc_sw128_mn(sx + kXBytes) : umma_desc_sw128(sx + kXBytes);
#pragma unroll
                for (int k = 0; k < kBK / kUmmaK; ++k) {
                    // per UMMA_K step: K-major +32 B inside the swizzle atom, MN-major +2 k-groups of 1024 B
                    umma_bf16<CG>(tmem_base + acc_col, dx + (uint64_t)(kx_step * k), dy + (uint64_t)(ky_step * k), idesc,
                                  (!first || k > 0) ? 1u : 0u);
                }
            };
            auto wait_full = [&](int st, uint32_t ph) {
                mbar_wait(full_bar(st), ph);               // TMA bytes (of both CTAs) have landed
                tc_fence_after();
            };
            auto wait_drained = [&](int b, uint32_t ph) {
                mbar_wait(tempty_bar(b), ph);              // every epilogue warp (of the pair) drained this accumulator
                tc_fence_after();
            };
            while (sched.next(sg)) {
                if constexpr (XH == 1) {
                    // two accumulators (acc_it & 1): the epilogue of tile i overlaps the whole main loop of tile i+1
                    const int buf = acc_it & 1;
                    wait_drained(buf, ((acc_it >> 1) & 1) ^ 1u);
                    for (int kb = sg.kb0; kb < sg.kb1; ++kb) {
                        wait_full(stage, phase);
                        issue_block(stage, 0, (uint32_t)(buf * BN), kb == sg.kb0);
                        umma_commit<CG>(empty_bar(stage), pair_mask);   // frees the smem stage (in both CTAs) when these MMAs retire
                        if (++stage == p.stages) { stage = 0; phase ^= 1u; }
                    }
                    umma_commit<CG>(tfull_bar(buf), pair_mask);         // accumulator complete (signals both CTAs' epilogues)
                } else {
                    // X block h accumulates in columns [h*BN, h*BN + BN); both belong to this tile, so the TMEM drain
                    // (64 B/clk: ~2k cycles per block) cannot hide behind a second buffer.  Instead the two blocks are
                    // skewed by D k-blocks at both ends of the tile: block 0 finishes D k-blocks early and is drained
                    // while block 1 finishes; in the next tile block 0 starts as soon as it is drained and runs D
                    // k-blocks ahead while block 1 is drained.  In between they run in lockstep so that a stage is
                    // held no longer than needed (D <= stages: a stage is released by block 1).
                    const uint32_t aph = (uint32_t)(acc_it & 1);
                    const int nkb = sg.kb1 - sg.kb0;
                    const int D = (p.skew > 0 && nkb >= 2 * p.skew) ? p.skew : 0;
                    int sb = stage, ia = 0, ib = 0;          // block 1's stage cursor; k-blocks issued per block
                    auto step_a = [&]() {
                        wait_full(stage, phase);
                        if (ia == 0) wait_drained(0, aph ^ 1u);
                        issue_block(stage, 0, 0u, ia == 0);
                        if (++stage == p.stages) { stage = 0; phase ^= 1u; }
                        ++ia;
                    };
                    auto step_b = [&]() {
                        if (ib == 0) wait_drained(1, aph ^ 1u);
                        issue_block(sb, 1, (uint32_t)BN, ib == 0);
                        umma_commit<CG>(empty_bar(sb), pair_mask);       // frees the smem stage (in both CTAs) when these MMAs retire
                        if (++sb == p.stages) sb = 0;
                        ++ib;
                    };
                    while (ia < D) step_a();                 // head: block 0 runs ahead
                    while (ib < D) step_b();                 //       block 1 catches up
                    while (ia < nkb - D) { step_a(); step_b(); }
                    while (ia < nkb) step_a();               // tail: block 0 finishes first ...
                    umma_commit<CG>(tfull_bar(0), pair_mask);
                    while (ib < nkb) step_b();               //       ... and is drained while block 1 finishes
                    umma_commit<CG>(tfull_bar(1), pair_mask);
                }
                ++acc_it;
            }
        }
    } else {
        // ================= epilogue (warps 2..5 of every CTA) =================
        const int quarter = warp & 3;                       // TMEM lane quarter this warp may read
        const int xl = quarter * 32 + lane;                 // row inside this CTA's 128-row slab
        const int et = threadIdx.x - 64;                    // 0..127
        // residency count-in (after the set-up barrier, so the atomic's round trip delays nothing: this warp's next
        // action is the wait for the first accumulator)
        if (et == 0) atomicMax(&g_gemm_max_resident, atomicAdd(&g_gemm_resident[my_sm], 1) + 1);
        Sched<DYN> sched(p, wid, nw, krank, 2);
        Seg sg;
        int acc_it = 0;
        uint32_t sbuf_it = 0;                               // staging-buffer rotation (per warp)
        const uint64_t polC = make_policy(p.hintC);
        while (sched.next(sg)) {
            const int buf = (XH == 1) ? (acc_it & 1) : 0;
            const uint32_t aphase = (XH == 1) ? ((acc_it >> 1) & 1) : (acc_it & 1);
            int tx, ty;
            tile_xy(p, sg.tile, tx, ty);
            const bool whole = (sg.kb0 == 0 && sg.kb1 == p.kb_per_tile);
            const int x = tx * kTileX + (int)rank * (kBM * XH) + xl;   // row of X block 0
            if (XH == 1 && p.ks > 1) {
                // ---- cluster split-K: part r of the cluster holds the sum over the r-th slice of the k-blocks.  Parts
                // 1 .. ks-1 stage their accumulators in their OWN (now idle) stage ring -- layout [32-column chunk][row]
                // [32 floats], the eight 16-byte pieces of a row XOR-swizzled by (row & 7) against bank conflicts -- and
                // ship them with one bulk copy each through distributed shared memory into a slot of part 0's ring
                // (register -> remote st.shared measured 6-7 us per 128 KiB accumulator; the bulk copy is asynchronous
                // and completes bytes on part 0's mbarrier).  Part 0 adds its own slice FIRST, then the slots in
                // ascending k, applies alpha/beta and stores.  No global-memory round trip, bit-reproducible.
                mbar_wait(tfull_bar(buf), aphase);
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(buf * BN);
                const uint32_t sw = (uint32_t)(xl & 7);
                constexpr uint32_t kSlotBytes = (uint32_t)kBM * BN * 4;
                if (krank >= 1) {
                    const uint32_t home = crank - (uint32_t)krank * CG;        // same CTA of the pair / tile, k-slice 0
#pragma unroll 1
                    for (int c = 0; c < BN / 32; ++c) {
                        uint32_t v[32];
                        tmem_ld32(taddr + c * 32, v);
                        tmem_ld_wait();
                        const uint32_t drow = smem_base + (uint32_t)((c * kBM + xl) * 128);   // own ring: the MMAs are done
#pragma unroll
                        for (int q = 0; q < 8; ++q)
                            st_shared_v4(drow + (((uint32_t)q ^ sw) << 4), v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
                    }
                    fence_async_smem();
                    epi_bar_sync();
                    if (et == 0) {
                        mbar_wait_acquire_cluster(ks_ready_bar, 0);            // part 0's MMAs no longer read its stages
                        dsmem_bulk_copy(mapa(smem_base, home) + (uint32_t)(krank - 1) * kSlotBytes, smem_base, kSlotBytes,
                                        mapa(ks_data_bar, home));
                    }
                } else {
                    __syncwarp();
                    if (lane == 0)
                        for (int r = 1; r < p.ks; ++r) mbar_arrive_release_cluster(mapa(ks_ready_bar, crank + (uint32_t)r * CG));
                    if (et == 0) mbar_expect_tx(ks_data_bar, (uint32_t)(p.ks - 1) * kSlotBytes);
                    mbar_wait_acquire_cluster(ks_data_bar, 0);
#pragma unroll 1
                    for (int c = 0; c < BN / 32; ++c) {
                        uint32_t v[32];
                        tmem_ld32(taddr + c * 32, v);
                        tmem_ld_wait();
                        float acc[32];
#pragma unroll
                        for (int j = 0; j < 32; ++j) acc[j] = __uint_as_float(v[j]);
#pragma unroll 1
                        for (int r = 1; r < p.ks; ++r) {                       // slots in ascending k
                            const uint32_t srow = smem_base + (uint32_t)(r - 1) * kSlotBytes + (uint32_t)((c * kBM + xl) * 128);
#pragma unroll
                            for (int q = 0; q < 8; ++q) {
                                uint32_t a, b, cc, d;
                                ld_shared_v4(srow + (((uint32_t)q ^ sw) << 4), a, b, cc, d);
                                acc[4 * q + 0] = __fadd_rn(acc[4 * q + 0], __uint_as_float(a));
                                acc[4 * q + 1] = __fadd_rn(acc[4 * q + 1], __uint_as_float(b));
                                acc[4 * q + 2] = __fadd_rn(acc[4 * q + 2], __uint_as_float(cc));
                                acc[4 * q + 3] = __fadd_rn(acc[4 * q + 3], __uint_as_float(d));
                            }
                        }
                        store_out(p, acc, x, ty * BN + c * 32);
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (CG == 1) mbar_arrive(tempty_bar(buf));
                    else mbar_arrive_cluster(mapa(tempty_bar(buf), lead));
                }
                ++acc_it;
                continue;
            }
            float* part = nullptr;
            if (!whole) {
                const int slot = 2 * wid + (sg.start_unit == sched.u0 ? 0 : 1);
                part = p.partials + (size_t)slot * (kBM * BN);
            }
#pragma unroll 1
            for (int h = 0; h < XH; ++h) {
                const int acc_idx = (XH == 1) ? buf : h;
                mbar_wait(tfull_bar(acc_idx), aphase);
                tc_fence_after();
                const uint32_t taddr = tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(acc_idx * BN);
                if (whole && p.epi_tma) {
                    // registers -> swizzled shared memory (this warp's 32 rows x 64 columns) -> one TMA store per box;
                    // full 128-byte lines leave the SM, the tensor map clips ragged edges.
                    const int row0 = tx * kTileX + (int)rank * (kBM * XH) + h * kBM + quarter * 32;
#pragma unroll 1
                    for (int cc = 0; cc < BN / kEpiBoxCols; ++cc) {
                        const uint32_t sbuf = epi_base + (uint32_t)((quarter * 2 + (sbuf_it & 1)) * kEpiBufBytes);
                        ++sbuf_it;
                        const int y0 = ty * BN + cc * kEpiBoxCols;
                        if (y0 + kEpiBoxCols > p.RY && (p.RY & 7)) {
                            // TMA stores clip at 16-byte granularity: with N % 8 != 0 the box holding the ragged edge
                            // would overwrite up to 7 pad elements after column N-1 (found by the guard-band test), so
                            // that one box per row of tiles goes out through predicated element stores instead.
#pragma unroll 1
                            for (int hf = 0; hf < 2; ++hf) {
                                uint32_t v[32];
                                tmem_ld32(taddr + cc * kEpiBoxCols + hf * 32, v);
                                tmem_ld_wait();
                                float acc[32];
#pragma unroll
                                for (int j = 0; j < 32; ++j) acc[j] = __uint_as_float(v[j]);
                                store_out(p, acc, row0 + lane, y0 + hf * 32);
                            }
                            --sbuf_it;      // no staging buffer was used: keep the two-deep rotation intact
                            continue;
                        }
                        if (lane == 0) bulk_wait_read<1>();       // the store that last read this buffer has drained it
                        __syncwarp();
                        const uint32_t srow = sbuf + (uint32_t)lane * 128u;
                        const uint32_t sw = (uint32_t)(lane & 7);
#pragma unroll
                        for (int hf = 0; hf < 2; ++hf) {
                            uint32_t v[32], o[16];
                            tmem_ld32(taddr + cc * kEpiBoxCols + hf * 32, v);
                            tmem_ld_wait();
                            pack_out(p, v, row0 + lane, y0 + hf * 32, o);
#pragma unroll
                            for (int q = 0; q < 4; ++q)
                                st_shared_v4(srow + (((uint32_t)(q + 4 * hf) ^ sw) << 4), o[4 * q], o[4 * q + 1], o[4 * q + 2], o[4 * q + 3]);
                        }
                        fence_async_smem();
                        __syncwarp();
                        if (lane == 0) {
                            if (row0 < p.RX && y0 < p.RY) tma_store_2d(&mapC, sbuf, y0, row0, polC);
                            bulk_commit();
                        }
                    }
                } else {
#pragma unroll 1
                    for (int c = 0; c < BN / 32; ++c) {
                        uint32_t v[32];
                        tmem_ld32(taddr + c * 32, v);
                        tmem_ld_wait();
                        float acc[32];
#pragma unroll
                        for (int j = 0; j < 32; ++j) acc[j] = __uint_as_float(v[j]);
                        if (whole) {
                            store_out(p, acc, x + h * kBM, ty * BN + c * 32);
                        } else {
#pragma unroll
                            for (int j = 0; j < 32; ++j) __stcg(part + (size_t)(c * 32 + j) * kBM + xl, acc[j]);
                        }
                    }
                }
                // this warp's quarter of the accumulator is drained: tell the (leader's) MMA issuer
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (CG == 1) mbar_arrive(tempty_bar(acc_idx));
                    else mbar_arrive_cluster(mapa(tempty_bar(acc_idx), lead));
                }
            }
            ++acc_it;

            if (!whole) {
                // ---- stream-K fix-up (CG == 1 only): last part to arrive reduces all parts in ascending-k order ----
                const long long U = (long long)p.n_tiles * p.kb_per_tile;
                const long long G = nw;
                const long long ua = (long long)sg.tile * p.kb_per_tile;          // first unit of the tile
                const long long ub = ua + p.kb_per_tile - 1;                      // last unit of the tile
                const int c_first = (int)(((ua + 1) * G - 1) / U);
                const int c_last = (int)(((ub + 1) * G - 1) / U);
                const int n_parts = c_last - c_first + 1;
                __threadfence();
                epi_bar_sync();
                volatile int* flag = reinterpret_cast<volatile int*>(smem_gen + (flag_slot - smem_base));
                if (et == 0) {
                    const int old = atomicAdd(p.counters + sg.tile, 1);
                    *flag = (old == n_parts - 1) ? 1 : 0;
                }
                epi_bar_sync();
                const bool last = (*flag != 0);
                epi_bar_sync();   // everyone has read the flag before a later segment overwrites it
                if (last) {
                    __threadfence();
#pragma unroll 1
                    for (int c = 0; c < BN / 32; ++c) {
                        float acc[32];
#pragma unroll 1
                        for (int cc = c_first; cc <= c_last; ++cc) {
                            const long long cu0 = (long long)cc * U / G;
                            const long long seg_start = cu0 > ua ? cu0 : ua;
                            const int slot = 2 * cc + (seg_start == cu0 ? 0 : 1);
                            const float* src = p.partials + (size_t)slot * (kBM * BN) + (size_t)(c * 32) * kBM + xl;
                            if (cc == c_first) {
#pragma unroll
                                for (int j = 0; j < 32; ++j) acc[j] = __ldcg(src + (size_t)j * kBM);
                            } else {
#pragma unroll
                                for (int j = 0; j < 32; ++j) acc[j] = __fadd_rn(acc[j], __ldcg(src + (size_t)j * kBM));
                            }
                        }
                        store_out(p, acc, x, ty * BN + c * 32);
                    }
                }
            }
        }
    }

    if (warp >= 2 && lane == 0 && p.epi_tma) bulk_wait_all();   // this warp's TMA stores have left shared memory

    // teardown: nobody may exit (or free TMEM) while the peer can still signal its barriers / read its stages
    tc_fence_before();
    if (CG == 2 || p.ks > 1) cluster_sync_all();
    else __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        if constexpr (CG == 1)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)kTmemCols) : "memory");
        else
            asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)kTmemCols) : "memory");
    }
    if (threadIdx.x == 64) atomicSub(&g_gemm_resident[my_sm], 1);
    if constexpr (DYN) if (threadIdx.x == 32) {
        // the last CTA to get here re-arms the slot for the next launch (every thread of every CTA is past its schedule)
        __threadfence();
        if (atomicAdd(p.dyn_ctr + 1, 1u) == gridDim.x - 1) {
            const unsigned g = *(volatile unsigned*)(p.dyn_ctr + 2);
            p.dyn_ctr[0] = 0u;
            p.dyn_ctr[1] = 0u;
            __threadfence();
            *(volatile unsigned*)(p.dyn_ctr + 2) = (g + 1u) & 0xFFFFFu;
        }
    }
    if (threadIdx.x == 0) trace_end(rec);
}

// C = beta * C  (K == 0 or alpha == 0: op(A), op(B) are not referenced, as in BLAS)
__global__ void scale_c_kernel(void* Cv, int M, int N, int ldc, float beta, int c_f32) {
    const size_t total = (size_t)M * N;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t r = i / N, c = i - r * N;
        if (c_f32) {
            float* ptr = static_cast<float*>(Cv) + r * ldc + c;
            *ptr = (beta == 0.f) ? 0.f : beta * *ptr;
        } else {
            __nv_bfloat16* ptr = static_cast<__nv_bfloat16*>(Cv) + r * ldc + c;
            *ptr = (beta == 0.f) ? __float2bfloat16_rn(0.f) : __float2bfloat16_rn(beta * __bfloat162float(*ptr));
        }
    }
}

// ---- host: tensor maps -------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn g_encode = nullptr;
static std::once_flag g_encode_once;

static ra_status get_encode(EncodeTiledFn* fn) {
    static cudaError_t err = cudaSuccess;
    std::call_once(g_encode_once, [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qres;
        err = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres);
        if (err == cudaSuccess && qres == cudaDriverEntryPointSuccess) g_encode = reinterpret_cast<EncodeTiledFn>(f);
    });
    if (g_encode == nullptr) return cuda_fail(err != cudaSuccess ? err : cudaErrorSymbolNotFound);
    *fn = g_encode;
    return RA_OK;
}

// K-major operand: rows x K bf16, row pitch ld; box = 64 (k) x box_rows.  MN-major operand: K x rows bf16 (rows
// contiguous), pitch ld; box = 64 (rows) x 64 (k).  128-byte swizzle, OOB -> zeros.
static ra_status make_map(CUtensorMap* map, const void* base, int rows, int K, int ld, int box_rows, int mn_major, int bk = kBK) {
    EncodeTiledFn enc;
    RA_TRY(get_encode(&enc));
    const cuuint64_t dims[2] = {(cuuint64_t)(mn_major ? rows : K), (cuuint64_t)(mn_major ? K : rows)};
    const cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
    const cuuint32_t box[2] = {(cuuint32_t)(mn_major ? 64 : bk), (cuuint32_t)(mn_major ? kBK : box_rows)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, (!mn_major && bk == 32) ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        g_last_cuda_error = (int)cudaErrorInvalidValue;
        return RA_ERR_CUDA;
    }
    return RA_OK;
}

// ---- host: kernel instantiations, their one-time attributes, and what the hardware says about residency --------
template <int KBK>
static const void* gemm_kernel_ptr_k(int bn, int cg, int xh, int dyn) {
    if (cg == 2 && xh == 2) return dyn ? reinterpret_cast<const void*>(&gemm_kernel<256, 2, 2, KBK, true>) : reinterpret_cast<const void*>(&gemm_kernel<256, 2, 2, KBK, false>);
    if (cg == 2) return dyn ? reinterpret_cast<const void*>(&gemm_kernel<256, 2, 1, KBK, true>) : reinterpret_cast<const void*>(&gemm_kernel<256, 2, 1, KBK, false>);
    switch (bn) {
        case 64: return reinterpret_cast<const void*>(&gemm_kernel<64, 1, 1, KBK, false>);
        case 128: return reinterpret_cast<const void*>(&gemm_kernel<128, 1, 1, KBK, false>);
        case 256: return reinterpret_cast<const void*>(&gemm_kernel<256, 1, 1, KBK, false>);
    }
    return nullptr;
}
static const void* gemm_kernel_ptr(int bn, int cg, int xh, int bk = kBK, int dyn = 0) {
    return bk == 32 ? gemm_kernel_ptr_k<32>(bn, cg, xh, dyn) : gemm_kernel_ptr_k<64>(bn, cg, xh, dyn);
}
static int kernel_slot(int bn, int cg, int xh, int bk, int dyn) {
    return (dyn ? 10 : 0) + (bk == 32 ? 5 : 0) + (cg == 2 ? (xh == 2 ? 4 : 3) : (bn == 64 ? 0 : (bn == 128 ? 1 : 2)));
}

static std::mutex g_gemm_mu;                 // guards the attribute flags and the launch cache below
static bool g_attr_set[64][20] = {};          // [device][instantiation]: MaxDynamicSharedMemorySize raised to the opt-in limit

// cudaFuncSetAttribute once per (device, instantiation), not once per launch.  Caller holds g_gemm_mu.
static ra_status prepare_kernel(const DeviceInfo& di, int bn, int cg, int xh, int bk, int dyn) {
    const int slot = kernel_slot(bn, cg, xh, bk, dyn);
    if (di.device >= 0 && di.device < 64 && g_attr_set[di.device][slot]) return RA_OK;
    RA_CUDA(cudaFuncSetAttribute(gemm_kernel_ptr(bn, cg, xh, bk, dyn), cudaFuncAttributeMaxDynamicSharedMemorySize, di.smem_per_block_optin));
    // The SM's shared-memory / L1 split is configured for the kernel that lands on it and is not changed while CTAs are
    // resident.  A GEMM CTA that was shrunk to honour smem_reserve_bytes must therefore ask for the FULL split, or the
    // memory it leaves free does not exist as shared memory and the collective's ring cannot move in beside it
    // (profiles/r03_residency.md: 0.000 co-residency before this).  The GEMM reads through TMA, not L1: nothing is lost.
    RA_CUDA(cudaFuncSetAttribute(gemm_kernel_ptr(bn, cg, xh, bk, dyn), cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    if (di.device >= 0 && di.device < 64) g_attr_set[di.device][slot] = true;
    return RA_OK;
}

// GEMM CTAs one SM can hold at this footprint: the minimum over the SM's launch-time resources -- registers,
// threads, shared memory.  On a device the inputs are read from it (the instantiation's real register count from
// cudaFuncGetAttributes, registers / threads / shared memory per SM from cudaDeviceGetAttribute); without one (plan
// queries on a CPU box) they are B200's: 128 registers x 192 threads -> 2 CTAs by registers.
//
// Why not cudaOccupancyMaxActiveBlocksPerMultiprocessor (what round 1's header promised): measured on B200 / CUDA 12.9
// it answers 1 for every instantiation of this kernel at EVERY footprint, down to 25 KiB of dynamic shared memory,
// while the %smid trace and the kernel's own per-SM counter (ra_gemm_residency) show two of these CTAs running on one
// SM at the same time at exactly that footprint (tests/test_overlap_gpu.py, reserve 200 KiB next to the allreduce).
// The API under-reports; the resource arithmetic below is the bound the hardware was seen to reach.
static int resident_ctas(const DeviceInfo* di, int bn, int cg, int xh, int dyn, int smem_per_sm, int reserved) {
    int regs_per_thread = 128, regs_per_sm = 65536, threads_per_sm = 2048;
    if (di != nullptr) {
        std::lock_guard<std::mutex> lk(g_gemm_mu);
        cudaFuncAttributes fa;
        int v = 0;
        if (cudaFuncGetAttributes(&fa, gemm_kernel_ptr(bn, cg, xh)) == cudaSuccess && fa.numRegs > 0) regs_per_thread = fa.numRegs;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxRegistersPerMultiprocessor, di->device) == cudaSuccess && v > 0) regs_per_sm = v;
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxThreadsPerMultiProcessor, di->device) == cudaSuccess && v > 0) threads_per_sm = v;
        (void)cudaGetLastError();
    }
    // registers are allocated per warp, in units of 8 per thread
    const int regs_per_cta = ((regs_per_thread + 7) / 8 * 8) * 32 * (kGemmThreads / 32);
    int n = smem_per_sm / (dyn + reserved);
    if (regs_per_sm / regs_per_cta < n) n = regs_per_sm / regs_per_cta;
    if (threads_per_sm / kGemmThreads < n) n = threads_per_sm / kGemmThreads;
    return n;
}

// ---- host: S3 planner ----------------------------------------------------------------------------
struct Plan {
    ra_gemm_plan pub;
    int bn;
    int epi_tma;       // whole tiles leave through the shared-memory staging area + TMA stores
    int hint_x;        // L2 policy of the X loads when an X panel is kept resident (2 = evict_last), else 0
    size_t counters_bytes, ws_bytes;
};

static ra_status validate_shape(int transA, int transB, int M, int N, int K) {
    if ((transA != 0 && transA != 1) || (transB != 0 && transB != 1)) return RA_ERR_INVALID_ARG;
    if (M < 0 || N < 0 || K < 0) return RA_ERR_INVALID_ARG;
    return RA_OK;
}

// cudaDevAttrMaxPersistingL2CacheSize of the current device, or B200's figure (79 MiB) where no device can be asked
// (the planner also runs host-only).  Asked once.
static long long max_persisting_l2() {
    static const long long v = [] {
        int dev = -1, bytes = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&bytes, cudaDevAttrMaxPersistingL2CacheSize, dev) == cudaSuccess && bytes > 0)
            return (long long)bytes;
        (void)cudaGetLastError();
        return (long long)79 << 20;
    }();
    return v;
}

static ra_status make_plan(int transA, int transB, int M, int N, int K, const ra_occupancy* occ_in, Plan* out) {
    RA_TRY(validate_shape(transA, transB, M, N, K));
    ra_occupancy occ = {0, 0, 0, 1, 0, 0, 0, 0, 0, 0};
    if (occ_in) occ = *occ_in;
    if (occ.smem_reserve_bytes < 0 || occ.sm_budget < 0 || occ.tiles_per_cta < 0) return RA_ERR_INVALID_ARG;

    // device facts (B200 constants when no device is present, so plans can be queried on a CPU box)
    int sm_count = kDefaultSmCount, smem_per_sm = kDefaultSmemPerSm, optin = kDefaultSmemPerBlockOptin,
        reserved = kDefaultSmemReservedPerBlock;
    DeviceInfo di;
    const DeviceInfo* dev = nullptr;               // non-NULL: an sm_100 device is current, ask it about residency
    if (device_info(&di) == RA_OK) {
        sm_count = di.sm_count;
        smem_per_sm = di.smem_per_sm;
        optin = di.smem_per_block_optin;
        reserved = di.smem_reserved_per_block;
        if (di.cc_major == 10) dev = &di;
    } else {
        g_last_cuda_error = 0;
        (void)cudaGetLastError();
    }
    Plan pl{};
    ra_gemm_plan& g = pl.pub;
    int clamped = 0;

    int budget = occ.sm_budget == 0 ? sm_count : occ.sm_budget;
    if (budget > sm_count) {
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        budget = sm_count;
        clamped = 1;
    }

    // skinny M (weight streaming): the long weight dimension becomes the 128-row X side, the M tokens the Y side
    // (BN = 64 or 128), so N/128 independent tiles stream the weights without any K split.
    const int swap = ((M <= 64 && N >= 128) || (M <= 128 && N >= 1024)) ? 1 : 0;
    const int RX = swap ? N : M, RY = swap ? M : N;
    int bn = RY > 128 ? 256 : (RY > 64 ? 128 : 64);
    // tile_k (N3: the paper's opt1 / opt2 differ in TILE_K): 32 halves every pipeline stage (64-byte
    // swizzle rows, two UMMA_K steps per stage).  K-contiguous operands only; cluster split-K keeps 64.
    if (occ.tile_k != 0 && occ.tile_k != 32 && occ.tile_k != 64) return RA_ERR_INVALID_ARG;
    int bk = kBK;
    if (occ.tile_k == 32) {
        if (transA == 0 && transB == 1 && occ.cluster_k < 2) {
            bk = 32;
        } else {
            if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
            clamped = 1;
        }
    }
    const int kb = (K + bk - 1) / bk;
    auto stage_bytes = [bk](int bn_, int cg_, int xh_) { return ra::stage_bytes(bn_, cg_, xh_) * bk / kBK; };
    // Small problems: when narrower tiles still fit in ONE wave, take them -- more CTAs share the work and each CTA's
    // serial tail (TMEM drain + stores, ~0.45 us per 64-column box per warp) shrinks with the tile; operand re-use per
    // byte is worse but nothing is bandwidth-bound at this size (1024^3: 13 us with 256 x 256 pair tiles on 32 CTAs).
    // Clusters of 4 CTAs cannot use every SM: cudaOccupancyMaxActiveClusters reports 33 of them (132 SMs) on B200 with
    // this kernel's shared memory (74 clusters of 2 = all 148 SMs; 15 of 8) -- GPC sizes are not multiples of 4.  One-wave
    // cluster plans are held to that count, scaled by the SM budget.  (It is also why the big-tile GEMM does not share
    // its Y tile between two pairs by TMA multicast: 11 % of the SMs would idle.)
    const int max_clusters4 = 33 * budget / sm_count;
    bool one_wave = false;
    if (!swap && occ.cta_group != 2 && occ.m_blocks != 2 && occ.tiles_per_cta == 0 && occ.cluster_k < 2) {
        const long long tx1 = (RX + kBM - 1) / kBM;
        // the alternative for mid-size problems with a long K: 256 x 256 pair tiles with the K range split over two
        // pairs of a 4-CTA cluster (half the L2->SM bytes per flop of a narrow single-CTA tile).  Cycle estimates per
        // CTA: narrow tile kb * (128 + bn) * 2 (load-bound), split pair tile kb/2 * 512 + ~4k for the hand-over.
        long long pair_ks_cost = -1;
        if (bn == 256 && RX >= 2 * kBM && occ.cta_group != 1 && occ.cluster_k != 1 && kb >= 16) {
            const long long T = (long long)((RX + 2 * kBM - 1) / (2 * kBM)) * ((RY + 255) / 256);
            const int pairs = budget / 2;
            if (2 * T <= pairs && 4 * T >= pairs && T <= max_clusters4) pair_ks_cost = (long long)(kb / 2) * 512 + 4096;
        }
        for (int cand = 64; cand < bn; cand <<= 1) {
            if (tx1 * ((RY + cand - 1) / cand) <= budget) {
                if (pair_ks_cost >= 0 && pair_ks_cost < (long long)kb * (kBM + cand) * 2) break;   // split pair tiles win
                bn = cand;
                one_wave = true;
                break;
            }
        }
    }
    if (occ.cta_group < 0 || occ.cta_group > 2) return RA_ERR_INVALID_ARG;
    if (occ.m_blocks < 0 || occ.m_blocks > 2) return RA_ERR_INVALID_ARG;
    if (occ.cluster_k < 0 || occ.cluster_k > 4 || occ.cluster_k == 3) return RA_ERR_INVALID_ARG;
    if (occ.l2_persist_bytes < 0) return RA_ERR_INVALID_ARG;
    if (occ.tile_order < 0 || occ.tile_order > 1) return RA_ERR_INVALID_ARG;

    // n_acc = GEMM CTAs per SM the shared-memory accounting assumes.  Pass 1 sizes the plan for ONE CTA per SM and makes
    // that a fact where it can (padding, below).  Where it cannot -- a reserve above ~half an SM leaves no room for the
    // padding -- the block scheduler DOES place two of the persistent grid's CTAs on one SM when collective CTAs crowd
    // the others (measured: tests/test_overlap_gpu.py, reserve 160 KiB x budget 74 next to the allreduce), so pass 2
    // sizes every CTA for the reserve to hold with TWO resident:  2 * (dyn + reserved) <= smem_per_sm - reserve.
    const int bn_start = bn;
    const int clamped_start = clamped;
    for (int n_acc = 1;; ++n_acc) {
    bn = bn_start;
    clamped = clamped_start;
    // shared memory the GEMM may allocate on an SM
    long avail = ((long)smem_per_sm - occ.smem_reserve_bytes) / n_acc - reserved;
    if (avail > optin) avail = optin;
    // non-swapped C leaves through a 32 KiB staging area + TMA stores (full-line writes); the skinny path keeps
    // direct stores (its C is tiny) and spends the space on pipeline depth
    // (nor does a GEMM squeezed below ~128 KiB by the reserve: there pipeline depth matters more)
    int epi_bytes = (!swap && avail - kAlignSlack - kBarrierBytes - kEpiStageBytes >= 96 * 1024) ? kEpiStageBytes : 0;
    long room = avail - kAlignSlack - kBarrierBytes - epi_bytes;
    auto stages_for = [&](int bn_, int cg_, int xh_) {
        int s = room > 0 ? (int)(room / stage_bytes(bn_, cg_, xh_)) : 0;
        return s > kMaxStages ? kMaxStages : s;
    };
    auto wave_eff = [](long long tiles, int workers) {
        const long long waves = (tiles + workers - 1) / workers;
        return waves > 0 ? (double)tiles / (double)(waves * workers) : 1.0;
    };

    // CTA pairs (cta_group::2, 256 x 256 tiles): each SM stages 128 rows of X and 128 of Y per k-block instead of
    // 128 + 256, i.e. 1/3 less L2->SM traffic per flop.  Used for the data-parallel schedule on large problems.
    int cg = 1;
    if (occ.cta_group != 1 && !swap && bn == 256 && RX >= 256 && budget >= 2 && stages_for(256, 2, 1) >= 2) {
        // measured on B200: pair tiles beat single-CTA stream-K even at low wave efficiency (1024^3: 13 vs 27 us at
        // 22 %, 3000x1000x2048: 19 vs 37 us at 65 %, 256x8192x8192: 54 vs 73 us at 43 %) -- half the L2->SM traffic
        // per flop and no partial-tile round trip -- so pairs are taken whenever the shape allows them.
        cg = 2;
    }
    if (occ.cta_group == 2 && cg != 2) {
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        clamped = 1;
    }

    // Big tiles (two 128-row X blocks per CTA sharing one Y stage; a pair covers 512 x 256): 48 B/clk/SM of
    // operand traffic instead of 64, which is the L2->SM limit the 256 x 256 pair tile runs into (the tensor pipe
    // was 85-88 % busy; cuBLAS's 256x256-per-CTA kernel 96 %).  Needs >= 3 stages of 48 KiB and enough tiles that
    // the coarser wave quantisation does not eat the gain.
    int xh = 1;
    if (cg == 2 && occ.m_blocks != 1 && RX >= 4 * kBM && stages_for(256, 2, 2) < 3 &&
        epi_bytes > 0 && room + epi_bytes >= 3 * stage_bytes(256, 2, 2)) {
        // three 48 KiB stages fit only without the store staging: operand traffic matters more than store width
        room += epi_bytes;
        epi_bytes = 0;
    }
    if (cg == 2 && occ.m_blocks != 1 && RX >= 4 * kBM && stages_for(256, 2, 2) >= 3) {
        const long long t1 = (long long)((RX + 2 * kBM - 1) / (2 * kBM)) * ((RY + bn - 1) / bn);
        const long long t2 = (long long)((RX + 4 * kBM - 1) / (4 * kBM)) * ((RY + bn - 1) / bn);
        const double e1 = wave_eff(t1, budget / 2) * 0.88, e2 = wave_eff(t2, budget / 2) * 0.96;
        if (e2 >= e1 || occ.m_blocks == 2) xh = 2;
    }
    if (occ.m_blocks == 2 && xh != 2) {
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        clamped = 1;
    }

    int stages = 0;
    for (;;) {
        stages = stages_for(bn, cg, xh);
        if (stages >= 2 || bn == 64) break;
        bn >>= 1;   // squeeze the tile before giving up pipelining
    }
    if (stages < 1) {
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        stages = 1;
        clamped = 1;
    }
    int dyn = stages * stage_bytes(bn, cg, xh) + kAlignSlack + kBarrierBytes + epi_bytes;

    const int tile_x = kBM * cg * xh;
    const int tiles_x = (RX + tile_x - 1) / tile_x, tiles_y = (RY + bn - 1) / bn;
    const long long n_tiles = (long long)tiles_x * tiles_y;
    if (n_tiles > 0x3fffffffLL) return RA_ERR_UNSUPPORTED;

    int grid, stream_k = 0, ctas_per_sm = n_acc, ks = 1;
    // Residency (A22 / A23): the plan's accounting -- smem_left_per_sm >= reserve -- assumes ONE GEMM CTA per SM.  That is
    // guaranteed by the footprint itself when a second CTA cannot fit: the request is padded past half of an SM's
    // shared memory whenever the hardware (resident_ctas(): registers, threads, shared memory -- NOT the occupancy API, see there) would otherwise admit two
    // and the padding still honours the reserve -- the paper's direction: more shared memory per block, fewer
    // resident blocks.
    const int half = (smem_per_sm - 2 * reserved) / 2 + 16;
    int hw = resident_ctas(dev, bn, cg, xh, dyn, smem_per_sm, reserved);
    if (n_acc == 1 && hw > 1 && dyn < half && half <= avail) {
        dyn = half;
        hw = resident_ctas(dev, bn, cg, xh, dyn, smem_per_sm, reserved);
    }
    if (n_acc == 1 && hw > 1 && occ.tiles_per_cta == 0) {
        // two CTAs fit and padding would break the reserve: account for two -- if a two-resident plan exists at all
        // (at least one stage of the narrowest tile, and two CTAs' accumulators in the 512 TMEM columns)
        const long avail2 = ((long)smem_per_sm - occ.smem_reserve_bytes) / 2 - reserved;
        if (avail2 - kAlignSlack - kBarrierBytes >= stage_bytes(64, 1, 1)) continue;
        // not even that fits (reserve ~200 KiB): nothing honours the knob -> clamp: keep the one-CTA sizing and
        // report the shared memory an SM really has left in the worst case (two resident)
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        clamped = 1;
        ctas_per_sm = hw;
    }
    if (n_acc == 2 && 2 * bn * hw > 512) {       // two residents' accumulators must both fit in TMEM
        if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
        clamped = 1;
    }
    if (occ.tiles_per_cta > 0) {
        // bounded work: more CTAs than SMs, so a second CTA WILL be placed wherever it fits (it would only wait for
        // TMEM): single residency is mandatory here, at the price of the reserve if need be (clamped).
        grid = cg * (int)((n_tiles + occ.tiles_per_cta - 1) / occ.tiles_per_cta);
        if (occ.cluster_k >= 2) {                 // cluster split-K is a one-tile-per-cluster schedule
            if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
            clamped = 1;
        }
        if (hw > 1 && dyn < half) {
            if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;   // half > avail: reserve and single residency conflict
            clamped = 1;
            dyn = half;
            hw = resident_ctas(dev, bn, cg, xh, dyn, smem_per_sm, reserved);
        }
    } else {
        const int workers = budget / cg;                 // CTAs, or CTA pairs
        int w = (int)(n_tiles < workers ? n_tiles : workers);
        if (w < 1) w = 1;
        // wave-quantisation efficiency of the data-parallel schedule.  Several waves with a ragged last one
        // (< 90 %): cut the k-block units evenly instead (stream-K, single-CTA tiles only).  A single partial
        // wave (MB: 128 tiles on 148 SMs = 86 %) stays data-parallel down to 80 %: one tile per CTA and no
        // partials measured 4 % faster than stream-K on all 148 SMs, since 128 SMs already saturate HBM.
        const long long U = n_tiles * kb;
        const double eff = wave_eff(n_tiles, workers);
        // Cluster split-K: when two CTAs per tile still fit in one wave, a 2-CTA cluster splits the tile's k-blocks
        // and hands one accumulator over through distributed shared memory -- twice the CTAs streaming operands and
        // no global-memory partials, counters or memset.  Taken when it fills at least half of the budgeted SMs (below
        // that stream-K's finer split wins) and the receiving stage ring can hold a 128 x BN fp32 accumulator.
        const long ring = (long)stages * stage_bytes(bn, cg, 1), slot = (long)kBM * bn * 4;
        // 4-CTA clusters (four single-CTA parts, or two CTA pairs) must also fit the chip's cluster capacity
        const bool ks2_fits = bk == kBK && xh == 1 && n_tiles > 0 && 2 * n_tiles <= workers && kb >= 2 && ring >= slot &&
                              (cg == 1 || n_tiles <= max_clusters4);
        const bool ks4_fits = bk == kBK && xh == 1 && cg == 1 && n_tiles > 0 && 4 * n_tiles <= workers && kb >= 4 && ring >= 3 * slot &&
                              n_tiles <= max_clusters4;
        if (ks4_fits && occ.cluster_k != 1 && occ.cluster_k != 2 && (kb >= 32 || occ.cluster_k == 4)) {
            ks = 4;                                   // four single-CTA parts per tile, three slots in part 0's ring
            w = (int)(4 * n_tiles);
        } else if (ks2_fits && occ.cluster_k != 1 && occ.cluster_k != 4 && (kb >= 16 || occ.cluster_k == 2)) {
            ks = 2;
            w = (int)(2 * n_tiles);                   // workers: CTAs, or CTA pairs (4-CTA clusters)
        } else if (occ.cluster_k >= 2) {
            if (!occ.allow_clamp) return RA_ERR_INFEASIBLE_KNOB;
            clamped = 1;
        }
        if (ks == 1 && cg == 1 && !one_wave && n_tiles > 0 && kb >= 8 && eff < (n_tiles <= workers ? 0.8 : 0.9)) {
            stream_k = 1;
            w = workers;
            if ((long long)w * 4 > U) w = (int)(U / 4);   // at least 4 k-blocks per CTA
        }
        grid = w * cg;
    }
    g.ctas_per_sm = ctas_per_sm;
    g.hw_ctas_per_sm = hw;
    g.grid = grid;
    g.stages = stages;
    g.tile_m = swap ? bn : tile_x;
    g.tile_n = swap ? kBM : bn;
    g.tile_k = bk;
    g.swap_ab = swap;
    g.dyn_smem_bytes = dyn;
    g.smem_left_per_sm = smem_per_sm - ctas_per_sm * (dyn + reserved);
    g.n_tiles = (int)n_tiles;
    g.clamped = clamped;
    g.split_k = 1;
    g.cta_group = cg;
    g.m_blocks = xh;
    g.cluster_k = ks;
    pl.bn = bn;
    pl.epi_tma = epi_bytes > 0;
    {
        // Rasterisation.  The W workers of one wave cover a gx x gy block of tiles and march through K together, so
        // the wave reads (gx*tile_x + gy*BN) rows of K from DRAM once and shares them through L2 in time.  Nothing
        // survives from one wave to the next under the default L2 policy once a wave's footprint passes ~50 MB
        // (measured, profiles/r02_l2_persist.md: 8192^3 reads waves x footprint), so DRAM traffic ~ waves *
        // (gx*tile_x + gy*BN) rows, minimised subject to gx*gy = W at gx = sqrt(W*BN/tile_x): 6 for 74 pairs of 512 x 256.
        const int workers = grid / (cg * ks);
        int gx = 1;
        while ((long long)(gx + 1) * (gx + 1) * tile_x <= (long long)workers * bn) ++gx;
        pl.hint_x = 0;
        g.l2_persist_bytes = 0;
        // l2_persist_bytes: the X panel of a group (gx*tile_x rows x K) is loaded with the evict_last policy and stays in
        // the persisting carve-out of L2 while the group's Y tiles stream past it, so X is read from DRAM once and Y once
        // per group.  The group is widened to what the carve-out holds; a carve-out smaller than the default group's
        // panel still keeps part of it.
        const long long xtile_bytes = (long long)tile_x * K * 2;
        if (occ.l2_persist_bytes > 0 && !swap && !stream_k && ks == 1 && tiles_x * tiles_y > workers && xtile_bytes > 0) {
            // what can actually persist: the request clamped to the device's maximum carve-out (the raster group is sized
            // from this, and the plan reports it, so a 1 GiB request does not widen the group past what L2 can hold)
            const long long l2_bytes = occ.l2_persist_bytes < max_persisting_l2() ? occ.l2_persist_bytes : max_persisting_l2();
            const int fit = (int)(l2_bytes / xtile_bytes);
            if (fit > gx) {
                gx = fit < tiles_x ? fit : tiles_x;
                const int groups = (tiles_x + gx - 1) / gx;
                gx = (tiles_x + groups - 1) / groups;         // equal groups: 16 tile rows at 9 that fit -> 8 + 8, not 9 + 7
            }
            pl.hint_x = 2;
            g.l2_persist_bytes = (int32_t)l2_bytes;
        }
        if (gx > tiles_x) gx = (int)tiles_x;
        g.group_x = gx < 1 ? 1 : gx;
    }
    if (stream_k) {
        const long long U = n_tiles * kb;
        // max number of CTA ranges one tile can span
        const long long per = U / grid;   // >= 4
        g.split_k = (int)((kb + per - 1) / per + 1);
        pl.counters_bytes = (((size_t)n_tiles * sizeof(int)) + 1023) & ~(size_t)1023;
        pl.ws_bytes = pl.counters_bytes + (size_t)2 * grid * kBM * bn * sizeof(float);
    }
    break;
    }   // n_acc
    *out = pl;
    return RA_OK;
}

template <int BN, int CG, int XH, int KBK, bool DYN>
static ra_status launch_gemm(const CUtensorMap& mx, const CUtensorMap& my, const CUtensorMap& mc, const GemmParams& p, int grid, int dyn,
                             cudaStream_t stream) {
    const int cluster = CG * p.ks;                      // CTA pair (tcgen05 cta_group::2) x split-K halves
    if (cluster == 1) {
        gemm_kernel<BN, CG, XH, KBK, DYN><<<grid, kGemmThreads, dyn, stream>>>(mx, my, mc, p, g_trace);
        RA_CUDA(cudaGetLastError());
        return RA_OK;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = (size_t)dyn;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    RA_CUDA(cudaLaunchKernelEx(&cfg, gemm_kernel<BN, CG, XH, KBK, DYN>, mx, my, mc, p, g_trace));
    return RA_OK;
}

// ---- host: launch cache -------------------------------------------------------------------------------------------
// Everything a launch needs besides (alpha, beta, workspace, stream) is a pure function of (device, shape, leading
// dimensions, operand addresses, output type, knobs): the plan, the kernel parameters and the two or three CUtensorMaps
// (encoding one costs a driver call).  Entries are kept in a small LRU list behind a mutex ("lazily-cached
// ... tensor-map descriptors", Appendix A: "cache them by (ptr, dims, ld, box)").
struct LaunchKey {
    int32_t device, transA, transB, M, N, K, lda, ldb, ldc, c_f32;
    const void *A, *B, *C;
    ra_occupancy occ;
};
struct LaunchEntry {
    LaunchKey key;
    Plan pl;
    GemmParams p;          // alpha, beta, partials, counters are filled per call
    CUtensorMap mx, my, mc;
    uint64_t stamp;
};
constexpr size_t kLaunchCacheEntries = 32;
static std::mutex g_launch_mu;
static std::vector<LaunchEntry> g_launch_cache;
static uint64_t g_launch_stamp = 0;

static void dyn_slots_clear();
void gemm_cache_clear() {
    {
        std::lock_guard<std::mutex> lk(g_launch_mu);
        g_launch_cache.clear();
    }
    dyn_slots_clear();     // ra_shutdown: the caller has no launch in flight any more
}

// Builds plan, parameters and tensor maps for one key (the slow path of a launch).
static ra_status build_entry(const LaunchKey& k, const DeviceInfo& di, LaunchEntry* e) {
    const int transA = k.transA, transB = k.transB, M = k.M, N = k.N, K = k.K;
    e->key = k;
    Plan& pl = e->pl;
    RA_TRY(make_plan(transA, transB, M, N, K, &k.occ, &pl));
    const int swap = pl.pub.swap_ab;
    GemmParams p{};
    p.RX = swap ? N : M;
    p.RY = swap ? M : N;
    p.K = K;
    const int cg = pl.pub.cta_group, xh = pl.pub.m_blocks;
    const int tile_x = kBM * cg * xh;
    p.tiles_x = (p.RX + tile_x - 1) / tile_x;
    p.tiles_y = (p.RY + pl.bn - 1) / pl.bn;
    p.n_tiles = pl.pub.n_tiles;
    p.bk = pl.pub.tile_k;
    p.kb_per_tile = (K + p.bk - 1) / p.bk;
    p.swap = swap;
    p.stream_k = pl.pub.split_k > 1;
    p.stages = pl.pub.stages;
    p.C = static_cast<__nv_bfloat16*>(const_cast<void*>(k.C));
    p.ldc = k.ldc;
    // L2 policy: an operand that is streamed exactly once (one tile along the other dimension) should
    // not displace anything; the small operand every CTA re-reads should stay.
    p.hintX = (p.tiles_y == 1 && p.tiles_x > 1) ? 1 : 0;
    p.hintY = (p.tiles_y == 1 && p.tiles_x > 1) ? 2 : 0;
    p.group_x = pl.pub.group_x;
    if (pl.hint_x) p.hintX = pl.hint_x;
    {
        // dynamic tile order: persistent data-parallel plans with more tiles than workers (see g_dyn)
        const int workers = pl.pub.grid / (cg * pl.pub.cluster_k);
        p.dyn = (cg == 2 && k.occ.tile_order != 1 && !p.stream_k && pl.pub.cluster_k == 1 && k.occ.tiles_per_cta == 0 && p.n_tiles > workers &&
                 workers <= kDynWorkers && p.n_tiles < kDynMaxSteps) ? 1 : 0;
    }
    const void* X = swap ? k.B : k.A;
    const void* Y = swap ? k.A : k.B;
    const int ldx = swap ? k.ldb : k.lda, ldy = swap ? k.lda : k.ldb;
    // op(A)(i,k): K-contiguous iff transA == 0;  op(B)(k,j): K-contiguous iff transB == 1
    const int a_mn = transA ? 1 : 0, b_mn = transB ? 0 : 1;
    p.xmn = swap ? b_mn : a_mn;
    p.ymn = swap ? a_mn : b_mn;
    RA_TRY(make_map(&e->mx, X, p.RX, K, ldx, kBM * xh, p.xmn, p.bk));
    RA_TRY(make_map(&e->my, Y, p.RY, K, ldy, pl.bn / cg, p.ymn, p.bk));
    p.c_f32 = k.c_f32;
    p.epi_tma = k.c_f32 ? 0 : pl.epi_tma;      // fp32 rows are written directly: 128 contiguous bytes per thread and chunk
    p.ks = pl.pub.cluster_k;
    p.skew = pl.pub.stages;   // measured on 8192^3 (4 stages): drain wait per tile 5.9k cycles at skew 0, 1.5k at 4
    if (p.epi_tma) RA_TRY(make_map(&e->mc, k.C, M, N, k.ldc, 32, 0));    // C: box = 64 columns x 32 rows (one epilogue warp)
    else e->mc = e->mx;                                                  // unused
    e->p = p;
    {
        std::lock_guard<std::mutex> lk(g_gemm_mu);
        RA_TRY(prepare_kernel(di, pl.bn, cg, xh, p.bk, p.dyn));
        if (p.dyn) RA_TRY(prepare_kernel(di, pl.bn, cg, xh, p.bk, 0));   // the static twin: taken when no launch slot is free
    }
    return RA_OK;
}

// ---- dynamic tile order: one g_dyn slot per launch IN FLIGHT ---------------------------------------------------------
// A slot (claim counter, exit counter, generation, ring) belongs to ONE running kernel: two kernels drawing from one claim
// counter would each skip the tiles the other claimed.  Launches are asynchronous, so "who still uses slot i" is answered by
// an event recorded behind every dynamic-order launch: a slot is handed out only if it was never used or its last launch
// has completed (cudaEventQuery), whatever stream, host thread or cache entry that launch came from.  When all kDynSlots are
// in flight, or the stream is being captured (a graph would keep the slot's address for as long as it lives), or the
// caller may not create an event (ra_gemm_static_ws), the launch takes the STATIC-order instantiation of the same plan --
// same tiles, same per-element k order, same bits (tests), a few per cent slower on multi-wave shapes.
struct DynSlot {
    cudaEvent_t done = nullptr;   // recorded behind the last launch that used the slot
    int device = -1;              // the device `done` was created on
    int state = 0;                // 0 = free, 1 = claimed (its launch is being enqueued), 2 = in flight until `done` completes
};
static DynSlot g_dyn_slot[kDynSlots];
static int g_dyn_cursor = 0;
static std::mutex g_dyn_mu;
static thread_local bool t_no_new_events = false;

static int dyn_slot_acquire(int device) {
    std::lock_guard<std::mutex> lk(g_dyn_mu);
    for (int n = 0; n < kDynSlots; ++n) {
        const int i = (g_dyn_cursor + n) % kDynSlots;
        DynSlot& sl = g_dyn_slot[i];
        if (sl.state == 1) continue;
        if (sl.state == 2) {
            if (cudaEventQuery(sl.done) != cudaSuccess) {
                (void)cudaGetLastError();          // cudaErrorNotReady (still running) or a dead context: not ours to take
                continue;
            }
            sl.state = 0;
        }
        if (sl.done != nullptr && sl.device != device) {   // an event records only on streams of its own device
            if (t_no_new_events) continue;
            (void)cudaEventDestroy(sl.done);
            sl.done = nullptr;
        }
        if (sl.done == nullptr) {
            if (t_no_new_events) continue;
            if (cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming) != cudaSuccess) {
                (void)cudaGetLastError();
                sl.done = nullptr;
                return -1;
            }
            sl.device = device;
        }
        sl.state = 1;
        g_dyn_cursor = (i + 1) % kDynSlots;
        return i;
    }
    return -1;
}

// After the launch: launched = the kernel was enqueued on `stream`.
static void dyn_slot_release(int i, bool launched, cudaStream_t stream) {
    std::lock_guard<std::mutex> lk(g_dyn_mu);
    DynSlot& sl = g_dyn_slot[i];
    if (launched && cudaEventRecord(sl.done, stream) == cudaSuccess) {
        sl.state = 2;
        return;
    }
    (void)cudaGetLastError();
    // No way to tell when that kernel ends: wait for it here rather than hand its slot to somebody else.
    if (launched) (void)cudaStreamSynchronize(stream);
    sl.state = 0;
}

static void dyn_slots_clear() {
    std::lock_guard<std::mutex> lk(g_dyn_mu);
    for (DynSlot& sl : g_dyn_slot) {
        if (sl.done != nullptr) (void)cudaEventDestroy(sl.done);
        sl = DynSlot{};
    }
    (void)cudaGetLastError();
}

ra_status gemm_launch(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                      int ldb, float beta, void* C, int ldc, const ra_occupancy* occ, void* workspace,
                      size_t workspace_bytes, cudaStream_t stream, ra_gemm_plan* plan_out, int c_f32) {
    RA_TRY(validate_shape(transA, transB, M, N, K));
    if (c_f32 != 0 && c_f32 != 1) return RA_ERR_INVALID_ARG;
    if (M == 0 || N == 0) return RA_OK;
    if (A == nullptr || B == nullptr || C == nullptr) return RA_ERR_INVALID_ARG;
    const int min_lda = transA ? M : K, min_ldb = transB ? K : N;
    if (lda < (min_lda > 1 ? min_lda : 1) || ldb < (min_ldb > 1 ? min_ldb : 1) || ldc < N) return RA_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(A) & 15u) || (reinterpret_cast<uintptr_t>(B) & 15u) ||
        (reinterpret_cast<uintptr_t>(C) & 15u))
        return RA_ERR_INVALID_ARG;
    if ((lda % 8) || (ldb % 8) || (ldc % (c_f32 ? 4 : 8))) return RA_ERR_UNSUPPORTED;   // 16-byte row pitches
    {
        // C must not overlap A or B
        const uintptr_t c0 = reinterpret_cast<uintptr_t>(C), c1 = c0 + ((size_t)(M - 1) * ldc + N) * (c_f32 ? 4 : 2);
        const size_t a_elems = transA ? ((size_t)(K > 0 ? K - 1 : 0) * lda + M) : ((size_t)(M - 1) * lda + K);
        const size_t b_elems = transB ? ((size_t)(N - 1) * ldb + K) : ((size_t)(K > 0 ? K - 1 : 0) * ldb + N);
        const uintptr_t a0 = reinterpret_cast<uintptr_t>(A), a1 = a0 + a_elems * 2;
        const uintptr_t b0 = reinterpret_cast<uintptr_t>(B), b1 = b0 + b_elems * 2;
        if (K > 0 && ((c0 < a1 && a0 < c1) || (c0 < b1 && b0 < c1))) return RA_ERR_INVALID_ARG;
    }
    ra_occupancy occ_v = {0, 0, 0, 1, 0, 0, 0, 0, 0, 0};
    if (occ) occ_v = *occ;

    if (K == 0 || alpha == 0.f) {
        Plan pl;
        RA_TRY(make_plan(transA, transB, M, N, K, &occ_v, &pl));      // knob errors are reported as for any other launch
        DeviceInfo di;
        RA_TRY(device_info(&di));
        RA_TRY(require_sm100(di));
        if (plan_out) *plan_out = pl.pub;
        const size_t total = (size_t)M * N;
        const int blocks = (int)((total + 255) / 256 < (size_t)di.sm_count * 8 ? (total + 255) / 256 : (size_t)di.sm_count * 8);
        scale_c_kernel<<<blocks, 256, 0, stream>>>(C, M, N, ldc, beta, c_f32);
        RA_CUDA(cudaGetLastError());
        return RA_OK;
    }

    LaunchKey key;
    memset(&key, 0, sizeof(key));                  // padding bytes too: keys are compared with memcmp
    key.transA = transA; key.transB = transB; key.M = M; key.N = N; key.K = K;
    key.lda = lda; key.ldb = ldb; key.ldc = ldc; key.c_f32 = c_f32;
    key.A = A; key.B = B; key.C = C;
    key.occ = occ_v;
    RA_CUDA(cudaGetDevice(&key.device));

    Plan pl;
    GemmParams p;
    CUtensorMap mx, my, mc;
    bool hit = false;
    {
        std::lock_guard<std::mutex> lk(g_launch_mu);
        for (size_t i = 0; i < g_launch_cache.size(); ++i) {
            LaunchEntry& e = g_launch_cache[i];
            if (memcmp(&e.key, &key, sizeof(key)) == 0) {
                e.stamp = ++g_launch_stamp;
                pl = e.pl; p = e.p; mx = e.mx; my = e.my; mc = e.mc;
                hit = true;
                break;
            }
        }
    }
    if (!hit) {
        DeviceInfo di;
        RA_TRY(device_info(&di));
        RA_TRY(require_sm100(di));
        LaunchEntry e;
        RA_TRY(build_entry(key, di, &e));
        pl = e.pl; p = e.p; mx = e.mx; my = e.my; mc = e.mc;
        std::lock_guard<std::mutex> lk(g_launch_mu);
        e.stamp = ++g_launch_stamp;
        if (g_launch_cache.size() < kLaunchCacheEntries) {
            g_launch_cache.push_back(e);
        } else {
            size_t lru = 0;
            for (size_t i = 1; i < g_launch_cache.size(); ++i)
                if (g_launch_cache[i].stamp < g_launch_cache[lru].stamp) lru = i;
            g_launch_cache[lru] = e;
        }
    }
    if (pl.ws_bytes > 0) {
        if (workspace == nullptr || workspace_bytes < pl.ws_bytes || (reinterpret_cast<uintptr_t>(workspace) & 15u))
            return RA_ERR_INVALID_ARG;
    }
    if (plan_out) *plan_out = pl.pub;
    // the carve-out the PLAN uses (0 when it ignores the knob); no driver call unless it has to change, none under capture
    RA_TRY(l2_persist_ensure_on(pl.pub.l2_persist_bytes, stream));
    p.alpha = alpha;
    p.beta = beta;
    int dyn_slot = -1;
    if (p.dyn) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) (void)cudaGetLastError();
        else if (cs == cudaStreamCaptureStatusNone) dyn_slot = dyn_slot_acquire(key.device);
        if (dyn_slot < 0) p.dyn = 0;               // no slot to be had: the static order of the same plan
    }
    if (p.dyn) {
        static void* g_dyn_base[64] = {};          // per device: the symbol's address never changes
        void* base = (key.device >= 0 && key.device < 64) ? g_dyn_base[key.device] : nullptr;
        if (base == nullptr) {
            const cudaError_t e = cudaGetSymbolAddress(&base, g_dyn);
            if (e != cudaSuccess) {
                dyn_slot_release(dyn_slot, false, stream);
                RA_CUDA(e);
            }
            if (key.device >= 0 && key.device < 64) g_dyn_base[key.device] = base;
        }
        unsigned long long* slot = static_cast<unsigned long long*>(base) + (size_t)dyn_slot * kDynSlotWords;
        p.dyn_ring = slot;
        p.dyn_ctr = reinterpret_cast<unsigned int*>(slot + kDynWorkers * kDynRing);
    }
    if (p.stream_k) {
        p.counters = static_cast<int*>(workspace);
        p.partials = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + pl.counters_bytes);
        RA_CUDA(cudaMemsetAsync(workspace, 0, pl.counters_bytes, stream));
    }
    const int cg = pl.pub.cta_group, xh = pl.pub.m_blocks;
    ra_status st = RA_ERR_UNSUPPORTED;
#define RA_LAUNCH(BN_, CG_, XH_, DYN_)                                                                                        \
    st = p.bk == 32 ? launch_gemm<BN_, CG_, XH_, 32, DYN_>(mx, my, mc, p, pl.pub.grid, pl.pub.dyn_smem_bytes, stream)           \
                    : launch_gemm<BN_, CG_, XH_, 64, DYN_>(mx, my, mc, p, pl.pub.grid, pl.pub.dyn_smem_bytes, stream)
    if (cg == 2 && xh == 2) {
        if (p.dyn) RA_LAUNCH(256, 2, 2, true);
        else RA_LAUNCH(256, 2, 2, false);
    } else if (cg == 2) {
        if (p.dyn) RA_LAUNCH(256, 2, 1, true);
        else RA_LAUNCH(256, 2, 1, false);
    } else {
        switch (pl.bn) {
            case 64: RA_LAUNCH(64, 1, 1, false); break;
            case 128: RA_LAUNCH(128, 1, 1, false); break;
            case 256: RA_LAUNCH(256, 1, 1, false); break;
        }
    }
#undef RA_LAUNCH
    if (dyn_slot >= 0) dyn_slot_release(dyn_slot, st == RA_OK, stream);
    return st;
}

}  // namespace ra

extern "C" {

ra_status ra_gemm_plan_query(int transA, int transB, int M, int N, int K, const ra_occupancy* occ, ra_gemm_plan* out) {
    if (out == nullptr) return RA_ERR_INVALID_ARG;
    ra::Plan pl;
    RA_TRY(ra::make_plan(transA, transB, M, N, K, occ, &pl));
    *out = pl.pub;
    return RA_OK;
}

ra_status ra_gemm_residency(int32_t* max_ctas_on_one_sm, int reset) {
    ra::DeviceInfo di;
    RA_TRY(ra::device_info(&di));
    RA_TRY(ra::require_sm100(di));
    RA_CUDA(cudaDeviceSynchronize());
    int v = 0;
    RA_CUDA(cudaMemcpyFromSymbol(&v, ra::g_gemm_max_resident, sizeof(int)));
    if (max_ctas_on_one_sm) *max_ctas_on_one_sm = v;
    if (reset) {
        const int zero = 0;
        RA_CUDA(cudaMemcpyToSymbol(ra::g_gemm_max_resident, &zero, sizeof(int)));
        static const int zeros[1024] = {};
        RA_CUDA(cudaMemcpyToSymbol(ra::g_gemm_resident, zeros, sizeof(zeros)));
    }
    return RA_OK;
}

size_t ra_gemm_workspace_bytes(int transA, int transB, int M, int N, int K, const ra_occupancy* occ) {
    ra::Plan pl;
    if (ra::make_plan(transA, transB, M, N, K, occ, &pl) != RA_OK) return 0;
    return pl.ws_bytes;
}

ra_status ra_gemm(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                  int ldb, float beta, void* C, int ldc, const ra_occupancy* occ, void* workspace,
                  size_t workspace_bytes, void* stream) {
    return ra::gemm_launch(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, occ, workspace,
                           workspace_bytes, static_cast<cudaStream_t>(stream), nullptr, 0);
}

ra_status ra_gemm_ex(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                     int ldb, float beta, void* C, int ldc, int c_dtype, const ra_occupancy* occ, void* workspace,
                     size_t workspace_bytes, void* stream) {
    if (c_dtype != RA_DTYPE_BF16 && c_dtype != RA_DTYPE_F32) return RA_ERR_INVALID_ARG;
    return ra::gemm_launch(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, occ, workspace,
                           workspace_bytes, static_cast<cudaStream_t>(stream), nullptr, c_dtype == RA_DTYPE_F32 ? 1 : 0);
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// ra_gemm_static_ws: the stream-K scratch lives in the library image instead of in a caller allocation (include/ra.h
// says who needs that and why).  The array is named only here: in host code `g_static_ws` is the host-side shadow of the
// symbol, NOT a device address -- handing it to a kernel or to cudaMemsetAsync would fault (or, on a machine whose GPU can
// reach host memory, quietly scribble over the wrong bytes) -- so the address every launch uses comes from
// cudaGetSymbolAddress, asked once per device with that device current.
// ---------------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_ws[RA_GEMM_STATIC_WS_BYTES];

namespace ra {
namespace {
constexpr int kStaticWsDevices = 64;
std::mutex g_static_ws_mu;
void* g_static_ws_addr[kStaticWsDevices] = {};   // per device ordinal: where that device's copy of the array lives

// Device address of g_static_ws on the CURRENT device.  Set-up (first call per device): one cudaGetSymbolAddress.
ra_status static_ws_address(void** out) {
    int dev = -1;
    RA_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticWsDevices) return RA_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_static_ws_mu);
    if (g_static_ws_addr[dev] == nullptr) {
        void* ptr = nullptr;
        RA_CUDA(cudaGetSymbolAddress((void**)&ptr, g_static_ws));
        if (ptr == nullptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) return RA_ERR_CUDA;
        g_static_ws_addr[dev] = ptr;
    }
    *out = g_static_ws_addr[dev];
    return RA_OK;
}
}  // namespace
}  // namespace ra

extern "C" ra_status ra_gemm_static_ws(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda,
                                       const void* B, int ldb, float beta, void* C, int ldc, const ra_occupancy* occ,
                                       void* stream) {
    // How much scratch would this launch take?  Host-only planning; a plan that cannot be made (bad shape, infeasible
    // knob) is left for gemm_launch to report with its usual code.
    ra::Plan pl;
    const bool planned = ra::make_plan(transA, transB, M, N, K, occ, &pl) == RA_OK;
    if (planned && pl.ws_bytes > RA_GEMM_STATIC_WS_BYTES) return RA_ERR_SCRATCH_LIMIT;
    void* ws = nullptr;
    if (planned && pl.ws_bytes > 0) RA_TRY(ra::static_ws_address(&ws));
    // From here on this is ra_gemm: gemm_launch zeroes the tile counters at the head of the workspace on `stream` before
    // the kernel (cudaMemsetAsync) and never reads a partial sum it has not written in the same launch.
    // Dynamic-order plans need an event per launch slot; this path creates none (it reuses slots whose event a plain ra_gemm
    // call made earlier, else it runs the static tile order: same bits).
    ra::t_no_new_events = true;
    const ra_status st = ra::gemm_launch(transA, transB, M, N, K, alpha, A, lda, B, ldb, beta, C, ldc, occ, ws,
                                         ws ? RA_GEMM_STATIC_WS_BYTES : 0, static_cast<cudaStream_t>(stream), nullptr, 0);
    ra::t_no_new_events = false;
    return st;
}
