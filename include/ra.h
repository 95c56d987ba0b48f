/*
 * ra.h -- C ABI of libra.so: the resource-aware GEMM + collective overlap hot path of
 * arxiv/paper_2606_09200 ("Resource-aware Computation-Communication Overlap for
 * multi-GPU ML Workloads"), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Conventions (all entry points)
 *   - extern "C"; plain pointers and sizes; no C++ or torch types cross this boundary.
 *   - Return value is an ra_status.  Nothing throws, aborts or prints.
 *   - "device pointer" = address in the current CUDA device's global memory;
 *     "host pointer"   = ordinary host memory.  Each argument says which.
 *   - Ownership: every device buffer (operands, results, GEMM workspace, trace buffer) is
 *     allocated and owned by the caller.  The library allocates no device memory; it lazily
 *     caches host-side objects only (streams, events, TMA descriptors), freed by ra_shutdown().
 *   - ra_gemm / ra_allreduce_emul / ra_alltoall_emul are ASYNCHRONOUS on `stream`
 *     (a cudaStream_t value passed as void*; NULL = legacy default stream).  Argument errors
 *     are detected before anything is enqueued, so a failing call has no side effects.
 *     ra_overlap_run / ra_overlap_sweep are SYNCHRONOUS.
 *   - Degenerate sizes: M, N or count == 0 -> RA_OK, nothing launched.  K == 0 -> C = beta*C.
 *   - There is NO CPU fallback: without an sm_100 device every compute entry point returns
 *     RA_ERR_ARCH (or RA_ERR_CUDA if no device/driver is present at all).
 */
#ifndef RA_H_
#define RA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RA_MAX_RANKS 16

typedef enum {
    RA_OK = 0,
    RA_ERR_INVALID_ARG = 1,     /* null pointer, negative dim, bad ld, misaligned pointer, P out of range, aliasing */
    RA_ERR_UNSUPPORTED = 2,     /* valid BLAS-wise but not implemented (ld not a multiple of 8 elements, ...) */
    RA_ERR_INFEASIBLE_KNOB = 3, /* smem_reserve_bytes / sm_budget cannot be honoured and allow_clamp == 0 */
    RA_ERR_CUDA = 4,            /* a CUDA call failed; ra_last_cuda_error() returns the cudaError_t value */
    RA_ERR_ARCH = 5,            /* current device is not compute capability 10.x */
    RA_ERR_SCRATCH_LIMIT = 6    /* ra_gemm_static_ws only: the plan needs more scratch than RA_GEMM_STATIC_WS_BYTES */
} ra_status;

/* Static string for a status code (never NULL). */
const char* ra_status_str(ra_status s);
/* cudaError_t of the most recent failing CUDA call made by this thread through the library (0 if none). */
int ra_last_cuda_error(void);
/* Destroys cached streams/events/descriptors.  Safe to call repeatedly. */
void ra_shutdown(void);

/* Device facts the occupancy planner uses (host out-pointers; any may be NULL).
 * Read from cudaDeviceGetAttribute at call time -- nothing is hard-coded. */
ra_status ra_device_info(int* sm_count, int* smem_per_sm, int* smem_per_block_optin, int* smem_reserved_per_block,
                         int* prio_least, int* prio_greatest);

/* ---------------------------------------------------------------------------------------------
 * S3  Occupancy shaping   (section 3.1: "by tuning the GEMM tile sizes, we
 * exploit the amount of shared memory allocated per block and therefore the number of resident
 * GEMM blocks";  PAPER.md:116, Fig. 3: thread-block count as the second axis.)
 *
 * smem_reserve_bytes  >= 0.  Shared memory PER SM that the GEMM must leave unallocated so that a
 *                     collective kernel can co-reside there.  The planner shrinks the GEMM's
 *                     pipeline depth, then its tile, until
 *                       ctas_per_sm * (dyn_smem_bytes + reserved_per_block) <= smem_per_sm - reserve.
 * sm_budget           number of GEMM CTAs of the persistent grid (one CTA per SM), 1..#SMs;
 *                     0 = all SMs.
 * tiles_per_cta       0 = fully persistent (grid = sm_budget, each CTA loops over its tiles);
 *                     t > 0 = bounded work: grid = ceil(n_tiles / t) and each CTA exits after
 *                     t tiles, so a higher-priority kernel gets SMs at CTA-exit granularity
 *                     (PAPER.md:59).  sm_budget is ignored in this mode.
 * allow_clamp         1: an infeasible knob is clamped to the nearest feasible value and the
 *                     plan reports what was used; 0: RA_ERR_INFEASIBLE_KNOB.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    int32_t smem_reserve_bytes;
    int32_t sm_budget;
    int32_t tiles_per_cta;
    int32_t allow_clamp;
    int32_t cta_group;        /* 0 = planner decides; 1 = single-CTA tiles (128 x N); 2 = CTA pairs (tcgen05
                                 cta_group::2, 256 x 256 tiles, 2-CTA clusters) where the shape allows */
    int32_t m_blocks;         /* 0 = planner decides; 1 = one 128-row MMA block per CTA (two TMEM accumulators, the
                                 epilogue fully overlaps the next tile); 2 = two blocks sharing one B stage (CTA
                                 pairs only: 512 x 256 tiles, 25 % less operand traffic per flop, one accumulator set) */
    int32_t cluster_k;        /* 0 = planner decides; 1 = never; 2 / 4 = cluster split-K in that many parts where the
                                 shape allows: the K range of one tile is split over the 2 or 4 CTAs of a cluster
                                 (single-CTA tiles) or the two CTA pairs of a 4-CTA cluster (256 x 256 pair tiles,
                                 2 parts only) and reduced through distributed shared memory in ascending-k order;
                                 needs parts * tiles <= #SMs (pairs: 4 * tiles) and room for the parts' accumulators
                                 in part 0's stage ring */
    int32_t l2_persist_bytes; /* 0 = off (default).  > 0: the GEMM claims this much of L2 as a persisting carve-out
                                 (cudaLimitPersistingL2CacheSize, clamped to the device maximum: 79 MiB on B200) and keeps
                                 the X-operand panel of one raster group resident in it (TMA loads with the evict_last
                                 policy, the group widened to what the carve-out holds), so X is read from DRAM once
                                 and Y once per group instead of both once per wave: 8192^3 moves 635 MB instead of 957 MB
                                 (profiles/r02_l2_persist.md).  The carve-out is DEVICE-WIDE and is taken from every
                                 other kernel's L2 -- the streaming collectives slow down next to it (measured: -10 % at
                                 24 MiB, 2.3x at 64 MiB and above) -- which makes it a resource traded between K_g and K_c
                                 like the shared-memory reserve.  ra_gemm sets the carve-out when it
                                 differs from what the library last set (one driver call, not inside a stream capture)
                                 and leaves it set; ra_overlap_run / _sweep / _autotune / _run_host set it for the run and
                                 take it back before returning; ra_l2_persist(0) takes it back too, and ra_shutdown puts back whatever
                                 carve-out the context had before the library first touched it.  With the knob at 0 the
                                 library still clears a carve-out it finds on first use (a foreign set-aside costs the
                                 collectives ~4 %), but only as best effort: if the driver refuses, the call carries on.
                                 Nothing is changed while `stream` is being captured.  Requests above the device maximum
                                 are clamped in the plan (ra_gemm_plan.l2_persist_bytes reports the clamped value).
                                 Ignored (reported as 0 in the plan) by swapped, stream-K, cluster split-K and
                                 single-wave plans.  Does not change results (same per-element k order). */
    int32_t tile_k;           /* 0 / 64 = default: 64 bf16 of K per pipeline stage (128-byte swizzle rows).  32: half-size
                                 stages (64-byte rows, two UMMA_K steps each) -- the tile-k axis of the paper's opt1 /
                                 opt2 study (a larger TILE_K gives every block a longer compute window
                                 and a larger shared-memory footprint).  K-contiguous operands only (transA = 0,
                                 transB = 1) and no cluster split-K: otherwise clamped to 64 / RA_ERR_INFEASIBLE_KNOB.
                                 Same per-element k order, so results are bit-identical to tile_k = 64.  Reported in
                                 ra_gemm_plan.tile_k. */
    int32_t tile_order;       /* 0 = default: persistent data-parallel plans with more tiles than workers hand out tiles
                                 DYNAMICALLY -- a worker's next tile is the next unclaimed one of the raster (one integer
                                 atomic per tile, claimed while the previous tile's loads are in flight), so workers that
                                 finish together start neighbouring tiles together and their loads of the shared operand
                                 rows coalesce in L2 (8192^3: 11 % fewer L2-slice reads, 2 % faster; profiles/r02_tile_order.md).
                                 1 = static: worker w owns tiles w, w + W, w + 2W, ...  Either way every C element is
                                 accumulated in the same ascending-k order, so results are bit-identical.  Single-CTA tiles,
                                 stream-K, cluster split-K, bounded-work and single-wave plans are always static.
                                 Concurrency: every dynamic-order launch IN FLIGHT owns one of 32 device-side launch slots
                                 (claim counter + ring), tracked with an event recorded behind the launch, so the same call
                                 on several streams or from several host threads is safe.  A launch that finds all slots in
                                 flight, or whose stream is being captured into a CUDA graph (the graph would hold the slot
                                 for as long as it lives), silently runs the static order instead -- same bits. */
} ra_occupancy;

/* What S3 decided -- for tests, logs and the sweep tables. */
typedef struct {
    int32_t ctas_per_sm;      /* GEMM CTAs per SM the plan's shared-memory accounting assumes (smem_left_per_sm is computed
                                 with it).  1 whenever single residency can be GUARANTEED by the footprint, i.e.
                                 hw_ctas_per_sm == 1.  2 for reserves above ~half an SM (> ~113 KiB), where no footprint can
                                 both honour the reserve and exclude a second CTA and the block scheduler does double up
                                 next to a busy collective (measured): every CTA is then sized so that the reserve holds
                                 with two resident.  Observable per launch: ra_gemm_residency(), the %smid trace */
    int32_t grid;             /* CTAs launched */
    int32_t stages;           /* depth of the TMA->MMA shared-memory ring */
    int32_t tile_m, tile_n, tile_k; /* CTA tile in C's coordinates (after operand swap) */
    int32_t split_k;          /* 1 = data-parallel tiles; >1 = stream-K (value = max parts of one tile) */
    int32_t swap_ab;          /* 1: computed as C^T = op(B)^T op(A)^T (skinny-M path) */
    int32_t dyn_smem_bytes;   /* dynamic shared memory per CTA, padding included */
    int32_t smem_left_per_sm; /* smem_per_sm - ctas_per_sm*(dyn_smem_bytes + reserved_per_block) */
    int32_t n_tiles;          /* output tiles */
    int32_t clamped;          /* 1 if a knob was clamped */
    int32_t cta_group;        /* 1, or 2 = CTA pairs: `grid` counts CTAs (2 per tile), sm_budget rounded down to even */
    int32_t m_blocks;         /* 128-row MMA blocks per CTA (1 or 2); tile_m = 128 * cta_group * m_blocks */
    int32_t cluster_k;        /* 1, or 2 / 4 = cluster split-K parts: `grid` = cluster_k * cta_group CTAs per tile, no workspace */
    int32_t hw_ctas_per_sm;   /* GEMM CTAs one SM COULD hold at this footprint = min over registers, threads and shared
                                 memory, from the device's own figures when an sm_100 device is current (the launched
                                 instantiation's register count, cudaFuncGetAttributes; registers / threads / shared memory
                                 per SM, cudaDeviceGetAttribute), else from B200's tables.  NOT taken from
                                 cudaOccupancyMaxActiveBlocksPerMultiprocessor: that call was measured to answer 1 for this
                                 kernel at every footprint while two of its CTAs were observed running on one SM.
                                 The planner pads dyn_smem_bytes past half an SM so that this is 1 whenever the padding
                                 fits under smem_reserve_bytes; otherwise ctas_per_sm follows it (see there).
                                 Bounded-work plans (tiles_per_cta > 0) always pad (clamping the reserve if they must).  A
                                 reserve so large that not even two minimal CTAs fit under it (~> 176 KiB) is clamped:
                                 clamped = 1 and smem_left_per_sm reports what two resident CTAs really leave. */
    int32_t group_x;          /* rasterisation: tile rows (of tile_m, or tile_n when swap_ab) per raster group; inside a
                                 group tiles are numbered row-fastest */
    int32_t l2_persist_bytes; /* the occupancy knob if this plan uses it, else 0 */
} ra_gemm_plan;

/* Host-only: computes the plan ra_gemm would use.  `occ` NULL = defaults {0,0,0,1,0,0,0,0,0,0}. */
ra_status ra_gemm_plan_query(int transA, int transB, int M, int N, int K, const ra_occupancy* occ, ra_gemm_plan* out);

/* S3 by measurement: every GEMM CTA counts itself in and out on its SM (%smid).  *max_ctas_on_one_sm receives the largest
 * number of GEMM CTAs (of any ra_gemm launch of this process on the current device) that were resident on one SM at the
 * same time since the last reset; reset != 0 clears the statistic afterwards.  Synchronises the device.  With
 * plan.ctas_per_sm == 1 a value of 2 means the reserve was NOT honoured on some SM.  Host out-pointer (may be NULL). */
ra_status ra_gemm_residency(int32_t* max_ctas_on_one_sm, int reset);

/* Bytes of device workspace ra_gemm needs for this problem and knob setting (0 if none).
 * Only stream-K plans (split_k > 1) need one. */
size_t ra_gemm_workspace_bytes(int transA, int transB, int M, int N, int K, const ra_occupancy* occ);

/* ---------------------------------------------------------------------------------------------
 * S1+S2  GEMM   (section 2.1:  C = alpha*op(A)*op(B) + beta*C,
 *                A in R^{MxK}, B in R^{KxN}, C in R^{MxN}.)
 *
 * bf16 operands, fp32 accumulation on the tcgen05 tensor cores (accumulator in TMEM), bf16
 * result (round-to-nearest-even).  Row-major buffers:
 *   transA = 0: A is M x K, lda >= K          transA = 1: A is K x M, lda >= M
 *   transB = 0: B is K x N, ldb >= N          transB = 1: B is N x K, ldb >= K
 *   C is M x N, ldc >= N.
 * A, B, C: device pointers, 16-byte aligned; lda, ldb, ldc multiples of 8 elements (TMA needs
 * 16-byte row pitch), else RA_ERR_UNSUPPORTED.  C must not overlap A or B.  All four (transA, transB)
 * combinations are implemented (K-contiguous operands use K-major, the others MN-major UMMA descriptors).
 * alpha, beta: host scalars by value.  beta == 0 => C is write-only (NaN/Inf already in C do not
 * propagate), as in BLAS.
 * workspace: device pointer, 16-byte aligned, at least ra_gemm_workspace_bytes(...) bytes (may be
 * NULL when that is 0).  Its contents are scratch; it must not be shared by two GEMMs in flight.
 * Thread-safety: calls on distinct streams from distinct host threads are safe (also with identical arguments) as
 * long as they do not share a workspace or write overlapping C.
 * Results are bit-reproducible run to run for a fixed (shape, plan): stream-K partial sums are
 * combined in ascending-k order, never with floating-point atomics.
 * ------------------------------------------------------------------------------------------- */
ra_status ra_gemm(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                  int ldb, float beta, void* C, int ldc, const ra_occupancy* occ, void* workspace,
                  size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * ra_gemm for callers that cannot provide scratch memory.
 *
 * ra_gemm leaves every device allocation to the caller, including the scratch a stream-K plan needs
 * (ra_gemm_workspace_bytes).  Some callers have no way to get that scratch: a plug-in that runs inside a
 * host application whose memory pool already owns the whole HBM and hands none out; code on a serving path
 * where cudaMalloc / cudaFree are forbidden because they stall every stream of the device -- exactly the
 * compute / communication concurrency this library exists to keep; a component that is only
 * given its operands and a stream and must not change the process's memory footprint after start-up.
 * This entry point is ra_gemm (bf16 output, same arguments, same kernels, same bits) with the workspace
 * taken from a fixed array that is part of the library image: RA_GEMM_STATIC_WS_BYTES of global memory,
 * 256-byte aligned, reserved on every GPU whose context loads libra.so and held until the process exits.
 * It calls no cudaMalloc, cudaFree or other allocating CUDA routine, on the first call or any later one.
 *
 *   - Plans that need no scratch behave exactly like ra_gemm with workspace = NULL.
 *   - A plan that needs more than RA_GEMM_STATIC_WS_BYTES is refused with RA_ERR_SCRATCH_LIMIT before
 *     anything is enqueued (nothing is written, nothing is launched): lower sm_budget, or use ra_gemm with
 *     a workspace of your own.  ra_gemm_workspace_bytes tells in advance (host only).
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that
 *     device current, return code checked) and remembers it.  Make that first call during start-up, outside
 *     any stream capture; later calls on that device only enqueue work on `stream`.
 *   - All calls, from every thread and on every stream, use the SAME array, and it keeps whatever the last
 *     call left in it.  The tile counters at its start are zeroed on `stream` ahead of every launch that
 *     uses them; the partial sums behind them are written before they are read, so stale contents never
 *     reach C.  But two calls whose kernels can run at the same time on one GPU (different streams, or
 *     different host threads without ordering between them) race on the array and produce wrong results
 *     without an error: order them on one stream or with events.  ra_gemm with per-call workspaces has no
 *     such restriction.
 *   - Errors otherwise as ra_gemm.
 * ------------------------------------------------------------------------------------------- */
#define RA_GEMM_STATIC_WS_BYTES ((size_t)16 << 20)   /* 16 MiB; config 5's stream-K plans need 4.6 - 6.9 MiB */
ra_status ra_gemm_static_ws(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                            int ldb, float beta, void* C, int ldc, const ra_occupancy* occ, void* stream);

/* The same GEMM with a choice of output type ("fp32 output").  c_dtype = RA_DTYPE_BF16 is ra_gemm.
 * RA_DTYPE_F32: C is M x N fp32, ldc in floats (ldc % 4 == 0, 16-byte aligned base); C = alpha*acc + beta*C_in is
 * stored as computed in fp32 (no bf16 rounding), and beta != 0 reads C_in as fp32.  Rounding that C to bf16 (RNE)
 * gives exactly ra_gemm's result.  RA_ERR_INVALID_ARG for any other c_dtype. */
typedef enum { RA_DTYPE_BF16 = 0, RA_DTYPE_F32 = 1 } ra_dtype;
ra_status ra_gemm_ex(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                     int ldb, float beta, void* C, int ldc, int c_dtype, const ra_occupancy* occ, void* workspace,
                     size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * S4  Allreduce stand-in   (section 2.2: "GEMM kernels compute local gradients, which
 * are then aggregated across all GPUs using allreduce"; BASELINE.json north_star: one device,
 * P rank buffers in HBM, fixed rank-order fp32 sum, result written back to all P buffers.)
 *
 *   for every e in [0,count):  s = bufs[0][e]; s = s + bufs[1][e]; ... ; s = s + bufs[P-1][e]
 *                              (each + one IEEE-754 binary32 round-to-nearest-even add, denormals kept)
 *                              bufs[r][e] = s  for all r.
 * bufs: HOST array of P DEVICE pointers (copied into the kernel parameters), 1 <= P <= RA_MAX_RANKS,
 * each 16-byte aligned, `count` floats, pairwise disjoint (overlap => RA_ERR_INVALID_ARG).
 * sm_budget: SMs' worth of CTAs to launch (0 = all SMs).
 * ------------------------------------------------------------------------------------------- */
ra_status ra_allreduce_emul(float* const* bufs, int P, size_t count, int sm_budget, void* stream);
/* Extended form.  variant 0: 128-bit loads/stores from registers, no shared memory; ctas_per_sm = CTAs (256 threads
 * each) per budgeted SM, 1..4 (0 = default 2).  variant 1: TMA ring -- a thread bulk-copies the P rank slices of a unit
 * into a shared-memory slot, 128 threads sum them there in the same rank order (bit-identical result), the first slice is
 * bulk-stored to all P buffers; smem_bytes_per_cta = two slots of P slices (0 = 64 KiB), ctas_per_sm 0 = 2.  This is
 * the variant whose co-residency with the GEMM depends on smem_reserve_bytes.  variant 2: the all-gather half on the
 * copy engines (the mechanism of ConCCL's DMA offload): variant 0's kernel writes the sum to bufs[0] only
 * (4P + 4 bytes per element through the SMs instead of 8P) and P-1 device-to-device cudaMemcpyAsync on the same stream
 * fan it out; same bits, 12P - 4 bytes of HBM traffic per element instead of 8P.  (Same argument order as
 * ra_alltoall_emul_ex.) */
ra_status ra_allreduce_emul_ex(float* const* bufs, int P, size_t count, int sm_budget, int smem_bytes_per_cta, int ctas_per_sm,
                               int variant, void* stream);

/* ---------------------------------------------------------------------------------------------
 * S5  Alltoall stand-in   ("expert-parallel workloads rely on alltoall to route
 * tokens between devices"; BASELINE.json: P x P chunk transpose on one device.)
 *
 *   recv[(j*P + i)*chunk_bytes + b] = send[(i*P + j)*chunk_bytes + b]   for i,j < P, b < chunk_bytes.
 * send, recv: device pointers, 16-byte aligned, P*P*chunk_bytes bytes each, disjoint
 * (overlap => RA_ERR_INVALID_ARG).  chunk_bytes % 16 == 0.  1 <= P <= 256.
 * Implemented with TMA bulk copies (global -> shared ring -> global), one issuing thread per ring.
 * sm_budget as above.
 * ------------------------------------------------------------------------------------------- */
ra_status ra_alltoall_emul(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget, void* stream);

/* Extended form: explicit shared-memory footprint and variant.
 *   smem_bytes_per_cta  shared-memory ring per CTA (0 = default 64 KiB).  This is what must fit
 *                       inside the GEMM's smem_reserve_bytes on SMs the two kernels share.
 *   ctas_per_sm         CTAs launched per budgeted SM (0 = default).
 *   variant             0 = TMA bulk-copy ring; 1 = plain 128-bit LDG/STG copy (no shared memory);
 *                       2 = copy engines (P*P cudaMemcpyAsync device-to-device copies, no SM residency). */
ra_status ra_alltoall_emul_ex(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget,
                              int smem_bytes_per_cta, int ctas_per_sm, int variant, void* stream);

/* ---------------------------------------------------------------------------------------------
 * S6-S8  Overlap driver   (section 3.2: two streams per device, event dependency
 * K_g^i -> K_c^i, K_g^{i+1} free to run concurrently with K_c^i;  PAPER.md:59, section 3.3:
 * the communication stream gets the higher priority;  PAPER.md:108-110: TimeRatio, overlap rate.)
 * ------------------------------------------------------------------------------------------- */
typedef enum { RA_COLL_ALLREDUCE = 0, RA_COLL_ALLTOALL = 1, RA_COLL_NONE = 2 } ra_coll_kind;
typedef enum { RA_MODE_SERIAL = 0, RA_MODE_OVERLAP = 1 } ra_mode;

typedef struct {
    /* GEMM K_g (same operands every iteration); set M = 0 to run the collective alone */
    int32_t transA, transB, M, N, K;
    float alpha, beta;
    const void* A; int32_t lda;
    const void* B; int32_t ldb;
    void* C; int32_t ldc;
    void* workspace; size_t workspace_bytes;
    /* collective K_c */
    int32_t kind;               /* ra_coll_kind */
    int32_t P;
    float* const* ar_bufs;      /* HOST array of P device pointers (allreduce, in place) */
    size_t ar_count;
    void* a2a_a; void* a2a_b;   /* device; iteration i copies a->b if i is even, b->a if odd */
    size_t chunk_bytes;
    int32_t n_iters;
    float* const* ar_pristine;  /* optional (NULL = off): HOST array of P device pointers, ar_count floats each, disjoint
                                   from ar_bufs.  ra_overlap_run / _sweep / _autotune copy ar_pristine[r] -> ar_bufs[r]
                                   device-to-device before EVERY run, outside the timed window, so that repeated runs of
                                   the in-place allreduce (magnitudes grow by P per iteration) always reduce the same
                                   finite data.  Ignored by ra_overlap_run_host (it uploads its inputs every step). */
} ra_workload;

typedef struct {
    int32_t mode;               /* ra_mode */
    ra_occupancy occ;           /* GEMM knobs */
    int32_t coll_sm_budget;     /* 0 = all SMs */
    int32_t coll_smem_bytes;    /* TMA-ring variants: ring bytes per CTA (0 = default 64 KiB) */
    int32_t coll_ctas_per_sm;   /* collective CTAs per budgeted SM; 0 = default */
    int32_t coll_variant;       /* alltoall: 0 = TMA ring, 1 = LDG/STG, 2 = copy engines;  allreduce: 0 = LDG/STG, 1 = TMA ring,
                                   2 = LDG/STG reduce into rank 0 + copy-engine fan-out */
    int32_t prio_compute, prio_comm; /* cudaStreamCreateWithPriority values; equal = "priority off" */
    int32_t dependent;          /* 1: K_c^i waits for K_g^i (the paper's schedule); 0: free-running streams */
    int32_t record_kernel_times;/* 1: per-kernel event pairs (perturbs the schedule slightly) */
    int32_t use_graph;          /* 1: capture the n_iters schedule (both streams, all dependencies) into a CUDA graph
                                   once per (workload, setting) and replay it with one launch -- for launch-bound
                                   steps.  Ignored when record_kernel_times = 1.  Graphs are cached until ra_shutdown;
                                   the caller's buffers must stay valid while they are cached. */
} ra_overlap_cfg;

typedef struct {
    float total_ms;             /* GPU time, first launch to last completion, events on both streams
                                   (ra_overlap_sweep: mean over the measured runs) */
    float median_ms, min_ms;    /* ra_overlap_sweep: median / min over the measured runs (run: = total_ms) */
    float gemm_ms_sum, coll_ms_sum; /* sums of per-kernel durations (record_kernel_times only, else 0) */
    float overlap_rate;         /* sum |K_c ∩ ∪K_g| / sum |K_c|; record_kernel_times only */
    ra_gemm_plan plan;
    float* kernel_times;        /* optional HOST array, 4*n_iters floats: g_start, g_end, c_start, c_end (ms from t0) */
} ra_overlap_result;

/* Runs n_iters iterations under `cfg`, synchronises, fills `res` (host pointers all). */
ra_status ra_overlap_run(const ra_workload* w, const ra_overlap_cfg* cfg, ra_overlap_result* res);

/* ---------------------------------------------------------------------------------------------
 * The same step from HOST buffers (the end-to-end entry point).  One step = copy this step's inputs
 * host -> device, run the n_iters iterations of ra_overlap_run under `cfg`, copy the results device ->
 * host.  The library software-pipelines consecutive steps on its own copy streams:
 *     H2D(step s+1)  ||  compute(step s)  ||  D2H(step s-1)
 * over the device buffer sets dev0 / dev1 (dev1 may be NULL: one set, copies and compute of
 * consecutive steps then serialise).  Every step reads the same host inputs and overwrites the same
 * host outputs (a serving loop would rotate them).
 *
 * ra_host_io   HOST pointers; pinned memory is needed for the copies to overlap (pageable memory is
 *              legal but makes cudaMemcpyAsync synchronous).  Sizes follow dev0:
 *   A, B       the GEMM operands exactly as ra_gemm takes them: rows x ld bf16 (rows = M or K by transA, ...)
 *   C          out, M x ldc bf16 (may be NULL: not copied back)
 *   ar_in      P host pointers of ar_count floats (the rank buffers before the step)
 *   ar_out     ar_count floats: rank 0's buffer after the step's n_iters allreduces (may be NULL)
 *   a2a_in     P*P*chunk_bytes, goes to a2a_a;  a2a_out: the buffer the last iteration wrote (may be NULL)
 * dev0, dev1   workloads of identical shape with disjoint DEVICE buffers (caller-owned, as in ra_overlap_run).
 * res          total_ms = GPU time from the first copy to the last, over all n_steps (events on the copy streams).
 * Synchronous.  RA_ERR_INVALID_ARG for a NULL required pointer, n_steps < 1 or mismatched sets.
 * --------------------------------------------------------------------------------------------- */
typedef struct {
    const void* A;
    const void* B;
    void* C;
    const float* const* ar_in;
    float* ar_out;
    const void* a2a_in;
    void* a2a_out;
} ra_host_io;

ra_status ra_overlap_run_host(const ra_workload* dev0, const ra_workload* dev1, const ra_host_io* io,
                              const ra_overlap_cfg* cfg, int n_steps, ra_overlap_result* res);

/* ---------------------------------------------------------------------------------------------
 * S7'  Knob policy from a roofline model (automating the knob selection is the
 * paper's future work).  Host only, runs nothing: predicts the setting the exhaustive sweep would pick
 * from the two kernels' flops / bytes and the chip's tensor and HBM peaks (csrc/ra_policy.cu states the
 * model).  `peaks` NULL or zero fields = built-in B200 figures (1400 TFLOP/s sustained bf16, 6450 GB/s).
 * Times are per pipelined iteration, in ms.  bench.py runs the suggestion inside the sweep and reports
 * its regret against the sweep's best.
 * --------------------------------------------------------------------------------------------- */
typedef struct {
    double tensor_tflops;       /* dense bf16 peak to model against (sustained) */
    double hbm_gbs;             /* HBM bandwidth to model against */
} ra_peaks;

typedef struct {
    ra_overlap_cfg cfg;         /* the suggested setting (mode = RA_MODE_OVERLAP) */
    int32_t gemm_bound;         /* 0: the GEMM alone is tensor-bound, 1: HBM-bound */
    double t_gemm_ms, t_coll_ms;/* each kernel alone at its roofline */
    double t_overlap_ms;        /* predicted per-iteration time of the n_iters pipeline (head and tail included) */
    double t_serial_ms;         /* t_gemm_ms + t_coll_ms */
    double t_roofline_ms;       /* max(flops / tensor peak, (gemm + collective bytes) / HBM peak) */
} ra_suggestion;

ra_status ra_overlap_suggest(const ra_workload* w, const ra_peaks* peaks, ra_suggestion* out);

/* Model + measurement: times the model's pick and its neighbours (collective variant, throttled collective
 * coll_sm_budget 24 / 32 / 48 for tensor-bound GEMMs, priority on) with ra_overlap_sweep(runs) -- at most ~14 settings
 * instead of the exhaustive grid -- and returns the fastest.  Runs the workload (an in-place allreduce keeps summing
 * its buffers, as in ra_overlap_sweep).  best_res (optional) receives that setting's result, n_tried (optional) the
 * number of settings timed.  Synchronous; host pointers all. */
ra_status ra_overlap_autotune(const ra_workload* w, const ra_peaks* peaks, int runs, ra_overlap_cfg* best_cfg,
                              ra_overlap_result* best_res, int* n_tried);

/* Times cfgs[0..n): every setting is run as one block of consecutive runs, the first of them warm-up, and the mean
 * of the remaining runs - runs/3 is stored in results[i].total_ms ("30 runs ... the first one-third of runs
 * are considered warm-up").  The warm-up lasts runs/3 runs or, with n > 1 and if that is longer, until the setting has run
 * for ~120 ms (at most 12 runs): a power-capped step is otherwise timed in the clock / power state the previous setting
 * left behind (measured on cb-ar: ~100 ms at 0.80 ms per iteration after a lighter setting before it settles at
 * 0.90-0.94).  *best = argmin over settings with mode == RA_MODE_OVERLAP (or over all if none).  Host pointers all. */
ra_status ra_overlap_sweep(const ra_workload* w, const ra_overlap_cfg* cfgs, int n, int runs,
                           ra_overlap_result* results, int* best);

/* ---------------------------------------------------------------------------------------------
 * N4: the stand-ins as real exchanges over peer memory ("aggregated across all GPUs using allreduce ...
 * alltoall to route tokens between devices"; 4 / 8 GPUs per node).  One process per GPU; every rank owns one
 * buffer and reaches the others' through CUDA IPC mappings (NVLink / NVSwitch peer memory).  K2 and K3 are unchanged:
 * they only ever take P device pointers.  No call here waits on another rank: the caller orders the ranks (a barrier of
 * its process group before -- inputs ready -- and after -- every slice / chunk written).  Unmeasured on NVLink
 * (one GPU at hand): exercised by P sequential ranks on one device and by two processes sharing one device through
 * real IPC handles (tests/test_peer_gpu.py).
 *
 * ra_ipc_handle   what a rank publishes for one device pointer: the CUDA IPC handle of the allocation that holds it,
 *                 the pointer's offset inside that allocation (so sub-allocated pointers, e.g. a caching allocator's,
 *                 can be shared) and the bytes that follow it.  Plain bytes: ship it over any transport.
 * ra_ipc_export   HOST out-pointer; dev_ptr a DEVICE pointer of this process (not itself an IPC mapping).
 * ra_ipc_open     maps a peer's handle into this process (peer access is enabled lazily by the driver) and returns the
 *                 DEVICE pointer that corresponds to the exported one.  Opening the same handle again returns the same
 *                 pointer and takes another reference: pair every ra_ipc_open with one ra_ipc_close.  NOTE: the handle
 *                 covers the whole ALLOCATION that holds the exported pointer (a caching allocator's segment, say), so a
 *                 peer can reach everything in it; export from dedicated allocations if that matters.
 * ra_ipc_close    drops one reference on a pointer ra_ipc_open returned (RA_ERR_INVALID_ARG for any other pointer) and
 *                 unmaps it with the last one; ra_shutdown unmaps whatever is still open.
 * ra_peer_slice   host-only: the floats [begin, end) of a count-float buffer that rank `rank` of P reduces; the slices
 *                 partition [0, count), boundaries are multiples of 4 floats (16-byte vectors).
 * ra_allreduce_peer  bufs: HOST array of the P DEVICE pointers IN RANK ORDER (own buffer at index rank, the rest opened
 *                 from the peers' handles), count floats each.  Launches K2 on this rank's slice: sum in the fixed order
 *                 0..P-1, one RNE binary32 add per rank, written back to the slice of ALL P buffers.  After every rank
 *                 has run, every buffer equals the oracle's allreduce bit for bit.  variant as ra_allreduce_emul_ex.
 * ra_alltoall_peer   send: this rank's P chunks (DEVICE); recv: HOST array of the P ranks' receive buffers (DEVICE
 *                 pointers in rank order, P chunks each).  Pushes chunk j into slot `rank` of recv[j]:
 *                 recv_j[rank] = send_rank[j].  variant as ra_alltoall_emul_ex (2 = copy engines, peer-to-peer).  The receive
 *                 buffers must be pairwise disjoint and disjoint from send (else RA_ERR_INVALID_ARG).
 * Errors as the emulation calls; 1 <= P <= RA_MAX_RANKS, 0 <= rank < P.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
    uint8_t opaque[64];   /* cudaIpcMemHandle_t */
    uint64_t offset;      /* of the exported pointer inside its allocation */
    uint64_t bytes;       /* from the exported pointer to the end of its allocation */
} ra_ipc_handle;

ra_status ra_ipc_export(const void* dev_ptr, ra_ipc_handle* out);
ra_status ra_ipc_open(const ra_ipc_handle* h, void** dev_ptr);
ra_status ra_ipc_close(void* dev_ptr);
ra_status ra_peer_slice(size_t count, int P, int rank, size_t* begin, size_t* end);
ra_status ra_allreduce_peer(float* const* bufs, int P, int rank, size_t count, int sm_budget, int variant, void* stream);
ra_status ra_alltoall_peer(const void* send, void* const* recv, int P, int rank, size_t chunk_bytes, int sm_budget, int variant,
                           void* stream);

/* Sets the current device's persisting-L2 carve-out to min(bytes, device maximum) and reports what was granted (host
 * out-pointer, may be NULL; the driver rounds up to sixteenths of the L2, 7.9 MiB steps on B200); bytes = 0 takes it back and turns the lines it held into normal ones.  This is the state
 * ra_occupancy.l2_persist_bytes manages for the GEMM (see there); the call exists so that a caller who ran ra_gemm with
 * the knob can give the L2 back before launching something else.  One driver call when the value changes, none
 * otherwise; not to be called while a stream of the device is being captured.  RA_ERR_INVALID_ARG for bytes < 0. */
ra_status ra_l2_persist(int64_t bytes, int64_t* granted);

/* ---------------------------------------------------------------------------------------------
 * Residency trace (evidence for "per-SM residency during overlap").  When a trace buffer is set,
 * every CTA of every library kernel appends one record {tag, block, t_start, t_end}:
 *   tag = kernel_id << 32 | %smid   (kernel_id: 1 = GEMM, 2 = allreduce, 3 = alltoall)
 *   t_* = %globaltimer (ns).
 * buf: DEVICE pointer to (1 + 4*capacity) uint64; buf[0] is the record counter (caller zeroes it).
 * Pass NULL to disable (default).  Not thread-safe with concurrent launches from other threads.
 * ------------------------------------------------------------------------------------------- */
ra_status ra_set_trace(uint64_t* buf, size_t capacity);

#ifdef __cplusplus
}
#endif
#endif /* RA_H_ */
