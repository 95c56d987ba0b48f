// ra_policy.cu -- knob policy from a roofline model (the paper's stated future work, PAPER.md:144, 160:
// "automating the selection of occupancy/priority settings").  Host only.
//
// The exhaustive sweep (ra_overlap_sweep) stays the ground truth; this predicts a setting without running
// anything, from the two kernels' work and the chip's two rooflines:
//   t_tensor(b) = flops / (tensor_peak * b/#SMs * wave_efficiency(b))      GEMM on b SMs
//   t_bytes     = (gemm_bytes + coll_bytes) / hbm_peak                     both kernels share HBM
//   t_overlap(b) = max(t_tensor(b), t_bytes)                               per pipelined iteration
//   t_step       = (t_gemm_alone + (n-1) * t_overlap + t_coll_alone) / n   K_g^0 and K_c^{n-1} have no partner
// What the B200 sweeps showed and the model encodes (profiles/r03_sweeps.md: full grid, block protocol, 30 runs):
//   * the collective stand-ins need no shared memory (allreduce, LDG alltoall) or 64 KiB (TMA alltoall) and
//     <= 64 registers/thread, and the tcgen05 GEMM is one 192-thread CTA of 128 registers per SM, so they
//     co-reside on every SM without any reserve: constraining the GEMM's SM budget only costs tensor time.
//     => sm_budget = the b that minimises t_overlap (all SMs unless a smaller even b quantises better).
//   * smem_reserve_bytes = 0: a reserve only shortens the GEMM's pipeline.
//   * the TMA-ring collectives need their ring somewhere: the alltoall's is chosen when the GEMM leaves SMs free
//     (skinny GEMM: 128 tiles on 148 SMs) or >= ring + 1 KiB per SM unallocated, otherwise the shared-memory-free
//     LDG/STG variant; the allreduce's only next to an HBM-bound GEMM (it saturates HBM from few SMs).
//   * priority: a persistent GEMM never yields an SM, so priority only orders pending grids; "off".  Measured Norm. time
//     (on / off) over ~160-200 like-for-like pairs per workload: median 1.000-1.001; +2.5-3 % at the best cb setting.
#include <cstring>

#include "ra_common.cuh"

namespace ra {

constexpr double kDefaultTensorTflops = 1400.0;   // sustained bf16, power-capped B200 (MEASURED_PEAKS.json of this pool)
constexpr double kDefaultHbmGbs = 6450.0;
constexpr int kA2aRingBytes = 64 * 1024;

static double wave_eff(long long tiles, int workers) {
    if (tiles <= 0 || workers <= 0) return 1.0;
    const long long waves = (tiles + workers - 1) / workers;
    return (double)tiles / (double)(waves * workers);
}

}  // namespace ra

extern "C" {

ra_status ra_overlap_suggest(const ra_workload* w, const ra_peaks* peaks, ra_suggestion* out) {
    if (w == nullptr || out == nullptr) return RA_ERR_INVALID_ARG;
    if (w->n_iters < 1) return RA_ERR_INVALID_ARG;
    if (w->kind != RA_COLL_ALLREDUCE && w->kind != RA_COLL_ALLTOALL && w->kind != RA_COLL_NONE) return RA_ERR_INVALID_ARG;
    const double tensor = (peaks && peaks->tensor_tflops > 0) ? peaks->tensor_tflops : ra::kDefaultTensorTflops;
    const double hbm = (peaks && peaks->hbm_gbs > 0) ? peaks->hbm_gbs : ra::kDefaultHbmGbs;

    int sm_count = ra::kDefaultSmCount;
    {
        ra::DeviceInfo di;
        if (ra::device_info(&di) == RA_OK) {
            sm_count = di.sm_count;
        } else {
            ra::g_last_cuda_error = 0;
            (void)cudaGetLastError();
        }
    }

    const bool has_gemm = w->M > 0 && w->N > 0;
    const double M = w->M, N = w->N, K = w->K;
    const double flops = has_gemm ? 2.0 * M * N * K : 0.0;
    const double gbytes = has_gemm ? 2.0 * (M * K + K * N + M * N) + (w->beta != 0.f ? 2.0 * M * N : 0.0) : 0.0;
    double cbytes = 0.0;
    if (w->kind == RA_COLL_ALLREDUCE) cbytes = 2.0 * 4.0 * (double)w->P * (double)w->ar_count;
    if (w->kind == RA_COLL_ALLTOALL) cbytes = 2.0 * (double)w->P * (double)w->P * (double)w->chunk_bytes;

    ra_suggestion s{};
    s.cfg.mode = RA_MODE_OVERLAP;
    s.cfg.occ = {0, 0, 0, 1, 0, 0, 0, 0, 0, 0};
    s.cfg.dependent = 1;
    s.cfg.prio_compute = 0;
    s.cfg.prio_comm = 0;                                  // priority off (persistent GEMM, see header)

    const double t_bytes = (gbytes + cbytes) / (hbm * 1e6);        // ms
    const double t_gemm_mem = gbytes / (hbm * 1e6);
    const double t_coll = cbytes / (hbm * 1e6);
    double best_t = 0.0, t_tensor_all = 0.0;
    int best_b = 0;
    ra_gemm_plan best_plan{};
    if (has_gemm) {
        // candidate budgets: all SMs and every smaller even count down to half the chip (the sweep's range)
        for (int b = sm_count; b >= sm_count / 2; b -= 2) {
            ra_occupancy occ = {0, b == sm_count ? 0 : b, 0, 1, 0, 0, 0};
            ra_gemm_plan pl{};
            RA_TRY(ra_gemm_plan_query(w->transA, w->transB, w->M, w->N, w->K, &occ, &pl));
            const int workers = pl.grid / (pl.cta_group > 0 ? pl.cta_group : 1);
            // stream-K plans split the k-blocks evenly: no quantisation loss
            const double eff = pl.split_k > 1 ? 1.0 : ra::wave_eff(pl.n_tiles, workers);
            const double t_tensor = flops / (tensor * 1e9 * ((double)pl.grid / sm_count) * eff);
            if (b == sm_count) t_tensor_all = t_tensor;
            const double t = t_tensor > t_bytes ? t_tensor : t_bytes;
            // prefer more SMs on ties (1 % hysteresis): fewer CTAs never helps the collective here
            if (best_b == 0 || t < best_t * 0.99) {
                best_t = t;
                best_b = b;
                best_plan = pl;
            }
        }
        s.cfg.occ.sm_budget = best_b == sm_count ? 0 : best_b;
        s.gemm_bound = (t_tensor_all >= t_gemm_mem) ? 0 : 1;
    } else {
        best_t = t_bytes;
    }

    {
        // TMA-ring collectives (alltoall variant 0, allreduce variant 1) saturate HBM from few SMs but need their ring
        // somewhere: on SMs the GEMM leaves free, or in shared memory it leaves unallocated
        const int free_sms = has_gemm ? sm_count - best_plan.grid : sm_count;
        const bool ring_fits = !has_gemm || best_plan.smem_left_per_sm >= ra::kA2aRingBytes + 1024 + 1024;
        const bool ring_ok = ring_fits || free_sms >= 16;
        if (w->kind == RA_COLL_ALLTOALL) s.cfg.coll_variant = ring_ok ? 0 : 1;
        // allreduce: the register variant is at least as fast under a tensor-bound GEMM (it co-resides everywhere);
        // next to an HBM-bound GEMM the ring variant measured 0.2517 vs 0.2561 ms per iteration (mb-ar)
        if (w->kind == RA_COLL_ALLREDUCE) s.cfg.coll_variant = (ring_ok && has_gemm && s.gemm_bound == 1) ? 1 : 0;
    }

    // Collective-bound step under a tensor-bound GEMM (the paper's literal cb workloads: 7.5 GB of collective against a
    // 0.7 ms GEMM).  The GEMM's default plan leaves 1.75 KiB of an SM's shared memory: room for ONE collective CTA (each
    // costs 1 KiB of system-reserved shared memory) and no L1 (carved from the same array): measured, the overlapped step
    // is then no faster than the serial one (2.02 vs 2.03 ms).  A 32 KiB reserve costs the GEMM a pipeline stage it does
    // not need here and gives the collective its second CTA and its L1 back: 1.55 ms.  This is the paper's knob doing the paper's job
    // (PAPER.md:45-47); when the GEMM is the long pole (cb-ar) the stage is worth more than the collective's speed.
    // The alltoall has a better answer in that regime: the copy engines move it without any SM, L1 or shared memory
    // (paper-cb-a2a: 1.54-1.63 ms for every GEMM setting against 1.74+ for the SM variants).
    if (has_gemm && w->kind != RA_COLL_NONE && s.gemm_bound == 0 && t_coll > t_tensor_all) {
        if (w->kind == RA_COLL_ALLTOALL) s.cfg.coll_variant = 2;
        else s.cfg.occ.smem_reserve_bytes = 32 * 1024;
    }

    const double t_gemm_alone = has_gemm ? (t_tensor_all > t_gemm_mem ? t_tensor_all : t_gemm_mem) : 0.0;
    const int n = w->n_iters;
    s.t_gemm_ms = t_gemm_alone;
    s.t_coll_ms = t_coll;
    s.t_overlap_ms = (w->kind == RA_COLL_NONE || !has_gemm) ? best_t : (t_gemm_alone + (n - 1) * best_t + t_coll) / n;
    s.t_serial_ms = t_gemm_alone + t_coll;
    s.t_roofline_ms = (has_gemm && t_tensor_all > t_bytes) ? t_tensor_all : t_bytes;
    // launch-bound steps (kernels of a few microseconds: Tiny): replay the schedule as one CUDA graph
    // (measured 12.2 -> 8.2 us per overlapped iteration on Tiny; no effect on the full-size workloads)
    s.cfg.use_graph = (s.t_serial_ms < 0.05) ? 1 : 0;
    *out = s;
    return RA_OK;
}

/* Model pick + its neighbours, measured: the short list the sweeps showed to contain the winner -- the collective's
 * variant (alltoall), a throttled collective (coll_sm_budget 24 / 32 / 48 when the GEMM is tensor-bound), priority on
 * for the model's pick -- is timed with ra_overlap_sweep and the best setting returned. */
ra_status ra_overlap_autotune(const ra_workload* w, const ra_peaks* peaks, int runs, ra_overlap_cfg* best_cfg,
                              ra_overlap_result* best_res, int* n_tried) {
    if (w == nullptr || best_cfg == nullptr || runs < 1) return RA_ERR_INVALID_ARG;
    ra_suggestion s{};
    RA_TRY(ra_overlap_suggest(w, peaks, &s));
    ra::DeviceInfo di;
    RA_TRY(ra::device_info(&di));
    RA_TRY(ra::require_sm100(di));

    ra_overlap_cfg cand[32];
    int n = 0;
    auto push = [&](const ra_overlap_cfg& c) {
        for (int i = 0; i < n; ++i)
            if (memcmp(&cand[i], &c, sizeof(c)) == 0) return;
        if (n < 32) cand[n++] = c;
    };
    const bool has_gemm = w->M > 0 && w->N > 0;
    const int variants = w->kind == RA_COLL_ALLTOALL ? 3 : (w->kind == RA_COLL_ALLREDUCE ? 2 : 1);
    push(s.cfg);
    for (int v = 0; v < variants; ++v) {
        ra_overlap_cfg c = s.cfg;
        c.coll_variant = v;
        push(c);
        if (has_gemm && s.gemm_bound == 0 && !(w->kind == RA_COLL_ALLTOALL && v == 2)) {   // the copy engines have no SM budget
            for (int csb : {24, 32, 48}) {
                ra_overlap_cfg t = c;
                t.coll_sm_budget = csb;
                push(t);
            }
        }
    }
    {
        ra_overlap_cfg c = s.cfg;
        c.prio_comm = di.prio_greatest;
        push(c);
    }
    ra_overlap_result res[32];
    memset(res, 0, sizeof(res));
    int best = -1;
    RA_TRY(ra_overlap_sweep(w, cand, n, runs, res, &best));
    if (best < 0) return RA_ERR_INVALID_ARG;
    *best_cfg = cand[best];
    if (best_res) {
        float* kt = best_res->kernel_times;
        *best_res = res[best];
        best_res->kernel_times = kt;
    }
    if (n_tried) *n_tried = n;
    return RA_OK;
}

}  // extern "C"
