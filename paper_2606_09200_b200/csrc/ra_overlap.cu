// ra_overlap.cu -- D1: the overlap driver (S6, S7, S8).
//
// Schedule (section 3.2): a compute stream carries K_g^0, K_g^1, ...; a communication
// stream carries K_c^0, K_c^1, ...; K_c^i waits on an event recorded after K_g^i; nothing orders
// K_g^{i+1} after K_c^i, so they may run concurrently.  Priority-aware variant (PAPER.md:59,
// section 3.3): the communication stream is created with the higher priority.  Serial baseline
// (Fig. 1a): everything on one stream.  Metrics.
#include <algorithm>
#include <map>
#include <mutex>
#include <vector>

#include "ra_common.cuh"

namespace ra {

ra_status gemm_launch(int transA, int transB, int M, int N, int K, float alpha, const void* A, int lda, const void* B,
                      int ldb, float beta, void* C, int ldc, const ra_occupancy* occ, void* workspace,
                      size_t workspace_bytes, cudaStream_t stream, ra_gemm_plan* plan_out);
ra_status allreduce_launch(float* const* bufs, int P, size_t count, int sm_budget, int ctas_per_sm, cudaStream_t stream);
ra_status alltoall_launch(const void* send, void* recv, int P, size_t chunk_bytes, int sm_budget,
                          int smem_bytes_per_cta, int ctas_per_sm, int variant, cudaStream_t stream);

// ---- cached host objects ----------------------------------------------------------------------
struct Cache {
    std::mutex mu;
    std::map<std::pair<int, int>, cudaStream_t> streams;   // (role, priority) -> stream
    std::vector<cudaEvent_t> dep_events;                   // no timing
    std::vector<cudaEvent_t> timed_events;                 // timing
};
static Cache g_cache;

static ra_status get_stream(int role, int prio, cudaStream_t* out) {
    auto key = std::make_pair(role, prio);
    auto it = g_cache.streams.find(key);
    if (it != g_cache.streams.end()) {
        *out = it->second;
        return RA_OK;
    }
    cudaStream_t s;
    RA_CUDA(cudaStreamCreateWithPriority(&s, cudaStreamNonBlocking, prio));
    g_cache.streams[key] = s;
    *out = s;
    return RA_OK;
}
static ra_status ensure_events(std::vector<cudaEvent_t>& v, size_t n, unsigned flags) {
    while (v.size() < n) {
        cudaEvent_t e;
        RA_CUDA(cudaEventCreateWithFlags(&e, flags));
        v.push_back(e);
    }
    return RA_OK;
}

static ra_status validate(const ra_workload* w, const ra_overlap_cfg* cfg, ra_overlap_result* res) {
    if (w == nullptr || cfg == nullptr || res == nullptr) return RA_ERR_INVALID_ARG;
    if (w->n_iters < 1 || w->n_iters > 4096) return RA_ERR_INVALID_ARG;
    if (cfg->mode != RA_MODE_SERIAL && cfg->mode != RA_MODE_OVERLAP) return RA_ERR_INVALID_ARG;
    if (w->kind != RA_COLL_ALLREDUCE && w->kind != RA_COLL_ALLTOALL && w->kind != RA_COLL_NONE) return RA_ERR_INVALID_ARG;
    if (w->kind == RA_COLL_NONE && w->M == 0) return RA_ERR_INVALID_ARG;
    return RA_OK;
}

static ra_status launch_coll(const ra_workload* w, const ra_overlap_cfg* cfg, int iter, cudaStream_t s) {
    if (w->kind == RA_COLL_ALLREDUCE) return allreduce_launch(w->ar_bufs, w->P, w->ar_count, cfg->coll_sm_budget, cfg->coll_ctas_per_sm, s);
    if (w->kind == RA_COLL_ALLTOALL) {
        const void* src = (iter & 1) ? w->a2a_b : w->a2a_a;
        void* dst = (iter & 1) ? w->a2a_a : w->a2a_b;
        return alltoall_launch(src, dst, w->P, w->chunk_bytes, cfg->coll_sm_budget, cfg->coll_smem_bytes,
                               cfg->coll_ctas_per_sm, cfg->coll_variant, s);
    }
    return RA_OK;
}

static ra_status run_once(const ra_workload* w, const ra_overlap_cfg* cfg, ra_overlap_result* res) {
    std::lock_guard<std::mutex> lk(g_cache.mu);
    const int n = w->n_iters;
    const bool has_gemm = w->M > 0 && w->N > 0;
    const bool has_coll = w->kind != RA_COLL_NONE;
    const bool overlap = cfg->mode == RA_MODE_OVERLAP;
    const bool rec = cfg->record_kernel_times != 0;

    DeviceInfo di;
    RA_TRY(device_info(&di));
    RA_TRY(require_sm100(di));
    if (cfg->prio_compute > di.prio_least || cfg->prio_compute < di.prio_greatest || cfg->prio_comm > di.prio_least ||
        cfg->prio_comm < di.prio_greatest)
        return RA_ERR_INVALID_ARG;

    cudaStream_t s_comp, s_comm;
    RA_TRY(get_stream(0, cfg->prio_compute, &s_comp));
    if (overlap) RA_TRY(get_stream(1, cfg->prio_comm, &s_comm));
    else s_comm = s_comp;

    RA_TRY(ensure_events(g_cache.dep_events, (size_t)n + 2, cudaEventDisableTiming));
    RA_TRY(ensure_events(g_cache.timed_events, 2 + (rec ? 4 * (size_t)n : 0), cudaEventDefault));
    cudaEvent_t ev_start = g_cache.timed_events[0], ev_end = g_cache.timed_events[1];
    auto kev = [&](int i, int which) { return g_cache.timed_events[2 + 4 * (size_t)i + which]; };
    cudaEvent_t ev_comm_done = g_cache.dep_events[n];

    ra_gemm_plan plan{};
    RA_CUDA(cudaEventRecord(ev_start, s_comp));
    if (overlap) RA_CUDA(cudaStreamWaitEvent(s_comm, ev_start, 0));
    for (int i = 0; i < n; ++i) {
        if (has_gemm) {
            if (rec) RA_CUDA(cudaEventRecord(kev(i, 0), s_comp));
            RA_TRY(gemm_launch(w->transA, w->transB, w->M, w->N, w->K, w->alpha, w->A, w->lda, w->B, w->ldb, w->beta,
                               w->C, w->ldc, &cfg->occ, w->workspace, w->workspace_bytes, s_comp, &plan));
            if (rec) RA_CUDA(cudaEventRecord(kev(i, 1), s_comp));
        }
        if (has_coll) {
            if (overlap && cfg->dependent && has_gemm) {
                RA_CUDA(cudaEventRecord(g_cache.dep_events[i], s_comp));
                RA_CUDA(cudaStreamWaitEvent(s_comm, g_cache.dep_events[i], 0));
            }
            if (rec) RA_CUDA(cudaEventRecord(kev(i, 2), s_comm));
            RA_TRY(launch_coll(w, cfg, i, s_comm));
            if (rec) RA_CUDA(cudaEventRecord(kev(i, 3), s_comm));
        }
    }
    if (overlap) {
        RA_CUDA(cudaEventRecord(ev_comm_done, s_comm));
        RA_CUDA(cudaStreamWaitEvent(s_comp, ev_comm_done, 0));
    }
    RA_CUDA(cudaEventRecord(ev_end, s_comp));
    RA_CUDA(cudaEventSynchronize(ev_end));
    RA_CUDA(cudaGetLastError());

    float total = 0.f;
    RA_CUDA(cudaEventElapsedTime(&total, ev_start, ev_end));
    res->total_ms = res->median_ms = res->min_ms = total;
    res->plan = plan;
    res->gemm_ms_sum = res->coll_ms_sum = 0.f;
    res->overlap_rate = 0.f;
    if (rec) {
        std::vector<float> t(4 * (size_t)n, 0.f);
        for (int i = 0; i < n; ++i) {
            if (has_gemm) {
                RA_CUDA(cudaEventElapsedTime(&t[4 * i + 0], ev_start, kev(i, 0)));
                RA_CUDA(cudaEventElapsedTime(&t[4 * i + 1], ev_start, kev(i, 1)));
            }
            if (has_coll) {
                RA_CUDA(cudaEventElapsedTime(&t[4 * i + 2], ev_start, kev(i, 2)));
                RA_CUDA(cudaEventElapsedTime(&t[4 * i + 3], ev_start, kev(i, 3)));
            }
        }
        // overlap rate: fraction of communication time concurrent with computation.
        // The GEMM intervals are disjoint (one stream), so the union is a plain sum.
        double csum = 0.0, gsum = 0.0, both = 0.0;
        for (int i = 0; i < n; ++i) {
            gsum += t[4 * i + 1] - t[4 * i + 0];
            csum += t[4 * i + 3] - t[4 * i + 2];
            for (int j = 0; j < n && has_gemm && has_coll; ++j) {
                const double lo = std::max(t[4 * i + 2], t[4 * j + 0]), hi = std::min(t[4 * i + 3], t[4 * j + 1]);
                if (hi > lo) both += hi - lo;
            }
        }
        res->gemm_ms_sum = (float)gsum;
        res->coll_ms_sum = (float)csum;
        res->overlap_rate = csum > 0.0 ? (float)(both / csum) : 0.f;
        if (res->kernel_times)
            for (size_t k = 0; k < t.size(); ++k) res->kernel_times[k] = t[k];
    }
    return RA_OK;
}

}  // namespace ra

extern "C" {

ra_status ra_overlap_run(const ra_workload* w, const ra_overlap_cfg* cfg, ra_overlap_result* res) {
    RA_TRY(ra::validate(w, cfg, res));
    return ra::run_once(w, cfg, res);
}

ra_status ra_overlap_sweep(const ra_workload* w, const ra_overlap_cfg* cfgs, int n, int runs, ra_overlap_result* results,
                           int* best) {
    if (cfgs == nullptr || results == nullptr || n < 1 || runs < 1) return RA_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) RA_TRY(ra::validate(w, &cfgs[i], &results[i]));
    const int warm = runs / 3;   // first third of the runs is warm-up
    std::vector<std::vector<float>> samples((size_t)n);
    for (int r = 0; r < runs; ++r) {
        for (int i = 0; i < n; ++i) {
            ra_overlap_result one = results[i];
            ra_overlap_cfg c = cfgs[i];
            // per-kernel events only on the last pass, so they cannot perturb the timed passes
            c.record_kernel_times = (r == runs - 1) ? cfgs[i].record_kernel_times : 0;
            RA_TRY(ra::run_once(w, &c, &one));
            if (r >= warm && !(c.record_kernel_times && runs - warm > 1)) samples[i].push_back(one.total_ms);
            if (r == runs - 1) {
                float* kt = results[i].kernel_times;
                results[i] = one;
                results[i].kernel_times = kt;
            }
        }
    }
    int arg = -1;
    bool any_overlap = false;
    for (int i = 0; i < n; ++i) any_overlap |= (cfgs[i].mode == RA_MODE_OVERLAP);
    for (int i = 0; i < n; ++i) {
        std::vector<float>& s = samples[i];
        std::sort(s.begin(), s.end());
        double sum = 0.0;
        for (float v : s) sum += v;
        results[i].total_ms = (float)(sum / (double)s.size());
        results[i].median_ms = s[s.size() / 2];
        results[i].min_ms = s[0];
        if (any_overlap && cfgs[i].mode != RA_MODE_OVERLAP) continue;
        if (arg < 0 || results[i].total_ms < results[arg].total_ms) arg = i;
    }
    if (best) *best = arg;
    return RA_OK;
}

void ra_shutdown(void) {
    std::lock_guard<std::mutex> lk(ra::g_cache.mu);
    for (auto& kv : ra::g_cache.streams) cudaStreamDestroy(kv.second);
    ra::g_cache.streams.clear();
    for (cudaEvent_t e : ra::g_cache.dep_events) cudaEventDestroy(e);
    for (cudaEvent_t e : ra::g_cache.timed_events) cudaEventDestroy(e);
    ra::g_cache.dep_events.clear();
    ra::g_cache.timed_events.clear();
}

}  // extern "C"
