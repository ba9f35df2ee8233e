// C ABI of libpairhmm_b200.so (include/pairhmm_b200.h): context, workspaces, launch orchestration.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <new>
#include <vector>

#include "../../include/pairhmm_b200.h"
#include "phmm_batcher.h"
#include "phmm_kernels.h"

using namespace phmm;

namespace {

struct DevBuf {  // grow-only device buffer
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t need(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaError_t e = cudaFree(p); p = nullptr; cap = 0; if (e != cudaSuccess) return e; }
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) { e = cudaMalloc(&p, bytes); want = bytes; }
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};
struct PinBuf {  // grow-only pinned host staging buffer
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t need(size_t bytes) {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaFreeHost(p); p = nullptr; cap = 0; }
        size_t want = bytes + bytes / 8 + 256;
        cudaError_t e = cudaMallocHost(&p, want);
        if (e == cudaSuccess) cap = want;
        return e;
    }
    void release() { if (p) cudaFreeHost(p); p = nullptr; cap = 0; }
};

}  // namespace

struct DeviceGuard {  // makes `device` current for the duration of an API call, then restores the caller's device
    int prev = -1;
    bool ok = false;
    explicit DeviceGuard(int device) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        ok = (prev == device) || cudaSetDevice(device) == cudaSuccess;
        if (prev == device) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

struct phmm_ctx {
    int device = 0;
    int n_sm = 0;
    phmm_options opt;
    phmm_stats stats;
    int last_cuda = 0;
    // The read-only plan arrays of a call live in one of two sets, uploaded on a copy stream of the context: the
    // uploads of call s+1 overlap the kernels of call s.  A set (and its pinned staging buffer) is reused once the
    // call that used it two calls ago has completed (ev_free, recorded on the caller's stream at the end of a call).
    struct PlanSet {
        DevBuf d_read_off, d_hap_off, d_pair_read, d_pair_hap, d_tasks, d_warp_first, d_srt_ent, d_srt_out, d_items, d_rq_enq;
        PinBuf h_stage;
        cudaEvent_t ev_free = nullptr, ev_up = nullptr;
        bool used = false;
    } set[2];
    int call_idx = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_last = nullptr;  // end of the device work of the most recent call: the next call's stream waits for it,
                                    // because the table, the counters, the queues and the boundary buffers exist once per context
    DevBuf d_lut, d_table;
    DevBuf d_counters, d_rescue, d_boundary, d_progress, d_scratch, d_totals;
    DevBuf d_rq, d_rq_queue, d_rq_sorted, d_rq_plan;  // fp64 sub-warp recomputation: counters, queue, ordered queue, plan, FP64-mode input list
    DevBuf d_payload, d_out, d_flags;  // phmm_forward_batch_host only
    std::vector<uint8_t> is_short;
    ShortPlan plan;
    int chain_grid[2] = {0, 0};  // resident CTAs of the fp64 chain kernel ([1]; [0] unused)
    int long_grid = 0, rescue_grid = 0;  // resident CTAs of the fp32 long kernel / of the fp64 sub-warp kernel on this device
    cudaEvent_t ev_prof[8] = {};   // profile_events: [2f], [2f+1] bracket family f (0 table, 1 short, 2 rescue, 3 long)
    bool prof_used[4] = {false, false, false, false};
    bool reuse_table = false;    // host entry, chunks after the first: the row-constant table of this payload is already on the device
    bool stats_final = false;    // host entry: n_rescued was counted from the flags, do not re-read the device counters
};

#define CK(call)                                                    \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) { ctx->last_cuda = (int)e__; return e__ == cudaErrorMemoryAllocation ? PHMM_E_NOMEM : PHMM_E_CUDA; } \
    } while (0)

#define RC(call) do { int rc__ = (call); if (rc__ != PHMM_OK) return rc__; } while (0)

extern "C" const char* phmm_strerror(int code) {
    switch (code) {
        case PHMM_OK: return "ok";
        case PHMM_E_ARG: return "invalid argument";
        case PHMM_E_OFFSETS: return "offsets not monotone or pair index out of range";
        case PHMM_E_EMPTY: return "pair references an empty read or haplotype";
        case PHMM_E_TOOLONG: return "sequence or batch too long";
        case PHMM_E_CUDA: return "CUDA error";
        case PHMM_E_NOMEM: return "out of memory";
        case PHMM_E_UNSUPPORTED: return "unsupported device or option";
        default: return "unknown error";
    }
}

extern "C" int phmm_create(phmm_ctx** out, int device, const phmm_options* opt) {
    if (!out) return PHMM_E_ARG;
    *out = nullptr;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return PHMM_E_CUDA;
    if (prop.major != 10) return PHMM_E_UNSUPPORTED;
    DeviceGuard guard(device);
    if (!guard.ok) return PHMM_E_CUDA;
    phmm_ctx* ctx = new (std::nothrow) phmm_ctx();
    if (!ctx) return PHMM_E_NOMEM;
    ctx->device = device;
    ctx->n_sm = prop.multiProcessorCount;
    memset(&ctx->opt, 0, sizeof(ctx->opt));
    if (opt) memcpy(&ctx->opt, opt, opt->size < sizeof(phmm_options) ? opt->size : sizeof(phmm_options));
    if (ctx->opt.rescue_log2_threshold == 0) ctx->opt.rescue_log2_threshold = -90;
    if (ctx->opt.long_min_hap_len <= 0 || ctx->opt.long_min_hap_len > SHORT_MAX_K) ctx->opt.long_min_hap_len = SHORT_MAX_K;
    if (ctx->opt.max_table_bytes <= 0) ctx->opt.max_table_bytes = (int64_t)64 << 30;
    if (ctx->opt.profile_events)
        for (int i = 0; i < 8; i++)
            if (cudaEventCreate(&ctx->ev_prof[i]) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    memset(&ctx->stats, 0, sizeof(ctx->stats));
    if (cudaEventCreateWithFlags(&ctx->ev_last, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    for (int i = 0; i < 2; i++)
        if (cudaEventCreateWithFlags(&ctx->set[i].ev_free, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ctx->set[i].ev_up, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    if (cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    // 10^(-q/10) for q = 0..255, the paper's "q64" table
    double lut[256];
    for (int q = 0; q < 256; q++) lut[q] = pow(10.0, -(double)q / 10.0);
    if (ctx->d_lut.need(sizeof(lut)) != cudaSuccess || cudaMemcpy(ctx->d_lut.p, lut, sizeof(lut), cudaMemcpyHostToDevice) != cudaSuccess) {
        phmm_destroy(ctx);
        return PHMM_E_CUDA;
    }
    ctx->chain_grid[1] = chain_ctas_per_sm(true) * ctx->n_sm;
    ctx->long_grid = long_ctas_per_sm() * ctx->n_sm;
    ctx->rescue_grid = rescue_ctas_per_sm() * ctx->n_sm;
    *out = ctx;
    return PHMM_OK;
}

extern "C" int phmm_destroy(phmm_ctx* ctx) {
    if (!ctx) return PHMM_E_ARG;
    DeviceGuard guard(ctx->device);
    cudaDeviceSynchronize();
    DevBuf* bufs[] = {&ctx->d_lut, &ctx->d_table, &ctx->d_counters, &ctx->d_rescue, &ctx->d_boundary, &ctx->d_progress, &ctx->d_scratch, &ctx->d_totals,
                      &ctx->d_payload, &ctx->d_out, &ctx->d_flags, &ctx->d_rq, &ctx->d_rq_queue, &ctx->d_rq_sorted, &ctx->d_rq_plan};
    for (DevBuf* b : bufs) b->release();
    for (int i = 0; i < 2; i++) {
        phmm_ctx::PlanSet& ps = ctx->set[i];
        DevBuf* sb[] = {&ps.d_read_off, &ps.d_hap_off, &ps.d_pair_read, &ps.d_pair_hap, &ps.d_tasks, &ps.d_warp_first,
                        &ps.d_srt_ent, &ps.d_srt_out, &ps.d_items, &ps.d_rq_enq};
        for (DevBuf* b : sb) b->release();
        ps.h_stage.release();
        if (ps.ev_free) cudaEventDestroy(ps.ev_free);
        if (ps.ev_up) cudaEventDestroy(ps.ev_up);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_last) cudaEventDestroy(ctx->ev_last);
    for (int i = 0; i < 8; i++)
        if (ctx->ev_prof[i]) cudaEventDestroy(ctx->ev_prof[i]);
    delete ctx;
    return PHMM_OK;
}

extern "C" int phmm_get_stats(phmm_ctx* ctx, phmm_stats* out) {
    if (!ctx || !out) return PHMM_E_ARG;
    if (!ctx->stats_final && ctx->d_counters.p && ctx->stats.n_pairs > 0) {  // rescue count lives on the device until the caller has synchronised
        int n = 0;
        DeviceGuard guard(ctx->device);
        int rq[16];
        if (cudaMemcpy(&n, ctx->d_counters.p, sizeof(int), cudaMemcpyDeviceToHost) == cudaSuccess && ctx->d_rq.p &&
            cudaMemcpy(rq, (int*)ctx->d_rq.p + RESCUE_NB, sizeof(rq), cudaMemcpyDeviceToHost) == cudaSuccess && ctx->stats.n_short_warps > 0)
            ctx->stats.n_rescued = (int64_t)n + rq[RQ_NQUEUE - RESCUE_NB] - rq[RQ_FALLBACK - RESCUE_NB];  // chain-kernel queue + sub-warp queue - passed on from one to the other
    }
    if (ctx->opt.profile_events) {
        double* dst[4] = {&ctx->stats.ms_table, &ctx->stats.ms_short, &ctx->stats.ms_rescue, &ctx->stats.ms_long};
        for (int f = 0; f < 4; f++) {
            float ms = 0.f;
            if (ctx->prof_used[f] && cudaEventSynchronize(ctx->ev_prof[2 * f + 1]) == cudaSuccess &&
                cudaEventElapsedTime(&ms, ctx->ev_prof[2 * f], ctx->ev_prof[2 * f + 1]) == cudaSuccess)
                *dst[f] = ms;
        }
    }
    *out = ctx->stats;
    return PHMM_OK;
}

extern "C" int phmm_last_cuda_error(phmm_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

extern "C" int phmm_plan_host(const phmm_batch* b, int long_min_hap_len, int task_rows, int64_t* plan_counts, int32_t* warp_first,
                              int64_t cap_warps, int32_t* tasks, int64_t cap_tasks, int32_t* sorted_pair, int64_t cap_pairs) {
    if (!b || !plan_counts || b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    if (b->n_pairs > 0) RC(validate_batch(hv));
    if (long_min_hap_len <= 0 || long_min_hap_len > SHORT_MAX_K) long_min_hap_len = SHORT_MAX_K;
    if (task_rows <= 0) task_rows = 3072;
    std::vector<uint8_t> is_short((size_t)b->n_pairs, 0);
    for (int64_t p = 0; p < b->n_pairs; p++) {
        const int r = b->h_pair_read[p], h = b->h_pair_hap[p];
        const int64_t l = b->h_read_off[r + 1] - b->h_read_off[r], k = b->h_hap_off[h + 1] - b->h_hap_off[h];
        is_short[(size_t)p] = !(k > long_min_hap_len || l > 4096);
    }
    ShortPlan pl;
    plan_short(hv, is_short.data(), SHORT_N2, task_rows, &pl);
    const int64_t nw = (int64_t)pl.warp_first.size() - 1, nt = (int64_t)pl.tasks.size(), ns = (int64_t)pl.srt_out.size();
    plan_counts[0] = nw; plan_counts[1] = nt; plan_counts[2] = ns; plan_counts[3] = SHORT_N2;
    if (warp_first) { if (cap_warps < nw) return PHMM_E_NOMEM; memcpy(warp_first, pl.warp_first.data(), (size_t)(nw + 1) * 4); }
    if (tasks) {
        if (cap_tasks < nt) return PHMM_E_NOMEM;
        for (int64_t i = 0; i < nt; i++) {
            tasks[4 * i] = pl.tasks[(size_t)i].hap; tasks[4 * i + 1] = pl.tasks[(size_t)i].pair_first;
            tasks[4 * i + 2] = pl.tasks[(size_t)i].n_pairs; tasks[4 * i + 3] = pl.tasks[(size_t)i].rows;
        }
    }
    if (sorted_pair) { if (cap_pairs < ns) return PHMM_E_NOMEM; memcpy(sorted_pair, pl.srt_out.data(), (size_t)ns * 4); }
    return PHMM_OK;
}

// ---------------------------------------------------------------- staging helper
namespace {
struct Stager {  // packs several host arrays into the pinned buffer and copies them with one memcpy each
    phmm_ctx* ctx;
    PinBuf* stage;
    cudaStream_t st;
    size_t used = 0;
    int upload(DevBuf& dst, const void* src, size_t bytes) {
        if (bytes == 0) return PHMM_OK;
        CK(dst.need(bytes));
        const size_t at = (used + 255) & ~(size_t)255;
        if (at + bytes > stage->cap) return PHMM_E_NOMEM;
        memcpy((char*)stage->p + at, src, bytes);
        used = at + bytes;
        CK(cudaMemcpyAsync(dst.p, (char*)stage->p + at, bytes, cudaMemcpyHostToDevice, st));
        return PHMM_OK;
    }
};
}  // namespace

#define PROF(f, second) do { if (ctx->opt.profile_events) { CK(cudaEventRecord(ctx->ev_prof[2 * (f) + (second)], st)); ctx->prof_used[f] = true; } } while (0)

extern "C" int phmm_forward_batch(phmm_ctx* ctx, const phmm_batch* b, int precision, double* d_out, uint8_t* d_flags,
                                  void* cuda_stream) {
    if (!ctx || !b) return PHMM_E_ARG;
    if (precision != PHMM_FP32_RESCUE && precision != PHMM_FP64) return PHMM_E_ARG;
    if (b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    memset(&ctx->stats, 0, sizeof(ctx->stats));
    ctx->stats_final = false;
    for (int f = 0; f < 4; f++) ctx->prof_used[f] = false;
    if (b->n_pairs == 0) return PHMM_OK;
    if (!d_out || !b->d_read_bases || !b->d_qual_base || !b->d_qual_ins || !b->d_qual_del || !b->d_qual_gcp || !b->d_hap_bases)
        return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    RC(validate_batch(hv));
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return PHMM_E_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const auto t0 = std::chrono::steady_clock::now();
    const bool fp64 = precision == PHMM_FP64;
    const int64_t np = b->n_pairs;

    // ---- classify: short (sub-warp systolic fp32 kernel) / chain-sequential (one warp per pair) / chain-strips
    const int strip_cols = chain_strip_cols(fp64);
    if (ctx->is_short.size() != (size_t)np) ctx->is_short.resize((size_t)np);
    std::vector<int> seq_pairs, strip_pairs, sub_pairs;  // chain kernel work lists, fp64 sub-warp list (caller pair indices)
    int64_t cells = 0, long_cells = 0, lane_rows = 0;  // lane_rows: sum over short pairs of read rows x lanes of the group
    int max_seq_l = 0, max_long_l = 0;  // longest read of the short class / of the long pairs
    {
        struct Part { std::vector<int> seq, strip, sub; int64_t cells = 0, long_cells = 0, lane_rows = 0; int max_l = 0, max_l_long = 0; };
        Part part[BATCHER_THREADS];
        const int long_k = ctx->opt.long_min_hap_len;
        uint8_t* is_short = ctx->is_short.data();
        const int T = parallel_chunks(np, 1 << 16, [&](int t, int64_t lo, int64_t hi) {
            Part& q = part[t];
            for (int64_t p = lo; p < hi; p++) {
                const int r = b->h_pair_read[p], h = b->h_pair_hap[p];
                const int64_t l = b->h_read_off[r + 1] - b->h_read_off[r], k = b->h_hap_off[h + 1] - b->h_hap_off[h];
                q.cells += l * k;
                uint8_t sh = 0;
                if (k > long_k || l > 4096) { q.strip.push_back((int)p); q.long_cells += l * k; if (l > q.max_l_long) q.max_l_long = (int)l; }
                else {
                    if (fp64 && k <= RESCUE_MAX_K && l <= RESCUE_MAX_L) q.sub.push_back((int)p);
                    else if (fp64) q.seq.push_back((int)p);
                    else { sh = 1; q.lane_rows += l * ((k + SHORT_N2 - 1) / SHORT_N2); }
                    if (l > q.max_l) q.max_l = (int)l;
                }
                is_short[p] = sh;
            }
        });
        for (int t = 0; t < T; t++) {  // chunks are contiguous and in order: the lists stay sorted by pair index
            seq_pairs.insert(seq_pairs.end(), part[t].seq.begin(), part[t].seq.end());
            strip_pairs.insert(strip_pairs.end(), part[t].strip.begin(), part[t].strip.end());
            sub_pairs.insert(sub_pairs.end(), part[t].sub.begin(), part[t].sub.end());
            cells += part[t].cells; long_cells += part[t].long_cells; lane_rows += part[t].lane_rows;
            if (part[t].max_l > max_seq_l) max_seq_l = part[t].max_l;
            if (part[t].max_l_long > max_long_l) max_long_l = part[t].max_l_long;
        }
    }
    ctx->stats.n_pairs = np;
    ctx->stats.cells = cells;
    ctx->stats.n_long_pairs = (int64_t)strip_pairs.size();
    ctx->stats.n_short_pairs = np - (int64_t)strip_pairs.size();
    // task size: as large as possible (fewer run-ins, pipeline fills and host work; 8192 rows measured best on
    // configs[1]) while leaving at least ~6 warps of work per resident warp slot
    int task_rows = ctx->opt.task_rows;
    if (task_rows <= 0) {
        const int64_t slots = (int64_t)ctx->n_sm * 12;
        task_rows = (int)std::max<int64_t>(1024, std::min<int64_t>(8192, lane_rows / 32 / (6 * slots)));
    }
    if (!fp64) plan_short(hv, ctx->is_short.data(), SHORT_N2, task_rows, &ctx->plan);
    else { ctx->plan.tasks.clear(); ctx->plan.warp_first.assign(1, 0); ctx->plan.srt_out.clear(); ctx->plan.srt_ent.clear(); ctx->plan.cells = 0; ctx->plan.padded_cells = 0; }
    const ShortPlan& pl = ctx->plan;
    const int n_warps = (int)pl.warp_first.size() - 1;
    ctx->stats.short_cells = pl.cells;
    ctx->stats.short_padded_cells = pl.padded_cells;
    ctx->stats.n_short_warps = n_warps;

    // ---- strip items of the long pairs, STRIP-major: strip s of every pair before strip s+1 of any.  A strip's
    // producer still holds an earlier ticket (forward progress), but it is far ahead or done by the time the
    // consumer starts, so consumers do not run in lock step with their producers and hardly ever poll (pair-major
    // order: 4.6 polls per step, 19 % of the stall samples; profiles/).  Boundary buffers are full-length per strip.
    std::vector<ChainItem> items;
    int64_t n_bnd_blocks = 0;
    int n_prog = 0;
    {
        struct PairStrips { int pair, ns, prog0; int64_t buf0; };
        std::vector<PairStrips> ps;
        ps.reserve(strip_pairs.size());
        int max_ns = 0;
        size_t total = 0;
        for (int p : strip_pairs) {
            const int r = b->h_pair_read[p], h = b->h_pair_hap[p];
            const int64_t l = b->h_read_off[r + 1] - b->h_read_off[r], k = b->h_hap_off[h + 1] - b->h_hap_off[h];
            const int ns = (int)((k + strip_cols - 1) / strip_cols);
            // fp64 chain kernel: 32-row boundary blocks; fp32 long kernel: one 16-byte record per stream entry
            const int64_t nblk = fp64 ? (l + CHAIN_EXTRA_ROWS + 31) / 32 : l + TABLE_EXTRA_ROWS;
            ps.push_back(PairStrips{p, ns, n_prog, n_bnd_blocks});
            n_bnd_blocks += (int64_t)(ns > 1 ? ns - 1 : 0) * nblk;
            n_prog += ns;  // one counter per strip (the last one is unused)
            if (ns > max_ns) max_ns = ns;
            total += (size_t)ns;
        }
        items.reserve(total);
        for (int s = 0; s < max_ns; s++)
            for (const PairStrips& q : ps)
                if (s < q.ns) items.push_back(ChainItem{q.pair, s, q.prog0, 0, q.buf0});
    }
    const auto t1 = std::chrono::steady_clock::now();
    ctx->stats.host_batch_ms = std::chrono::duration<double, std::milli>(t1 - t0).count();

    // ---- uploads.  The plan arrays go to this call's plan set on the context's copy stream (overlapping the kernels
    // of the previous call, which read the other set); the small per-call counters and lists that kernels also write
    // stay on the caller's stream.
    phmm_ctx::PlanSet& ps = ctx->set[ctx->call_idx & 1];
    ctx->call_idx++;
    if (ps.used) CK(cudaEventSynchronize(ps.ev_free));  // the call that used this set (two calls ago) has completed
    const size_t n_seq = fp64 ? seq_pairs.size() : 0;
    size_t stage_bytes = 4096 + (size_t)(b->n_reads + 1) * 8 + (size_t)(b->n_haps + 1) * 8 + (size_t)np * 8 +
                         pl.tasks.size() * sizeof(ShortTask) + pl.warp_first.size() * 4 + pl.srt_out.size() * 16 +
                         items.size() * sizeof(ChainItem) + n_seq * 4 + sub_pairs.size() * 4 + 20 * 256;
    CK(ps.h_stage.need(stage_bytes));
    Stager sg{ctx, &ps.h_stage, ctx->copy_stream};
    RC(sg.upload(ps.d_read_off, b->h_read_off, (size_t)(b->n_reads + 1) * 8));
    RC(sg.upload(ps.d_hap_off, b->h_hap_off, (size_t)(b->n_haps + 1) * 8));
    RC(sg.upload(ps.d_pair_read, b->h_pair_read, (size_t)np * 4));
    RC(sg.upload(ps.d_pair_hap, b->h_pair_hap, (size_t)np * 4));
    RC(sg.upload(ps.d_tasks, pl.tasks.data(), pl.tasks.size() * sizeof(ShortTask)));
    RC(sg.upload(ps.d_warp_first, pl.warp_first.data(), pl.warp_first.size() * 4));
    RC(sg.upload(ps.d_srt_ent, pl.srt_ent.data(), pl.srt_ent.size() * 4));
    RC(sg.upload(ps.d_srt_out, pl.srt_out.data(), pl.srt_out.size() * 4));
    RC(sg.upload(ps.d_items, items.data(), items.size() * sizeof(ChainItem)));
    RC(sg.upload(ps.d_rq_enq, sub_pairs.data(), sub_pairs.size() * 4));
    CK(cudaEventRecord(ps.ev_up, ctx->copy_stream));
    CK(cudaStreamWaitEvent(st, ps.ev_up, 0));
    CK(cudaStreamWaitEvent(st, ctx->ev_last, 0));  // calls on different streams of one context run one after the other
    // counters: [0] rescue count (= n_items of the rescue launch)  [1] ticket rescue  [2] n strip items  [3] ticket strips
    //           [4] n sequential fp64 items  [5] ticket sequential
    sg.st = st;  // from here on: buffers that kernels write as well, in stream order with them
    int h_counters[8] = {0, 0, (int)items.size(), 0, (int)n_seq, 0, 0, 0};
    RC(sg.upload(ctx->d_counters, h_counters, sizeof(h_counters)));
    // rescue list (fp32 mode: filled by the short kernel) / sequential list (fp64 mode: all non-long pairs)
    CK(ctx->d_rescue.need((size_t)np * 4 + 4));
    RC(sg.upload(ctx->d_rescue, seq_pairs.data(), n_seq * 4));
    CK(ctx->d_rq.need(RQ_INTS * 4));
    CK(ctx->d_rq_plan.need(RESCUE_PLAN_INTS * 4));
    CK(ctx->d_rq_queue.need((size_t)np * 16 + 16));
    CK(ctx->d_rq_sorted.need((size_t)np * 4 + 4));
    CK(cudaMemsetAsync(ctx->d_rq.p, 0, RQ_INTS * 4, st));
    ps.used = true;
    struct FreeMark {  // whatever path leaves the call: the set is free once everything enqueued so far on st has run
        cudaEvent_t ev, ev_last; cudaStream_t st;
        ~FreeMark() { cudaEventRecord(ev, st); cudaEventRecord(ev_last, st); }
    } free_mark{ps.ev_free, ctx->ev_last, st};

    DevBatch db;
    db.read_bases = b->d_read_bases; db.qual_base = b->d_qual_base; db.qual_ins = b->d_qual_ins;
    db.qual_del = b->d_qual_del; db.qual_gcp = b->d_qual_gcp; db.hap_bases = b->d_hap_bases;
    db.read_off = (const int64_t*)ps.d_read_off.p; db.hap_off = (const int64_t*)ps.d_hap_off.p;
    db.n_reads = b->n_reads; db.n_haps = b->n_haps;
    int* counters = (int*)ctx->d_counters.p;
    int launches = 0;

    // ---- fp32: row-constant table of every read (short and long pairs use the same one)
    const bool long32 = !fp64 && !items.empty();
    if (n_warps > 0 || long32) {
        const int64_t n_entries = table_run_start(b->h_read_off[b->n_reads], b->n_reads) + 2;
        if (n_entries > INT32_MAX) return PHMM_E_TOOLONG;
        const size_t table_bytes = (size_t)(n_entries + 192) * 64;  // (slack: the long kernel prefetches up to 96 entries past a run)
        if ((int64_t)table_bytes > ctx->opt.max_table_bytes) return PHMM_E_NOMEM;
        CK(ctx->d_table.need(table_bytes));
        ctx->stats.table_bytes = (int64_t)table_bytes;
        PROF(0, 0);
        if (!ctx->reuse_table)
            CK(launch_lut_table(db, (const double*)ctx->d_lut.p, (float*)ctx->d_table.p, std::max(max_seq_l, max_long_l), st));
        PROF(0, 1);
        launches++;
    }
    // ---- short path: systolic kernel, then (below) fp64 rescue of what underflowed
    if (n_warps > 0) {
        ShortLaunch sl;
        sl.table = (const float*)ctx->d_table.p;
        sl.tasks = (const ShortTask*)ps.d_tasks.p;
        sl.warp_first = (const int*)ps.d_warp_first.p;
        sl.n_warps = n_warps;
        sl.srt_ent = (const int2*)ps.d_srt_ent.p;
        sl.srt_out = (const int*)ps.d_srt_out.p;
        sl.out = d_out;
        sl.flags = d_flags;
        sl.rescue_thr = (float)ldexp(1.0, ctx->opt.rescue_log2_threshold);
        sl.rescue.queue = (int4*)ctx->d_rq_queue.p;
        sl.rescue.cnt = (int*)ctx->d_rq.p;
        sl.pair_read = (const int*)ps.d_pair_read.p;
        sl.rescue_count = counters + 0;
        sl.rescue_list = (int*)ctx->d_rescue.p;
        PROF(1, 0);
        CK(launch_short_f32(db, sl, st));
        PROF(1, 1);
        launches++;
    }
    // ---- long path.  fp32: table-driven strips with per-lane exponents (phmm_long.cu); what it cannot represent joins
    // the rescue list of the fp64 chain launch below.  fp64: concurrent strips of the chain kernel.
    if (!items.empty()) {
        CK(ctx->d_progress.need((size_t)n_prog * 4 + 4));
        CK(cudaMemsetAsync(ctx->d_progress.p, 0, (size_t)n_prog * 4 + 4, st));
        // no more CTAs than there are strips: with fewer strips than resident warps the block scheduler would fill
        // some SMs completely and leave others empty (configs[4]: 1648 strips, 2368 slots: 1.36 vs 1.76 TCUPS)
        const int wpc = fp64 ? chain_warps_per_cta(true) : long_warps_per_cta();
        const int need_ctas = (int)((items.size() + (size_t)wpc - 1) / (size_t)wpc);
        PROF(3, 0);
        if (fp64) {
            CK(ctx->d_boundary.need((size_t)(n_bnd_blocks + 1) * chain_block_bytes(true)));
            ChainLaunch cl;
            memset(&cl, 0, sizeof(cl));
            cl.items = (const ChainItem*)ps.d_items.p;
            cl.n_items = counters + 2;
            cl.ticket = counters + 3;
            cl.pair_read = (const int*)ps.d_pair_read.p;
            cl.pair_hap = (const int*)ps.d_pair_hap.p;
            cl.lut = (const double*)ctx->d_lut.p;
            cl.boundary = ctx->d_boundary.p;
            cl.scratch_blocks = 0;
            cl.progress = (int*)ctx->d_progress.p;
            cl.out = d_out;
            cl.flags = d_flags;
            cl.flag_bits = PHMM_FLAG_LONG;
            cl.log2C = 0;
            CK(launch_chain(db, cl, true, false, std::min(ctx->chain_grid[1], need_ctas), st));
        } else {
            CK(ctx->d_boundary.need((size_t)(n_bnd_blocks + 1) * 16));
            CK(ctx->d_totals.need((size_t)n_prog * 16 + 16));
            LongLaunch ll;
            memset(&ll, 0, sizeof(ll));
            ll.table = (const float*)ctx->d_table.p;
            ll.items = (const ChainItem*)ps.d_items.p;
            ll.n_items = counters + 2;
            ll.ticket = counters + 3;
            ll.pair_read = (const int*)ps.d_pair_read.p;
            ll.pair_hap = (const int*)ps.d_pair_hap.p;
            ll.records = (float4*)ctx->d_boundary.p;
            ll.totals = (float4*)ctx->d_totals.p;
            ll.progress = (int*)ctx->d_progress.p;
            ll.out = d_out;
            ll.flags = d_flags;
            ll.flag_bits = PHMM_FLAG_LONG;
            // every strip resident at once (configs[4]): the wavefront's pipeline depth decides, publish often;
            // many more strips than warp slots: a consumer hardly ever waits, publish (MEMBAR) rarely
            ll.publish = need_ctas <= ctx->long_grid ? 16 : 64;
            ll.fallback_count = counters + 0;
            ll.fallback_list = (int*)ctx->d_rescue.p;
            CK(launch_long_f32(db, ll, std::min(ctx->long_grid, need_ctas), st));
        }
        PROF(3, 1);
        launches++;
    }
    // fp64 sub-warp kernel: fp32 mode = what the short kernel queued, fp64 mode = the short pairs it can hold
    const bool sub = n_warps > 0 || !sub_pairs.empty();
    if (sub) {
        RescueLaunch rl;
        memset(&rl, 0, sizeof(rl));
        rl.queue.queue = (int4*)ctx->d_rq_queue.p;
        rl.queue.cnt = (int*)ctx->d_rq.p;
        rl.table = fp64 ? nullptr : (const float*)ctx->d_table.p;
        rl.max_queue = (int)(fp64 ? (int64_t)sub_pairs.size() : ctx->stats.n_short_pairs);
        rl.enqueue_pairs = fp64 ? (const int*)ps.d_rq_enq.p : nullptr;
        rl.n_enqueue = fp64 ? (int)sub_pairs.size() : 0;
        rl.plan = (int*)ctx->d_rq_plan.p;
        rl.sorted = (int*)ctx->d_rq_sorted.p;
        rl.pair_read = (const int*)ps.d_pair_read.p;
        rl.pair_hap = (const int*)ps.d_pair_hap.p;
        rl.lut = (const double*)ctx->d_lut.p;
        rl.out = d_out;
        rl.flags = d_flags;
        rl.flag_bits = fp64 ? 0 : PHMM_FLAG_RESCUED;
        rl.fallback_count = counters + (fp64 ? 4 : 0);
        rl.fallback_list = (int*)ctx->d_rescue.p;
        PROF(2, 0);
        CK(launch_rescue_f64(db, rl, ctx->rescue_grid, st));
        launches += 3 + (fp64 ? 1 : 0);
    }
    // sequential chain launch (one warp per pair, its strips in sequence, fp64, rescaled): fp32 mode = the rescue list
    // (device-side count: short pairs too wide for the sub-warp kernel, what that kernel passed on, long pairs the fp32
    // long kernel could not represent), fp64 mode = the short-class pairs the sub-warp kernel does not take
    if (n_warps > 0 || n_seq > 0 || sub || long32) {
        int grid = ctx->chain_grid[1];
        const int max_l = long32 ? std::max(max_seq_l, max_long_l) : max_seq_l;
        const int64_t blocks = (max_l + CHAIN_EXTRA_ROWS + 31) / 32 + 1;
        const int max_strips_seq = long32 ? 2 : (ctx->opt.long_min_hap_len + chain_strip_cols(true) - 1) / chain_strip_cols(true);
        const size_t per_cta = (size_t)chain_warps_per_cta(true) * 2 * blocks * chain_block_bytes(true);  // ping-pong boundary buffers
        if (long32) grid = (int)std::max<size_t>(8, std::min<size_t>((size_t)grid, ((size_t)1 << 30) / per_cta));  // fallbacks of long pairs are rare: at most 1 GiB
        size_t scratch = max_strips_seq > 1 ? (size_t)grid * per_cta : 256;
        CK(ctx->d_scratch.need(scratch));
        ChainLaunch cl;
        memset(&cl, 0, sizeof(cl));
        cl.items = (const ChainItem*)ctx->d_rescue.p;
        cl.n_items = counters + (fp64 ? 4 : 0);
        cl.ticket = counters + (fp64 ? 5 : 1);
        cl.pair_read = (const int*)ps.d_pair_read.p;
        cl.pair_hap = (const int*)ps.d_pair_hap.p;
        cl.lut = (const double*)ctx->d_lut.p;
        cl.boundary = ctx->d_scratch.p;
        cl.scratch_blocks = blocks;
        cl.progress = nullptr;
        cl.out = d_out;
        cl.flags = d_flags;
        cl.flag_bits = fp64 ? 0 : PHMM_FLAG_RESCUED;
        cl.long_k = ctx->opt.long_min_hap_len;
        cl.log2C = 0;
        if (!sub) PROF(2, 0);
        CK(launch_chain(db, cl, true, true, grid, st));
        PROF(2, 1);
        launches++;
    }
    ctx->stats.n_kernel_launches = launches;
    ctx->stats.n_slices = 1;
    return PHMM_OK;
}

// ---------------------------------------------------------------- end-to-end entry with host buffers
extern "C" int phmm_forward_batch_host(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out, uint8_t* h_flags) {
    if (!ctx || !b) return PHMM_E_ARG;
    if (b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    if (b->n_pairs == 0) { memset(&ctx->stats, 0, sizeof(ctx->stats)); return PHMM_OK; }
    if (!h_out || !b->h_read_off || !b->h_hap_off) return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    RC(validate_batch(hv));
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return PHMM_E_CUDA;
    const size_t R = (size_t)b->h_read_off[b->n_reads], H = (size_t)b->h_hap_off[b->n_haps];
    const size_t Ra = (R + 255) & ~(size_t)255, Ha = (H + 255) & ~(size_t)255;
    CK(ctx->d_payload.need(5 * Ra + Ha + 256));
    CK(ctx->d_out.need((size_t)b->n_pairs * 8));
    CK(ctx->d_flags.need((size_t)b->n_pairs));
    uint8_t* base = (uint8_t*)ctx->d_payload.p;
    const uint8_t* src[5] = {b->d_read_bases, b->d_qual_base, b->d_qual_ins, b->d_qual_del, b->d_qual_gcp};
    cudaStream_t st = nullptr;
    for (int i = 0; i < 5; i++) {
        if (!src[i]) return PHMM_E_ARG;
        CK(cudaMemcpyAsync(base + i * Ra, src[i], R, cudaMemcpyHostToDevice, st));
    }
    if (!b->d_hap_bases) return PHMM_E_ARG;
    CK(cudaMemcpyAsync(base + 5 * Ra, b->d_hap_bases, H, cudaMemcpyHostToDevice, st));
    phmm_batch db = *b;
    db.d_read_bases = base; db.d_qual_base = base + Ra; db.d_qual_ins = base + 2 * Ra; db.d_qual_del = base + 3 * Ra;
    db.d_qual_gcp = base + 4 * Ra; db.d_hap_bases = base + 5 * Ra;
    // The pair list is processed in chunks: phmm_forward_batch only enqueues, so the host batcher of chunk c+1 runs
    // while the GPU works on chunk c, and each chunk's results start their way back as soon as it is done.  The
    // row-constant table depends on the payload only and is built with the first chunk.
    const int64_t np = b->n_pairs;
    int n_chunks = (int)std::max<int64_t>(1, std::min<int64_t>(8, np / 400000));
    if (n_chunks > 1) {  // only worth it if the chunks use disjoint haplotypes: a shuffled list would split every task
        int hmin[8], hmax[8];
        for (int c = 0; c < n_chunks; c++) {
            const int64_t lo = np * c / n_chunks, hi = np * (c + 1) / n_chunks;
            int mn = INT32_MAX, mx = -1;
            for (int64_t p = lo; p < hi; p++) { const int h = b->h_pair_hap[p]; mn = std::min(mn, h); mx = std::max(mx, h); }
            hmin[c] = mn; hmax[c] = mx;
        }
        for (int c = 0; c + 1 < n_chunks; c++)
            if (hmax[c] >= hmin[c + 1]) { n_chunks = 1; break; }
    }
    phmm_stats sum;
    memset(&sum, 0, sizeof(sum));
    int rc = PHMM_OK;
    for (int c = 0; c < n_chunks && rc == PHMM_OK; c++) {
        const int64_t lo = np * c / n_chunks, hi = np * (c + 1) / n_chunks;
        phmm_batch cb = db;
        cb.n_pairs = hi - lo;
        cb.h_pair_read = b->h_pair_read + lo;
        cb.h_pair_hap = b->h_pair_hap + lo;
        ctx->reuse_table = c > 0 && sum.n_short_warps > 0;
        rc = phmm_forward_batch(ctx, &cb, precision, (double*)ctx->d_out.p + lo, (uint8_t*)ctx->d_flags.p + lo, st);
        ctx->reuse_table = false;
        if (rc != PHMM_OK) break;
        const phmm_stats& t = ctx->stats;
        sum.n_pairs += t.n_pairs; sum.cells += t.cells; sum.n_short_pairs += t.n_short_pairs; sum.n_long_pairs += t.n_long_pairs;
        sum.short_cells += t.short_cells; sum.short_padded_cells += t.short_padded_cells; sum.n_short_warps += t.n_short_warps;
        sum.n_kernel_launches += t.n_kernel_launches; sum.host_batch_ms += t.host_batch_ms;
        if (t.table_bytes > sum.table_bytes) sum.table_bytes = t.table_bytes;
        if (cudaMemcpyAsync(h_out + lo, (double*)ctx->d_out.p + lo, (size_t)(hi - lo) * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = PHMM_E_CUDA;
    }
    if (rc != PHMM_OK) { cudaStreamSynchronize(st); return rc; }
    std::vector<uint8_t> tmp_flags;
    uint8_t* fl = h_flags;
    if (!fl) { tmp_flags.resize((size_t)np); fl = tmp_flags.data(); }
    CK(cudaMemcpyAsync(fl, ctx->d_flags.p, (size_t)np, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    sum.n_slices = n_chunks;
    for (int64_t p = 0; p < np; p++) sum.n_rescued += fl[p] & PHMM_FLAG_RESCUED;
    ctx->stats = sum;
    ctx->stats_final = true;
    return PHMM_OK;
}

