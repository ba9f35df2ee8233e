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
    // Read-only arrays live in double-buffered sets, uploaded on a copy stream of the context so that the uploads of the
    // next call / slice overlap the kernels of the current one.  A set (and its pinned staging buffer) is reused once the
    // work that used it two calls / slices ago has completed (ev_free, recorded on the caller's stream).
    struct CallSet {  // per call: the batch's offset arrays and pair list
        DevBuf d_read_off, d_hap_off, d_pair_read, d_pair_hap;
        PinBuf h_stage;
        cudaEvent_t ev_free = nullptr, ev_up = nullptr;
        bool used = false;
    } cset[2];
    struct PlanSet {  // per slice of a call: the work plan
        DevBuf d_tasks, d_warp_first, d_srt_ent, d_srt_out, d_items, d_rq_enq, d_seq;
        PinBuf h_stage;
        cudaEvent_t ev_free = nullptr, ev_up = nullptr;
        bool used = false;
    } set[2];
    int call_idx = 0, slice_idx = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_pay = nullptr;   // copy stream: a slice's read arrays (and everything uploaded before them) are on the device
    cudaEvent_t ev_last = nullptr;  // end of the device work of the most recent call: the next call's stream waits for it,
                                    // because the table, the counters, the queues and the boundary buffers exist once per context
    DevBuf d_lut, d_table;
    DevBuf d_counters, d_rescue, d_boundary, d_progress, d_scratch, d_totals, d_acc, d_risk;
    DevBuf d_rq, d_rq_queue, d_rq_sorted, d_rq_plan;  // fp64 sub-warp recomputation: counters, queue, ordered queue, plan
    // Host entries (phmm_forward_batch_host, phmm_forward_batch_host_async): two sets of device copies of the payload and of
    // the outputs, so that the copies and the host plan of one call run under the kernels of the call before it.
    struct HostSet {
        DevBuf d_payload, d_out, d_flags;
        PinBuf h_flags;              // where the caller passes no flags array
        cudaEvent_t done = nullptr;  // the call's outputs are in the caller's host arrays
        bool pending = false;
        int ticket = -1;
        int64_t np = 0;
        const uint8_t* fl = nullptr;
        phmm_stats stats;
    } hset[2];
    int host_calls = 0;
    cudaStream_t host_stream = nullptr;  // the kernels of the host entries
    std::vector<uint8_t> is_short, read_slice;
    std::vector<int> sorted_all, slice_ids, short_ids;
    ShortPlan plan;
    int chain_grid[2] = {0, 0};  // resident CTAs of the fp64 chain kernel ([1]; [0] unused)
    int long_grid = 0, rescue_grid = 0, long64_grid = 0;  // resident CTAs of the fp32 long kernel / of the fp64 sub-warp kernel on this device
    // profile_events: per slice s and kernel family f (0 table, 1 short, 2 rescue, 3 long) the events [8s + 2f], [8s + 2f + 1]
    std::vector<cudaEvent_t> ev_prof;
    std::vector<uint8_t> prof_used;  // [4s + f]
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
    if (ctx->opt.max_table_bytes <= 0) ctx->opt.max_table_bytes = (int64_t)4 << 30;
    memset(&ctx->stats, 0, sizeof(ctx->stats));
    if (cudaEventCreateWithFlags(&ctx->ev_last, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    if (cudaEventCreateWithFlags(&ctx->ev_pay, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    for (int i = 0; i < 2; i++)
        if (cudaEventCreateWithFlags(&ctx->set[i].ev_free, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ctx->set[i].ev_up, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ctx->cset[i].ev_free, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&ctx->cset[i].ev_up, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    if (cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    if (cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    for (int i = 0; i < 2; i++)
        if (cudaEventCreateWithFlags(&ctx->hset[i].done, cudaEventDisableTiming) != cudaSuccess) { phmm_destroy(ctx); return PHMM_E_CUDA; }
    // 10^(-q/10) for every quality byte, the paper's "q64" table: [0..255] for insertion, deletion and
    // continuation qualities, [256..511] for base qualities (with the optional floor), both after the optional offset
    if (ctx->opt.qual_offset < 0 || ctx->opt.qual_offset > 255 || ctx->opt.min_base_qual < 0) { phmm_destroy(ctx); return PHMM_E_ARG; }
    double lut[512];
    for (int q = 0; q < 256; q++) {
        const int v = std::max(0, q - ctx->opt.qual_offset);
        lut[q] = pow(10.0, -(double)v / 10.0);
        lut[256 + q] = pow(10.0, -(double)std::max(v, ctx->opt.min_base_qual) / 10.0);
    }
    if (ctx->d_lut.need(sizeof(lut)) != cudaSuccess || cudaMemcpy(ctx->d_lut.p, lut, sizeof(lut), cudaMemcpyHostToDevice) != cudaSuccess) {
        phmm_destroy(ctx);
        return PHMM_E_CUDA;
    }
    ctx->chain_grid[1] = chain_ctas_per_sm(true) * ctx->n_sm;
    ctx->long_grid = long_ctas_per_sm() * ctx->n_sm;
    ctx->rescue_grid = rescue_ctas_per_sm() * ctx->n_sm;
    ctx->long64_grid = long64_ctas_per_sm() * ctx->n_sm;
    *out = ctx;
    return PHMM_OK;
}

extern "C" int phmm_destroy(phmm_ctx* ctx) {
    if (!ctx) return PHMM_E_ARG;
    DeviceGuard guard(ctx->device);
    cudaDeviceSynchronize();
    DevBuf* bufs[] = {&ctx->d_lut, &ctx->d_table, &ctx->d_counters, &ctx->d_rescue, &ctx->d_boundary, &ctx->d_progress, &ctx->d_scratch, &ctx->d_totals, &ctx->d_acc, &ctx->d_risk,
                      &ctx->d_rq, &ctx->d_rq_queue, &ctx->d_rq_sorted, &ctx->d_rq_plan};
    for (DevBuf* b : bufs) b->release();
    for (int i = 0; i < 2; i++) {
        phmm_ctx::HostSet& hs = ctx->hset[i];
        hs.d_payload.release(); hs.d_out.release(); hs.d_flags.release(); hs.h_flags.release();
        if (hs.done) cudaEventDestroy(hs.done);
    }
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    for (int i = 0; i < 2; i++) {
        phmm_ctx::PlanSet& ps = ctx->set[i];
        DevBuf* sb[] = {&ps.d_tasks, &ps.d_warp_first, &ps.d_srt_ent, &ps.d_srt_out, &ps.d_items, &ps.d_rq_enq, &ps.d_seq};
        for (DevBuf* b : sb) b->release();
        ps.h_stage.release();
        if (ps.ev_free) cudaEventDestroy(ps.ev_free);
        if (ps.ev_up) cudaEventDestroy(ps.ev_up);
        phmm_ctx::CallSet& cs = ctx->cset[i];
        DevBuf* cb[] = {&cs.d_read_off, &cs.d_hap_off, &cs.d_pair_read, &cs.d_pair_hap};
        for (DevBuf* b : cb) b->release();
        cs.h_stage.release();
        if (cs.ev_free) cudaEventDestroy(cs.ev_free);
        if (cs.ev_up) cudaEventDestroy(cs.ev_up);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_last) cudaEventDestroy(ctx->ev_last);
    if (ctx->ev_pay) cudaEventDestroy(ctx->ev_pay);
    for (cudaEvent_t e : ctx->ev_prof)
        if (e) cudaEventDestroy(e);
    delete ctx;
    return PHMM_OK;
}

extern "C" int phmm_get_stats(phmm_ctx* ctx, phmm_stats* out) {
    if (!ctx || !out) return PHMM_E_ARG;
    if (!ctx->stats_final && ctx->d_acc.p && ctx->stats.n_pairs > 0) {  // the rescue count lives on the device until the call has completed
        DeviceGuard guard(ctx->device);
        if (ctx->ev_last) cudaEventSynchronize(ctx->ev_last);  // (the end of the call's device work, whatever stream it ran on)
        long long acc[2] = {0, 0};
        if (cudaMemcpy(acc, ctx->d_acc.p, sizeof(acc), cudaMemcpyDeviceToHost) == cudaSuccess) ctx->stats.n_rescued = (int64_t)acc[0];
    }
    if (ctx->opt.profile_events) {
        double* dst[4] = {&ctx->stats.ms_table, &ctx->stats.ms_short, &ctx->stats.ms_rescue, &ctx->stats.ms_long};
        for (int f = 0; f < 4; f++) *dst[f] = 0.0;
        for (size_t i = 0; i < ctx->prof_used.size(); i++) {  // summed over the slices of the call
            float ms = 0.f;
            if (ctx->prof_used[i] && cudaEventSynchronize(ctx->ev_prof[2 * i + 1]) == cudaSuccess &&
                cudaEventElapsedTime(&ms, ctx->ev_prof[2 * i], ctx->ev_prof[2 * i + 1]) == cudaSuccess)
                *dst[i & 3] += ms;
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
        is_short[(size_t)p] = !long_class(k, l, long_min_hap_len, long_min_hap_len * 7 / 8);  // (the PHMM_FP32_RESCUE classification)
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

extern "C" int phmm_plan_slices_host(const phmm_batch* b, int64_t max_table_bytes, int min_slices, int64_t* n_slices,
                                     int64_t* read_first, int64_t* pair_count, int64_t cap_slices) {
    if (!b || !n_slices || b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    if (b->n_pairs > 0) RC(validate_batch(hv));
    if (max_table_bytes <= 0) max_table_bytes = (int64_t)4 << 30;
    std::vector<int64_t> bound;
    const int ns = b->n_reads > 0 ? slice_reads(hv, max_table_bytes, min_slices, &bound) : 0;
    *n_slices = ns;
    if (read_first || pair_count) {
        if (cap_slices < ns) return PHMM_E_NOMEM;
        if (read_first) for (int s = 0; s <= ns; s++) read_first[s] = bound[(size_t)s];
        if (pair_count) {
            for (int s = 0; s < ns; s++) pair_count[s] = 0;
            for (int64_t p = 0; p < b->n_pairs; p++) {
                const int64_t r = b->h_pair_read[p];
                const int s = (int)(std::upper_bound(bound.begin(), bound.end(), r) - bound.begin()) - 1;
                pair_count[s]++;
            }
        }
    }
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
        if (bytes >= ((size_t)8 << 20)) {  // (plans of millions of tasks: 100 MB and more)
            char* d = (char*)stage->p + at;
            const char* s0 = (const char*)src;
            parallel_chunks((int64_t)bytes, 1 << 20, [&](int, int64_t lo, int64_t hi) { memcpy(d + lo, s0 + lo, (size_t)(hi - lo)); });
        } else {
            memcpy((char*)stage->p + at, src, bytes);
        }
        used = at + bytes;
        CK(cudaMemcpyAsync(dst.p, (char*)stage->p + at, bytes, cudaMemcpyHostToDevice, st));
        return PHMM_OK;
    }
};
}  // namespace

#define PROF(f, second) do { if (ctx->opt.profile_events) { CK(cudaEventRecord(ctx->ev_prof[8 * (size_t)sw.slice + 2 * (f) + (second)], st)); ctx->prof_used[4 * (size_t)sw.slice + (f)] = 1; } } while (0)

namespace {

__global__ void k_accumulate_rescued(long long* acc, const int* counters, const int* rq) {
    // chain-kernel queue + sub-warp queue - what the sub-warp kernel passed on to the chain kernel
    acc[0] += (long long)counters[0] + rq[RQ_NQUEUE] - rq[RQ_FALLBACK];
}

struct HostPayload {  // phmm_forward_batch_host: where the payload comes from (host) and goes to (device)
    const uint8_t* src[5];
    uint8_t* dst[5];
};

struct SliceWork {  // one slice of reads [r0, r1) of a call and the pairs that use them
    int slice = 0, n_slices = 1;
    int64_t r0 = 0, r1 = 0;
    int64_t table_base = 0;     // absolute table position of the slice's zero run
    int64_t table_entries = 0;  // entries of the slice's table (zero run and slack included)
    const int* ids = nullptr;   // the slice's pairs (caller pair indices, ascending); nullptr: all pairs of the batch
    int64_t n_ids = 0;
    int64_t n_short = 0;        // pairs of the sub-warp systolic fp32 kernel
    std::vector<int> seq_pairs, strip_pairs, sub_pairs;  // chain kernel work lists, fp64 sub-warp list (caller pair indices)
    int64_t n_pairs = 0, lane_rows = 0;
    int max_seq_l = 0, max_long_l = 0;  // longest read of the short class / of the long pairs
};

}  // namespace

static int run_slice(phmm_ctx* ctx, const phmm_batch* b, const HostBatchView& hv, bool fp64, double* d_out, uint8_t* d_flags,
                     cudaStream_t st, const phmm_ctx::CallSet& cs, SliceWork& sw, const HostPayload* hp);

// phmm_options.validate: one device pass over the payload (device pointers in `b`), then a synchronisation
static int validate_payload(phmm_ctx* ctx, const phmm_batch* b, cudaStream_t st) {
    DevBatch db;
    memset(&db, 0, sizeof(db));
    db.read_bases = b->d_read_bases; db.qual_base = b->d_qual_base; db.qual_ins = b->d_qual_ins;
    db.qual_del = b->d_qual_del; db.qual_gcp = b->d_qual_gcp; db.hap_bases = b->d_hap_bases;
    CK(ctx->d_acc.need(16));
    CK(cudaMemsetAsync(ctx->d_acc.p, 0, 16, st));
    CK(launch_validate(db, (const double*)ctx->d_lut.p, b->h_read_off[0], b->h_read_off[b->n_reads], b->h_hap_off[0],
                       b->h_hap_off[b->n_haps], ctx->opt.qual_offset, (int*)ctx->d_acc.p, st));
    int err = 0;
    CK(cudaMemcpyAsync(&err, ctx->d_acc.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return err ? PHMM_E_ARG : PHMM_OK;
}

// The whole call: validation, classification, the global haplotype-major order of the short pairs, the cut into slices of
// reads (so that the row-constant table of a slice fits the workspace budget), then slice after slice: host plan, uploads
// and launches.  Everything is enqueued; the host work of slice s+1 runs while the GPU works on slice s.
static int forward_impl(phmm_ctx* ctx, const phmm_batch* b, int precision, double* d_out, uint8_t* d_flags, cudaStream_t st,
                        const HostPayload* hp, int min_slices) {
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    const auto t0 = std::chrono::steady_clock::now();
    const bool fp64 = precision == PHMM_FP64;
    const int64_t np = b->n_pairs, nr = b->n_reads;

    // ---- slices of reads: equal shares of the table, each within the budget
    std::vector<int64_t> bound;
    const int n_slices = slice_reads(hv, ctx->opt.max_table_bytes, min_slices, &bound);
    if (n_slices > 1) {
        ctx->read_slice.resize((size_t)nr);
        for (int s = 0; s < n_slices; s++) memset(ctx->read_slice.data() + bound[(size_t)s], s, (size_t)(bound[(size_t)s + 1] - bound[(size_t)s]));
    }
    std::vector<SliceWork> sl((size_t)n_slices);
    for (int s = 0; s < n_slices; s++) {
        SliceWork& w = sl[(size_t)s];
        w.slice = s; w.n_slices = n_slices; w.r0 = bound[(size_t)s]; w.r1 = bound[(size_t)s + 1];
        w.table_base = table_run_start(b->h_read_off[w.r0], w.r0) - TABLE_ZERO_RUN;
        w.table_entries = table_run_start(b->h_read_off[w.r1], w.r1) - w.table_base + 192;  // (slack: prefetches run past a run)
        if (w.table_entries > INT32_MAX) return PHMM_E_TOOLONG;
        if (w.table_entries * 64 > ctx->opt.max_table_bytes && n_slices >= std::min<int64_t>(250, nr)) return PHMM_E_NOMEM;
    }

    // ---- the pairs of each slice (stable: ascending pair index within a slice)
    std::vector<int64_t> first((size_t)n_slices + 1, 0);
    if (n_slices > 1) {
        bucket_pairs_by_slice(hv, ctx->read_slice.data(), n_slices, &ctx->slice_ids, &first);
        for (int s = 0; s < n_slices; s++) { sl[(size_t)s].ids = ctx->slice_ids.data() + first[(size_t)s]; sl[(size_t)s].n_ids = first[(size_t)s + 1] - first[(size_t)s]; }
    } else {
        sl[0].n_ids = np;
    }
    ctx->stats.n_pairs = np;
    ctx->stats.n_slices = n_slices;
    ctx->stats.host_batch_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();

    // ---- per call: offsets and pair list to the device, on the copy stream (under the kernels of the previous call)
    phmm_ctx::CallSet& cs = ctx->cset[ctx->call_idx & 1];
    ctx->call_idx++;
    if (cs.used) CK(cudaEventSynchronize(cs.ev_free));  // the call that used this set (two calls ago) has completed
    CK(cs.h_stage.need(4096 + (size_t)(nr + 1) * 8 + (size_t)(b->n_haps + 1) * 8 + (size_t)np * 8));
    {
        Stager sg{ctx, &cs.h_stage, ctx->copy_stream};
        RC(sg.upload(cs.d_read_off, b->h_read_off, (size_t)(nr + 1) * 8));
        RC(sg.upload(cs.d_hap_off, b->h_hap_off, (size_t)(b->n_haps + 1) * 8));
        RC(sg.upload(cs.d_pair_read, b->h_pair_read, (size_t)np * 4));
        RC(sg.upload(cs.d_pair_hap, b->h_pair_hap, (size_t)np * 4));
    }
    CK(cudaStreamWaitEvent(st, ctx->ev_last, 0));  // calls on different streams of one context run one after the other
    cs.used = true;
    struct CallMark {  // whatever path leaves the call: the set is free once everything enqueued so far on st has run
        cudaEvent_t ev, ev_last; cudaStream_t st;
        ~CallMark() { cudaEventRecord(ev, st); cudaEventRecord(ev_last, st); }
    } call_mark{cs.ev_free, ctx->ev_last, st};
    CK(ctx->d_acc.need(16));
    CK(cudaMemsetAsync(ctx->d_acc.p, 0, 16, st));
    if (ctx->opt.profile_events) {
        while (ctx->ev_prof.size() < 8 * (size_t)n_slices) {
            cudaEvent_t e = nullptr;
            CK(cudaEventCreate(&e));
            ctx->ev_prof.push_back(e);
        }
        ctx->prof_used.assign(4 * (size_t)n_slices, 0);
    }

    // ---- slice after slice
    for (int s = 0; s < n_slices; s++) {
        if (sl[(size_t)s].n_ids == 0) continue;
        RC(run_slice(ctx, b, hv, fp64, d_out, d_flags, st, cs, sl[(size_t)s], hp));
    }
    return PHMM_OK;
}

static int run_slice(phmm_ctx* ctx, const phmm_batch* b, const HostBatchView& hv, bool fp64, double* d_out, uint8_t* d_flags,
                     cudaStream_t st, const phmm_ctx::CallSet& cs, SliceWork& sw, const HostPayload* hp) {
    const int64_t np_slice = sw.n_ids;
    DevBatch db;
    db.read_bases = b->d_read_bases; db.qual_base = b->d_qual_base; db.qual_ins = b->d_qual_ins;
    db.qual_del = b->d_qual_del; db.qual_gcp = b->d_qual_gcp; db.hap_bases = b->d_hap_bases;
    db.read_off = (const int64_t*)cs.d_read_off.p; db.hap_off = (const int64_t*)cs.d_hap_off.p;
    db.n_reads = b->n_reads; db.n_haps = b->n_haps;
    db.table_base = sw.table_base;
    db.n_wild = ctx->opt.n_is_wildcard ? 1 : 0;
    int launches = 0;
    // ---- fp32: the slice's share of the read arrays (host entry: pinned or pageable host memory) and its row-constant table
    // (short and long pairs use the same one) go first: they need nothing of the plan, so the copy and the table kernel run
    // while the host plans the slice (configs[1] through the host entry: within the run-to-run noise of the box, about +1 %)
    if (hp) {
        const int64_t o0 = b->h_read_off[sw.r0], o1 = b->h_read_off[sw.r1];
        for (int i = 0; i < 5 && o1 > o0; i++)
            CK(cudaMemcpyAsync(hp->dst[i] + o0, hp->src[i] + o0, (size_t)(o1 - o0), cudaMemcpyHostToDevice, ctx->copy_stream));
    }
    if (!fp64) {
        int max_len = 0;
        for (int64_t r = sw.r0; r < sw.r1; r++) max_len = std::max(max_len, (int)(b->h_read_off[r + 1] - b->h_read_off[r]));
        CK(cudaEventRecord(ctx->ev_pay, ctx->copy_stream));  // (behind the call's offset arrays, uploaded on the same stream)
        CK(cudaStreamWaitEvent(st, ctx->ev_pay, 0));
        const size_t table_bytes = (size_t)sw.table_entries * 64;
        CK(ctx->d_table.need(table_bytes));
        ctx->stats.table_bytes = std::max<int64_t>(ctx->stats.table_bytes, (int64_t)table_bytes);
        PROF(0, 0);
        CK(launch_lut_table(db, (const double*)ctx->d_lut.p, (float*)ctx->d_table.p, sw.r0, sw.r1, max_len, st));
        PROF(0, 1);
        launches++;
    }
    const auto t0 = std::chrono::steady_clock::now();
    // ---- classify: short (sub-warp systolic fp32 kernel) / fp64 sub-warp / chain-sequential (one warp per pair) / strips
    {
        struct Part { std::vector<int> seq, strip, sub, sh; int64_t cells = 0, lane_rows = 0; int max_l = 0, max_l_long = 0; };
        Part part[BATCHER_THREADS];
        const int long_k = ctx->opt.long_min_hap_len;
        const int tall_k = fp64 ? 0 : long_k * 7 / 8;  // (phmm_kernels.h, long_class)
        const int* ids = sw.ids;
        const int T = parallel_chunks(np_slice, 1 << 16, [&](int t, int64_t lo, int64_t hi) {
            Part& q = part[t];
            for (int64_t i = lo; i < hi; i++) {
                const int p = ids ? ids[i] : (int)i;
                const int r = b->h_pair_read[p], h = b->h_pair_hap[p];
                const int64_t l = b->h_read_off[r + 1] - b->h_read_off[r], k = b->h_hap_off[h + 1] - b->h_hap_off[h];
                q.cells += l * k;
                if (long_class(k, l, long_k, tall_k)) { q.strip.push_back(p); if (l > q.max_l_long) q.max_l_long = (int)l; }
                else {
                    if (fp64 && k <= RESCUE_MAX_K && l <= RESCUE_MAX_L) q.sub.push_back(p);
                    else if (fp64) q.seq.push_back(p);
                    else { q.sh.push_back(p); q.lane_rows += l * ((k + SHORT_N2 - 1) / SHORT_N2); }
                    if (l > q.max_l) q.max_l = (int)l;
                }
            }
        });
        ctx->short_ids.clear();
        for (int t = 0; t < T; t++) {  // chunks are contiguous and in order: the lists stay sorted by pair index
            sw.seq_pairs.insert(sw.seq_pairs.end(), part[t].seq.begin(), part[t].seq.end());
            sw.strip_pairs.insert(sw.strip_pairs.end(), part[t].strip.begin(), part[t].strip.end());
            sw.sub_pairs.insert(sw.sub_pairs.end(), part[t].sub.begin(), part[t].sub.end());
            ctx->short_ids.insert(ctx->short_ids.end(), part[t].sh.begin(), part[t].sh.end());
            ctx->stats.cells += part[t].cells; sw.lane_rows += part[t].lane_rows;
            if (part[t].max_l > sw.max_seq_l) sw.max_seq_l = part[t].max_l;
            if (part[t].max_l_long > sw.max_long_l) sw.max_long_l = part[t].max_l_long;
        }
        sw.n_short = (int64_t)ctx->short_ids.size();
        ctx->stats.n_long_pairs += (int64_t)sw.strip_pairs.size();
        ctx->stats.n_short_pairs += np_slice - (int64_t)sw.strip_pairs.size();
        if (!fp64) sort_ids_by_hap(hv, ctx->short_ids.data(), sw.n_short, &ctx->sorted_all);  // haplotype-major
    }
    // task size: as large as possible (fewer run-ins, pipeline fills and host work; 8192 rows measured best on
    // configs[1]) while leaving at least ~6 warps of work per resident warp slot
    int task_rows = ctx->opt.task_rows;
    if (task_rows <= 0) {
        const int64_t slots = (int64_t)ctx->n_sm * 12;
        task_rows = (int)std::max<int64_t>(1024, std::min<int64_t>(8192, sw.lane_rows / 32 / (6 * slots)));
    }
    if (!fp64) plan_tasks(hv, ctx->sorted_all.data(), sw.n_short, sw.table_base, SHORT_N2, task_rows, &ctx->plan);
    else { ctx->plan.tasks.clear(); ctx->plan.warp_first.assign(1, 0); ctx->plan.srt_out.clear(); ctx->plan.srt_ent.clear(); ctx->plan.cells = 0; ctx->plan.padded_cells = 0; ctx->plan.max_read_len = 0; }
    const ShortPlan& pl = ctx->plan;
    const int n_warps = (int)pl.warp_first.size() - 1;
    const int max_seq_l = std::max(sw.max_seq_l, pl.max_read_len), max_long_l = sw.max_long_l;
    ctx->stats.short_cells += pl.cells;
    ctx->stats.short_padded_cells += pl.padded_cells;
    ctx->stats.n_short_warps += n_warps;

    // ---- strip items of the long pairs, STRIP-major: strip s of every pair before strip s+1 of any.  A strip's
    // producer still holds an earlier ticket (forward progress), but it is far ahead or done by the time the
    // consumer starts, so consumers do not run in lock step with their producers and hardly ever poll (pair-major
    // order: 4.6 polls per step, 19 % of the stall samples; profiles/).  Boundary buffers are full-length per strip.
    const int strip_cols = fp64 ? long64_strip_cols() : chain_strip_cols(false);
    std::vector<ChainItem> items;
    int64_t n_bnd_blocks = 0;
    int n_prog = 0;
    {
        struct PairStrips { int pair, ns, prog0; int64_t buf0; };
        std::vector<PairStrips> ps;
        ps.reserve(sw.strip_pairs.size());
        int max_ns = 0;
        size_t total = 0;
        for (int p : sw.strip_pairs) {
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
    ctx->stats.host_batch_ms += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();

    // ---- uploads.  The plan arrays go to this slice's plan set on the context's copy stream (overlapping the kernels
    // of the previous slice / call, which read the other set); the small counters and lists that kernels also write
    // stay on the caller's stream.
    phmm_ctx::PlanSet& ps = ctx->set[ctx->slice_idx & 1];
    ctx->slice_idx++;
    if (ps.used) CK(cudaEventSynchronize(ps.ev_free));  // the slice that used this set (two slices ago) has completed
    const size_t n_seq = fp64 ? sw.seq_pairs.size() : 0;
    size_t stage_bytes = 4096 + pl.tasks.size() * sizeof(ShortTask) + pl.warp_first.size() * 4 + pl.srt_out.size() * 16 +
                         items.size() * sizeof(ChainItem) + n_seq * 4 + sw.sub_pairs.size() * 4 + 20 * 256;
    CK(ps.h_stage.need(stage_bytes));
    Stager sg{ctx, &ps.h_stage, ctx->copy_stream};
    RC(sg.upload(ps.d_tasks, pl.tasks.data(), pl.tasks.size() * sizeof(ShortTask)));
    RC(sg.upload(ps.d_warp_first, pl.warp_first.data(), pl.warp_first.size() * 4));
    RC(sg.upload(ps.d_srt_ent, pl.srt_ent.data(), pl.srt_ent.size() * 4));
    RC(sg.upload(ps.d_srt_out, pl.srt_out.data(), pl.srt_out.size() * 4));
    RC(sg.upload(ps.d_items, items.data(), items.size() * sizeof(ChainItem)));
    RC(sg.upload(ps.d_rq_enq, sw.sub_pairs.data(), sw.sub_pairs.size() * 4));
    RC(sg.upload(ps.d_seq, sw.seq_pairs.data(), n_seq * 4));
    CK(cudaEventRecord(ps.ev_up, ctx->copy_stream));
    CK(cudaStreamWaitEvent(st, ps.ev_up, 0));  // (covers the call's offset arrays and pair list too: same stream, earlier)
    ps.used = true;
    struct FreeMark {
        cudaEvent_t ev; cudaStream_t st;
        ~FreeMark() { cudaEventRecord(ev, st); }
    } free_mark{ps.ev_free, st};
    // counters: [0] rescue count (= n_items of the rescue launch)  [1] ticket rescue  [2] n strip items  [3] ticket strips
    //           [4] n sequential fp64 items  [5] ticket sequential
    sg.st = st;  // from here on: buffers that kernels write as well, in stream order with them
    int h_counters[8] = {0, 0, (int)items.size(), 0, (int)n_seq, 0, 0, 0};
    RC(sg.upload(ctx->d_counters, h_counters, sizeof(h_counters)));
    // rescue list (fp32 mode: filled by the kernels) / sequential list (fp64 mode: the short-class pairs the sub-warp kernel does not take)
    CK(ctx->d_rescue.need((size_t)np_slice * 4 + 4));
    if (n_seq) CK(cudaMemcpyAsync(ctx->d_rescue.p, ps.d_seq.p, n_seq * 4, cudaMemcpyDeviceToDevice, st));
    CK(ctx->d_rq.need(RQ_INTS * 4));
    CK(ctx->d_rq_plan.need(RESCUE_PLAN_INTS * 4));
    CK(ctx->d_rq_queue.need((size_t)np_slice * 16 + 16));
    CK(ctx->d_rq_sorted.need((size_t)np_slice * 4 + 4));
    CK(cudaMemsetAsync(ctx->d_rq.p, 0, RQ_INTS * 4, st));

    const int* d_pair_read = (const int*)cs.d_pair_read.p;
    const int* d_pair_hap = (const int*)cs.d_pair_hap.p;
    int* counters = (int*)ctx->d_counters.p;
    const bool long32 = !fp64 && !items.empty();
    if (fp64 && (!sw.sub_pairs.empty() || !items.empty())) {  // PHMM_FP64: the same table in double, for the sub-warp kernel and the strips
        const size_t table_bytes = (size_t)sw.table_entries * 64;
        CK(ctx->d_table.need(table_bytes));
        ctx->stats.table_bytes = std::max<int64_t>(ctx->stats.table_bytes, (int64_t)table_bytes);
        PROF(0, 0);
        CK(launch_table_f64(db, (const double*)ctx->d_lut.p, (double*)ctx->d_table.p, sw.r0, sw.r1, std::max(max_seq_l, max_long_l), st));
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
        sl.pair_read = d_pair_read;
        sl.rescue_count = counters + 0;
        sl.rescue_list = (int*)ctx->d_rescue.p;
        PROF(1, 0);
        CK(launch_short_f32(db, sl, st));
        PROF(1, 1);
        launches++;
    }
    // ---- long path.  fp32: table-driven strips with per-lane exponents (phmm_long.cu); what it cannot represent joins
    // the rescue list of the fp64 chain launch below.  fp64: table-driven strips in double with per-thread exponents (phmm_long64.cu).
    if (!items.empty()) {
        CK(ctx->d_progress.need((size_t)n_prog * 4 + 4));
        CK(cudaMemsetAsync(ctx->d_progress.p, 0, (size_t)n_prog * 4 + 4, st));
        // no more CTAs than there are strips: with fewer strips than resident warps the block scheduler would fill
        // some SMs completely and leave others empty (configs[4]: 1648 strips, 2368 slots: 1.36 vs 1.76 TCUPS)
        const int wpc = fp64 ? 1 : long_warps_per_cta();
        const int need_ctas = (int)((items.size() + (size_t)wpc - 1) / (size_t)wpc);
        PROF(3, 0);
        if (fp64) {
            CK(ctx->d_boundary.need((size_t)(n_bnd_blocks + 1) * long64_block_bytes()));
            ChainLaunch cl;
            memset(&cl, 0, sizeof(cl));
            cl.items = (const ChainItem*)ps.d_items.p;
            cl.n_items = counters + 2;
            cl.ticket = counters + 3;
            cl.pair_read = d_pair_read;
            cl.pair_hap = d_pair_hap;
            cl.lut = (const double*)ctx->d_lut.p;
            cl.boundary = ctx->d_boundary.p;
            cl.scratch_blocks = 0;
            cl.progress = (int*)ctx->d_progress.p;
            cl.out = d_out;
            cl.flags = d_flags;
            cl.flag_bits = PHMM_FLAG_LONG;
            cl.log2C = 0;
            CK(launch_long_f64(db, cl, (const double*)ctx->d_table.p, std::min(ctx->long64_grid, need_ctas), st));
        } else {
            CK(ctx->d_boundary.need((size_t)(n_bnd_blocks + 1) * 16));
            CK(ctx->d_totals.need((size_t)n_prog * 16 + 16));
            CK(ctx->d_risk.need((size_t)b->n_reads + 16));
            CK(launch_read_risk(db, ctx->opt.qual_offset, sw.r0, sw.r1, (uint8_t*)ctx->d_risk.p, st));
            launches++;
            LongLaunch ll;
            memset(&ll, 0, sizeof(ll));
            ll.table = (const float*)ctx->d_table.p;
            ll.items = (const ChainItem*)ps.d_items.p;
            ll.n_items = counters + 2;
            ll.ticket = counters + 3;
            ll.pair_read = d_pair_read;
            ll.pair_hap = d_pair_hap;
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
            ll.risk = (const uint8_t*)ctx->d_risk.p;
            CK(launch_long_f32(db, ll, std::min(ctx->long_grid, need_ctas), st));
        }
        PROF(3, 1);
        launches++;
    }
    // fp64 sub-warp kernel: fp32 mode = what the short kernel queued, fp64 mode = the short pairs it can hold
    const bool sub = n_warps > 0 || !sw.sub_pairs.empty();
    if (sub) {
        RescueLaunch rl;
        memset(&rl, 0, sizeof(rl));
        rl.queue.queue = (int4*)ctx->d_rq_queue.p;
        rl.queue.cnt = (int*)ctx->d_rq.p;
        rl.table = ctx->d_table.p;
        rl.table_f64 = fp64 ? 1 : 0;
        rl.max_queue = (int)(fp64 ? (int64_t)sw.sub_pairs.size() : sw.n_short);
        rl.enqueue_pairs = fp64 ? (const int*)ps.d_rq_enq.p : nullptr;
        rl.n_enqueue = fp64 ? (int)sw.sub_pairs.size() : 0;
        rl.plan = (int*)ctx->d_rq_plan.p;
        rl.sorted = (int*)ctx->d_rq_sorted.p;
        rl.pair_read = d_pair_read;
        rl.pair_hap = d_pair_hap;
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
        cl.pair_read = d_pair_read;
        cl.pair_hap = d_pair_hap;
        cl.lut = (const double*)ctx->d_lut.p;
        cl.boundary = ctx->d_scratch.p;
        cl.scratch_blocks = blocks;
        cl.progress = nullptr;
        cl.out = d_out;
        cl.flags = d_flags;
        cl.flag_bits = fp64 ? 0 : PHMM_FLAG_RESCUED;
        cl.long_k = ctx->opt.long_min_hap_len;
        cl.tall_k = fp64 ? 0 : ctx->opt.long_min_hap_len * 7 / 8;
        cl.log2C = 0;
        if (!sub) PROF(2, 0);
        CK(launch_chain(db, cl, true, true, grid, st));
        PROF(2, 1);
        launches++;
    }
    if (!fp64 && (n_warps > 0 || long32)) {  // pairs recomputed in fp64 so far (phmm_get_stats)
        k_accumulate_rescued<<<1, 1, 0, st>>>((long long*)ctx->d_acc.p, counters, (const int*)ctx->d_rq.p);
        CK(cudaGetLastError());
        launches++;
    }
    ctx->stats.n_kernel_launches += launches;
    return PHMM_OK;
}

extern "C" int phmm_forward_batch(phmm_ctx* ctx, const phmm_batch* b, int precision, double* d_out, uint8_t* d_flags,
                                  void* cuda_stream) {
    if (!ctx || !b) return PHMM_E_ARG;
    if (precision != PHMM_FP32_RESCUE && precision != PHMM_FP64) return PHMM_E_ARG;
    if (b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    memset(&ctx->stats, 0, sizeof(ctx->stats));
    ctx->stats_final = false;
    ctx->prof_used.clear();
    if (b->n_pairs == 0) return PHMM_OK;
    if (!d_out || !b->d_read_bases || !b->d_qual_base || !b->d_qual_ins || !b->d_qual_del || !b->d_qual_gcp || !b->d_hap_bases)
        return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    RC(validate_batch(hv));
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return PHMM_E_CUDA;
    if (ctx->opt.validate) {
        CK(cudaStreamWaitEvent((cudaStream_t)cuda_stream, ctx->ev_last, 0));
        RC(validate_payload(ctx, b, (cudaStream_t)cuda_stream));
    }
    // (one slice unless the table budget asks for more: slicing a device-resident batch costs 1-2 % of throughput per
    // extra slice and takes only ~4 of the ~15 ms that one isolated configs[1] call spends outside its kernels)
    return forward_impl(ctx, b, precision, d_out, d_flags, (cudaStream_t)cuda_stream, nullptr, 1);
}

// ---------------------------------------------------------------- end-to-end entries with host buffers
// Completion of a host call: its outputs are in the caller's arrays; the statistics become those of this call.
static int host_wait(phmm_ctx* ctx, int set) {
    phmm_ctx::HostSet& hs = ctx->hset[set];
    if (!hs.pending) return PHMM_OK;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return PHMM_E_CUDA;
    hs.pending = false;
    CK(cudaEventSynchronize(hs.done));
    int64_t n_resc = 0;
    for (int64_t p = 0; p < hs.np; p++) n_resc += hs.fl[p] & PHMM_FLAG_RESCUED;
    hs.stats.n_rescued = n_resc;
    ctx->stats = hs.stats;
    ctx->stats_final = true;
    return PHMM_OK;
}

// Enqueues everything of one host call (copies in, plan, kernels, copies out) and returns; `pipelined`: the call is one of a
// stream of calls, so the copies and the plan of the next one will overlap this one's kernels and slices within the call
// buy nothing.
static int host_submit(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out, uint8_t* h_flags, bool pipelined, int* ticket) {
    if (!ctx || !b) return PHMM_E_ARG;
    if (precision != PHMM_FP32_RESCUE && precision != PHMM_FP64) return PHMM_E_ARG;
    if (b->n_pairs < 0 || b->n_reads < 0 || b->n_haps < 0) return PHMM_E_ARG;
    const int set = ctx->host_calls & 1;
    phmm_ctx::HostSet& hs = ctx->hset[set];
    RC(host_wait(ctx, set));  // the call that used this set two calls ago (its outputs are complete, its statistics superseded)
    if (ticket) *ticket = ctx->host_calls;
    hs.ticket = ctx->host_calls;
    ctx->host_calls = (ctx->host_calls + 1) & 0x3fffffff;
    memset(&ctx->stats, 0, sizeof(ctx->stats));
    ctx->stats_final = false;
    ctx->prof_used.clear();
    if (b->n_pairs == 0) return PHMM_OK;
    if (!h_out || !b->h_read_off || !b->h_hap_off) return PHMM_E_ARG;
    HostBatchView hv = {b->n_reads, b->n_haps, b->n_pairs, b->h_read_off, b->h_hap_off, b->h_pair_read, b->h_pair_hap};
    RC(validate_batch(hv));
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return PHMM_E_CUDA;
    const size_t R = (size_t)b->h_read_off[b->n_reads], H = (size_t)b->h_hap_off[b->n_haps];
    const size_t Ra = (R + 255) & ~(size_t)255, Ha = (H + 255) & ~(size_t)255;
    const int64_t np = b->n_pairs;
    CK(hs.d_payload.need(5 * Ra + Ha + 256));
    CK(hs.d_out.need((size_t)np * 8));
    CK(hs.d_flags.need((size_t)np));
    uint8_t* fl = h_flags;
    if (!fl) { CK(hs.h_flags.need((size_t)np)); fl = (uint8_t*)hs.h_flags.p; }
    uint8_t* base = (uint8_t*)hs.d_payload.p;
    HostPayload hp;
    const uint8_t* src[5] = {b->d_read_bases, b->d_qual_base, b->d_qual_ins, b->d_qual_del, b->d_qual_gcp};
    for (int i = 0; i < 5; i++) {
        if (!src[i]) return PHMM_E_ARG;
        hp.src[i] = src[i] - b->h_read_off[0];  // (indexed by absolute read offsets)
        hp.dst[i] = base + i * Ra - b->h_read_off[0];
    }
    if (!b->d_hap_bases) return PHMM_E_ARG;
    cudaStream_t st = ctx->host_stream;
    // (this set's payload buffer is free: the call that read it was waited for above)
    CK(cudaMemcpyAsync(base + 5 * Ra, b->d_hap_bases, H, cudaMemcpyHostToDevice, ctx->copy_stream));
    phmm_batch db = *b;
    db.d_read_bases = hp.dst[0]; db.d_qual_base = hp.dst[1]; db.d_qual_ins = hp.dst[2]; db.d_qual_del = hp.dst[3];
    db.d_qual_gcp = hp.dst[4]; db.d_hap_bases = base + 5 * Ra - b->h_hap_off[0];
    // A call on its own: the reads are processed in slices (at least one per 48 MB of read payload, up to 16), so that the copy
    // of slice s+1 and its host plan run while the GPU works on slice s (the "with transfers" convention).
    const int min_slices = pipelined ? 1 : (int)std::max<size_t>(1, std::min<size_t>(16, 5 * R / ((size_t)48 << 20)));  // (configs[1]: 1 / 2 / 4 / 7 / 10 slices: 53.6 / 51.5 / 48.6 / 50.7 / 50.0 ms)
    const HostPayload* hpp = &hp;
    if (ctx->opt.validate) {  // the whole payload first, then the check: nothing may be written for a bad batch
        CK(cudaStreamWaitEvent(st, ctx->ev_last, 0));
        for (int i = 0; i < 5; i++) CK(cudaMemcpyAsync(base + i * Ra, src[i], R, cudaMemcpyHostToDevice, ctx->copy_stream));
        CK(cudaStreamSynchronize(ctx->copy_stream));
        RC(validate_payload(ctx, &db, st));
        hpp = nullptr;
    }
    int rc = forward_impl(ctx, &db, precision, (double*)hs.d_out.p, (uint8_t*)hs.d_flags.p, st, hpp, min_slices);
    if (rc != PHMM_OK) { cudaStreamSynchronize(st); return rc; }
    CK(cudaMemcpyAsync(h_out, hs.d_out.p, (size_t)np * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(fl, hs.d_flags.p, (size_t)np, cudaMemcpyDeviceToHost, st));
    CK(cudaEventRecord(hs.done, st));
    hs.pending = true;
    hs.np = np;
    hs.fl = fl;
    hs.stats = ctx->stats;
    return PHMM_OK;
}

extern "C" int phmm_forward_batch_host(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out, uint8_t* h_flags) {
    int ticket = 0;
    RC(host_submit(ctx, b, precision, h_out, h_flags, false, &ticket));
    return host_wait(ctx, ticket & 1);
}

extern "C" int phmm_forward_batch_host_async(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out, uint8_t* h_flags, int* ticket) {
    if (!ticket) return PHMM_E_ARG;
    return host_submit(ctx, b, precision, h_out, h_flags, true, ticket);
}

extern "C" int phmm_wait_host(phmm_ctx* ctx, int ticket) {
    if (!ctx || ticket < 0) return PHMM_E_ARG;
    if (ctx->hset[ticket & 1].ticket != ticket) return PHMM_OK;  // completed already: a later call took over its set
    return host_wait(ctx, ticket & 1);
}
