#include "phmm_batcher.h"

#include <math.h>
#include <string.h>

#include <algorithm>

#include "../../include/pairhmm_b200.h"

namespace phmm {

int validate_batch(const HostBatchView& b) {
    if (b.n_reads < 0 || b.n_haps < 0 || b.n_pairs < 0) return PHMM_E_ARG;
    if (b.n_pairs == 0) return PHMM_OK;
    if (!b.read_off || !b.hap_off || !b.pair_read || !b.pair_hap) return PHMM_E_ARG;
    if (b.n_reads > INT32_MAX || b.n_haps > INT32_MAX || b.n_pairs > INT32_MAX) return PHMM_E_TOOLONG;
    for (int64_t i = 0; i < b.n_reads; i++) {
        const int64_t l = b.read_off[i + 1] - b.read_off[i];
        if (l < 0) return PHMM_E_OFFSETS;
        if (l > PHMM_MAX_LEN) return PHMM_E_TOOLONG;
    }
    for (int64_t i = 0; i < b.n_haps; i++) {
        const int64_t k = b.hap_off[i + 1] - b.hap_off[i];
        if (k < 0) return PHMM_E_OFFSETS;
        if (k > PHMM_MAX_LEN) return PHMM_E_TOOLONG;
    }
    if ((b.n_reads > 0 && b.read_off[0] < 0) || (b.n_haps > 0 && b.hap_off[0] < 0)) return PHMM_E_OFFSETS;
    int rc[BATCHER_THREADS] = {0};
    parallel_chunks(b.n_pairs, 1 << 16, [&](int t, int64_t lo, int64_t hi) {
        for (int64_t p = lo; p < hi; p++) {
            const int64_t r = b.pair_read[p], h = b.pair_hap[p];
            if (r < 0 || r >= b.n_reads || h < 0 || h >= b.n_haps) { rc[t] = PHMM_E_OFFSETS; return; }
            if (b.read_off[r + 1] == b.read_off[r] || b.hap_off[h + 1] == b.hap_off[h]) { if (!rc[t]) rc[t] = PHMM_E_EMPTY; }
        }
    });
    for (int t = 0; t < BATCHER_THREADS; t++) if (rc[t] == PHMM_E_OFFSETS) return PHMM_E_OFFSETS;
    for (int t = 0; t < BATCHER_THREADS; t++) if (rc[t]) return rc[t];
    return PHMM_OK;
}

// Stable counting sort of the selected pairs by haplotype (chunks of the pair list in parallel: per-chunk histograms,
// then every chunk scatters into its own slice of each haplotype's run).  sorted: caller pair indices, haplotype-major.
void sort_pairs_by_hap(const HostBatchView& b, const uint8_t* is_short, std::vector<int>* sorted) {
    const int64_t np = b.n_pairs, nh = b.n_haps;
    std::vector<std::vector<int>> hist(BATCHER_THREADS);
    const int T = parallel_chunks(np, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& hs = hist[t];
        hs.assign((size_t)nh, 0);
        for (int64_t p = lo; p < hi; p++)
            if (is_short[p]) hs[b.pair_hap[p]]++;
    });
    int64_t n_sel = 0;
    for (int64_t h = 0; h < nh; h++)  // hist[t][h] = start of chunk t's slice of haplotype h's run
        for (int t = 0; t < T; t++) { const int c = hist[t][h]; hist[t][h] = (int)n_sel; n_sel += c; }
    if (sorted->size() != (size_t)n_sel) sorted->resize((size_t)n_sel);  // steady state: same size as the last call
    if (n_sel == 0) return;
    int* out = sorted->data();
    parallel_chunks(np, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& pos = hist[t];
        for (int64_t p = lo; p < hi; p++)
            if (is_short[p]) out[pos[b.pair_hap[p]]++] = (int)p;
    });
}

// Slices of consecutive reads: equal shares of the row-constant table (64 bytes per entry), as many as it takes for a
// share to stay within max_table_bytes (at least min_slices, at most 250 and one per read).  bound: n_slices + 1 read indices.
int slice_reads(const HostBatchView& b, int64_t max_table_bytes, int min_slices, std::vector<int64_t>* bound) {
    const int64_t nr = b.n_reads;
    const int64_t total_entries = table_run_start(b.read_off[nr], nr) - TABLE_ZERO_RUN;
    const int64_t budget_entries = std::max<int64_t>(max_table_bytes / 64 - 1024, 1 << 16);
    int n_slices = (int)std::min<int64_t>(250, (total_entries + budget_entries - 1) / budget_entries);
    n_slices = (int)std::max<int64_t>(1, std::min<int64_t>(std::max(n_slices, min_slices), nr));
    bound->assign((size_t)n_slices + 1, 0);
    (*bound)[(size_t)n_slices] = nr;
    for (int s = 1; s < n_slices; s++) {  // first read whose run starts at or behind the s-th share
        const int64_t want = TABLE_ZERO_RUN + total_entries * s / n_slices;
        int64_t lo = (*bound)[(size_t)s - 1], hi = nr;
        while (lo < hi) { const int64_t mid = (lo + hi) / 2; if (table_run_start(b.read_off[mid], mid) < want) lo = mid + 1; else hi = mid; }
        (*bound)[(size_t)s] = lo;
    }
    return n_slices;
}

// Stable counting sort of all pair indices by the slice their read belongs to: slice_first[s] = first position of slice s.
void bucket_pairs_by_slice(const HostBatchView& b, const uint8_t* read_slice, int n_slices, std::vector<int>* out,
                           std::vector<int64_t>* slice_first) {
    const int64_t n = b.n_pairs;
    out->resize((size_t)n);
    slice_first->assign((size_t)n_slices + 1, 0);
    std::vector<int64_t> hist((size_t)BATCHER_THREADS * (size_t)n_slices, 0);
    const int T = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        int64_t* hs = hist.data() + (size_t)t * n_slices;
        for (int64_t p = lo; p < hi; p++) hs[read_slice[b.pair_read[p]]]++;
    });
    int64_t run = 0;
    for (int s = 0; s < n_slices; s++) {
        (*slice_first)[(size_t)s] = run;
        for (int t = 0; t < T; t++) { int64_t& c = hist[(size_t)t * n_slices + s]; const int64_t v = c; c = run; run += v; }
    }
    (*slice_first)[(size_t)n_slices] = run;
    int* dst = out->data();
    parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        int64_t* pos = hist.data() + (size_t)t * n_slices;
        for (int64_t p = lo; p < hi; p++) dst[pos[read_slice[b.pair_read[p]]]++] = (int)p;
    });
}

// Stable counting sort of a list of pair indices by haplotype; the histogram spans only the haplotypes the list uses.
void sort_ids_by_hap(const HostBatchView& b, const int* ids, int64_t n, std::vector<int>* sorted) {
    if (sorted->size() != (size_t)n) sorted->resize((size_t)n);
    if (n == 0) return;
    int hmin[BATCHER_THREADS], hmax[BATCHER_THREADS];
    const int T0 = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        int mn = INT32_MAX, mx = -1;
        for (int64_t i = lo; i < hi; i++) { const int h = b.pair_hap[ids[i]]; mn = std::min(mn, h); mx = std::max(mx, h); }
        hmin[t] = mn; hmax[t] = mx;
    });
    int h0 = INT32_MAX, h1 = -1;
    for (int t = 0; t < T0; t++) { h0 = std::min(h0, hmin[t]); h1 = std::max(h1, hmax[t]); }
    const int64_t nh = (int64_t)h1 - h0 + 1;
    std::vector<std::vector<int>> hist(BATCHER_THREADS);
    const int T = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& hs = hist[t];
        hs.assign((size_t)nh, 0);
        for (int64_t i = lo; i < hi; i++) hs[b.pair_hap[ids[i]] - h0]++;
    });
    int64_t run = 0;
    for (int64_t h = 0; h < nh; h++)
        for (int t = 0; t < T; t++) { const int c = hist[t][h]; hist[t][h] = (int)run; run += c; }
    int* out = sorted->data();
    parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& pos = hist[t];
        for (int64_t i = lo; i < hi; i++) { const int p = ids[i]; out[pos[b.pair_hap[p] - h0]++] = p; }
    });
}

void plan_short(const HostBatchView& b, const uint8_t* is_short, int N2, int task_rows, ShortPlan* out) {
    std::vector<int> sorted;
    sort_pairs_by_hap(b, is_short, &sorted);
    plan_tasks(b, sorted.data(), (int64_t)sorted.size(), 0, N2, task_rows, out);
}

// Tasks and warps for a haplotype-major list of n short pairs (`sorted`: caller pair indices).  table_base: what is
// subtracted from a read's absolute table position (the slice's table starts at its first read).
void plan_tasks(const HostBatchView& b, const int* sorted, int64_t n_sel, int64_t table_base, int N2, int task_rows, ShortPlan* out) {
    out->tasks.clear(); out->warp_first.clear();  // the sorted arrays keep their size: they are overwritten in full
    out->cells = 0; out->padded_cells = 0; out->max_read_len = 0;
    if (n_sel == 0) { out->srt_out.clear(); out->srt_ent.clear(); out->warp_first.push_back(0); return; }
    if (out->srt_out.size() != (size_t)n_sel) {  // steady state: same size as the last call, nothing to (re)initialise
        out->srt_out.resize((size_t)n_sel);
        out->srt_ent.resize((size_t)n_sel * 2);
    }
    // ---- 1. positions of the reads' runs in the table
    parallel_chunks(n_sel, 1 << 17, [&](int, int64_t lo, int64_t hi) {
        for (int64_t q = lo; q < hi; q++) {
            const int p = sorted[q];
            const int r = b.pair_read[p];
            out->srt_out[(size_t)q] = p;
            out->srt_ent[2 * (size_t)q] = (int)(table_run_start(b.read_off[r], r) - table_base);
            out->srt_ent[2 * (size_t)q + 1] = table_run_len((int)(b.read_off[r + 1] - b.read_off[r]));
        }
    });
    // ---- 2. cut each haplotype's run of reads into tasks of about task_rows read rows (chunks of the list in parallel,
    //         every chunk starting where the haplotype changes)
    std::vector<ShortTask> tasks;
    {
        std::vector<ShortTask> part[BATCHER_THREADS];
        int64_t pcells[BATCHER_THREADS] = {0};
        int pmax[BATCHER_THREADS] = {0};
        const int T2 = parallel_chunks(n_sel, 1 << 15, [&](int t, int64_t lo, int64_t hi) {
            auto hap_at = [&](int64_t q) { return b.pair_hap[sorted[q]]; };
            while (lo > 0 && lo < n_sel && hap_at(lo) == hap_at(lo - 1)) lo++;  // this run belongs to the chunk before
            while (hi > 0 && hi < n_sel && hap_at(hi) == hap_at(hi - 1)) hi++;
            std::vector<ShortTask>& tv = part[t];
            int64_t cells = 0;
            int mx = 0;
            int64_t q = lo;
            while (q < hi) {
                const int h = hap_at(q);
                const int64_t k = b.hap_off[h + 1] - b.hap_off[h];
                ShortTask tk = {h, (int)q, 0, 0, 0};
                for (; q < n_sel && hap_at(q) == h; q++) {
                    const int r = b.pair_read[sorted[q]];
                    const int l = (int)(b.read_off[r + 1] - b.read_off[r]);
                    cells += (int64_t)l * k;
                    if (l > mx) mx = l;
                    tk.n_pairs++;
                    tk.rows += l;
                    tk.ents += out->srt_ent[2 * (size_t)q + 1];
                    if (tk.rows >= task_rows) {
                        tv.push_back(tk);
                        tk.pair_first = (int)q + 1; tk.n_pairs = 0; tk.rows = 0; tk.ents = 0;
                    }
                }
                if (tk.n_pairs > 0) tv.push_back(tk);
            }
            pcells[t] = cells; pmax[t] = mx;
        });
        size_t nt = 0;
        for (int t = 0; t < T2; t++) nt += part[t].size();
        tasks.reserve(nt);
        for (int t = 0; t < T2; t++) {
            tasks.insert(tasks.end(), part[t].begin(), part[t].end());
            out->cells += pcells[t];
            if (pmax[t] > out->max_read_len) out->max_read_len = pmax[t];
        }
    }
    // ---- 3. pack tasks into warps: duration classes (longest first), lanes bin-packed largest-fit
    const int NCLS = 8 * 40;  // class = floor(8 * log2(duration)), duration < 2^40
    auto cls_of = [&](const ShortTask& t) {
        const double d = (double)t.ents;
        int c = (int)floor(8.0 * log2(d < 1 ? 1 : d));
        return c < 0 ? 0 : (c >= NCLS ? NCLS - 1 : c);
    };
    auto lanes_of = [&](const ShortTask& t) {
        const int64_t k = b.hap_off[t.hap + 1] - b.hap_off[t.hap];
        return (int)((k + N2 - 1) / N2);
    };
    // bucket index = cls * 33 + g ; counting sort of task ids
    std::vector<int> bstart((size_t)NCLS * 33 + 1, 0);
    std::vector<int> tb(tasks.size());
    parallel_chunks((int64_t)tasks.size(), 1 << 14, [&](int, int64_t lo, int64_t hi) {
        for (int64_t i = lo; i < hi; i++) tb[(size_t)i] = cls_of(tasks[(size_t)i]) * 33 + lanes_of(tasks[(size_t)i]);
    });
    for (size_t i = 0; i < tasks.size(); i++) bstart[tb[i] + 1]++;
    for (size_t i = 0; i + 1 < bstart.size(); i++) bstart[i + 1] += bstart[i];
    std::vector<int> ids(tasks.size());
    {
        std::vector<int> pos(bstart.begin(), bstart.end() - 1);
        for (size_t i = 0; i < tasks.size(); i++) ids[pos[tb[i]]++] = (int)i;
    }
    std::vector<int> avail(bstart.begin(), bstart.end() - 1);  // next unused id per bucket
    std::vector<uint64_t> nonempty((size_t)NCLS, 0);  // bit g of nonempty[c] <=> bucket (c, g) still has tasks
    for (int c = 0; c < NCLS; c++)
        for (int g = 1; g <= 32; g++)
            if (avail[c * 33 + g] < bstart[c * 33 + g + 1]) nonempty[c] |= 1ull << g;
    // the classes are packed in parallel: contiguous class ranges of about equal task counts, longest classes first;
    // inside a range the open bin carries over from a class to the next shorter one, at the end of a range it is closed
    struct Part { std::vector<ShortTask> tasks; std::vector<int> warp_end; int64_t padded = 0; };
    Part part[BATCHER_THREADS];
    int range_hi[BATCHER_THREADS + 1];
    const int TP = (int)std::min<int64_t>(BATCHER_THREADS, std::max<int64_t>(1, (int64_t)tasks.size() / (1 << 14)));
    {
        const int64_t per = ((int64_t)tasks.size() + TP - 1) / TP;
        int t = 0;
        range_hi[0] = NCLS - 1;
        int64_t acc = 0;
        for (int c = NCLS - 1; c >= 0 && t + 1 < TP; c--) {
            acc += bstart[(size_t)(c + 1) * 33] - bstart[(size_t)c * 33];
            if (acc >= per * (t + 1)) range_hi[++t] = c - 1;
        }
        while (t < TP) range_hi[++t] = -1;
    }
    auto pack_range = [&](int t) {
        Part& P = part[t];
        if (range_hi[t] > range_hi[t + 1]) {
            const size_t n_range = (size_t)(bstart[(size_t)(range_hi[t] + 1) * 33] - bstart[(size_t)(range_hi[t + 1] + 1) * 33]);
            P.tasks.reserve(n_range);
            P.warp_end.reserve(n_range / 2 + 1);
        }
        int cap = 32, bin_steps = 0;
        auto close_bin = [&]() {
            if (cap < 32) {
                P.warp_end.push_back((int)P.tasks.size());
                P.padded += (int64_t)bin_steps * 32 * N2;
            }
            cap = 32; bin_steps = 0;
        };
        for (int c = range_hi[t]; c > range_hi[t + 1]; c--) {
            uint64_t best_mask = 0;  // best[q] = most lanes of a q-lane gap that lane counts of best_mask can fill (unbounded knapsack)
            int best[33];
            while (nonempty[c]) {
                const uint64_t fit = nonempty[c] & ((2ull << cap) - 1);  // lane counts <= cap
                if (!fit) { close_bin(); continue; }  // nothing of this class fits the open bin
                if (best_mask != nonempty[c]) {
                    best_mask = nonempty[c];
                    best[0] = 0;
                    for (int q = 1; q <= 32; q++) {
                        int bq = best[q - 1];
                        for (uint64_t m = best_mask & ((2ull << q) - 1); m; m &= m - 1) {
                            const int gg = __builtin_ctzll(m);
                            bq = std::max(bq, gg + best[q - gg]);
                        }
                        best[q] = bq;
                    }
                }
                int g = 0, gfill = -1;  // the lane count after which the rest of the gap can be filled best; ties: the larger one
                for (uint64_t m = fit; m; m &= m - 1) {
                    const int gg = __builtin_ctzll(m);
                    const int f = gg + best[cap - gg];
                    if (f >= gfill) { gfill = f; g = gg; }
                }
                const int bk = c * 33 + g;
                const ShortTask& tk = tasks[ids[avail[bk]++]];
                if (avail[bk] == bstart[bk + 1]) nonempty[c] &= ~(1ull << g);
                P.tasks.push_back(tk);
                cap -= g;
                bin_steps = std::max(bin_steps, tk.ents + 2 * g - 1);
                if (cap == 0) close_bin();
            }
        }
        close_bin();
    };
    {
        std::vector<std::thread> th;
        for (int t = 1; t < TP; t++) th.emplace_back(pack_range, t);
        pack_range(0);
        for (auto& x : th) x.join();
    }
    out->tasks.reserve(tasks.size());
    out->warp_first.push_back(0);
    for (int t = 0; t < TP; t++) {
        const int base = (int)out->tasks.size();
        out->tasks.insert(out->tasks.end(), part[t].tasks.begin(), part[t].tasks.end());
        for (int e : part[t].warp_end) out->warp_first.push_back(base + e);
        out->padded_cells += part[t].padded;
    }
}

}  // namespace phmm
