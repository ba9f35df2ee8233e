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
    {
        int rcs[BATCHER_THREADS] = {0};
        auto scan = [&](const int64_t* off, int64_t n) {
            parallel_chunks(n, 1 << 18, [&](int t, int64_t lo, int64_t hi) {
                for (int64_t i = lo; i < hi; i++) {
                    const int64_t l = off[i + 1] - off[i];
                    if (l < 0) { rcs[t] = PHMM_E_OFFSETS; return; }
                    if (l > PHMM_MAX_LEN && !rcs[t]) rcs[t] = PHMM_E_TOOLONG;
                }
            });
        };
        scan(b.read_off, b.n_reads);
        scan(b.hap_off, b.n_haps);
        for (int t = 0; t < BATCHER_THREADS; t++) if (rcs[t] == PHMM_E_OFFSETS) return PHMM_E_OFFSETS;
        for (int t = 0; t < BATCHER_THREADS; t++) if (rcs[t]) return rcs[t];
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

// Stable sort of a list of pair indices by haplotype: nothing to do if the list is grouped already; a counting sort with
// per-thread histograms over the haplotypes the list uses; or, where those are many more than pairs per thread, a radix sort.
void sort_ids_by_hap(const HostBatchView& b, const int* ids, int64_t n, std::vector<int>* sorted) {
    if (sorted->size() != (size_t)n) sorted->resize((size_t)n);
    if (n == 0) return;
    int hmin[BATCHER_THREADS], hmax[BATCHER_THREADS], first[BATCHER_THREADS], last[BATCHER_THREADS];
    bool mono[BATCHER_THREADS];
    const int T0 = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        int mn = INT32_MAX, mx = -1, prev = -1;
        bool m = true;
        for (int64_t i = lo; i < hi; i++) {
            const int h = b.pair_hap[ids[i]];
            mn = std::min(mn, h); mx = std::max(mx, h);
            m &= h >= prev;
            prev = h;
        }
        hmin[t] = mn; hmax[t] = mx; mono[t] = m; first[t] = b.pair_hap[ids[lo]]; last[t] = prev;
    });
    int h0 = INT32_MAX, h1 = -1;
    bool sorted_already = true;
    for (int t = 0; t < T0; t++) {
        h0 = std::min(h0, hmin[t]); h1 = std::max(h1, hmax[t]);
        sorted_already &= mono[t] && (t == 0 || first[t] >= last[t - 1]);
    }
    int* out = sorted->data();
    if (sorted_already) {  // a pair list that is grouped by haplotype already (the common case for callers that emit region by region)
        parallel_chunks(n, 1 << 17, [&](int, int64_t lo, int64_t hi) { memcpy(out + lo, ids + lo, (size_t)(hi - lo) * sizeof(int)); });
        return;
    }
    const int64_t nh = (int64_t)h1 - h0 + 1;
    if (nh * T0 > 8 * n && nh > 4096) {
        // many more haplotypes than a per-thread histogram is worth: stable LSD radix sort on the haplotype index, digits of
        // at most 11 bits, per-thread digit histograms (2048 counters) instead of per-thread histograms over all haplotypes
        int bits = 1;
        while (((int64_t)1 << bits) < nh) bits++;
        const int passes = (bits + 10) / 11, db = (bits + passes - 1) / passes, nd = 1 << db;
        std::vector<int> tmp((size_t)n);
        const int* src = ids;
        int* bufs[2] = {out, tmp.data()};
        int cur = (passes & 1) ? 0 : 1;  // so that the last pass writes `out`
        std::vector<int64_t> hist((size_t)BATCHER_THREADS * nd);
        for (int ps = 0; ps < passes; ps++) {
            const int sh = ps * db;
            std::fill(hist.begin(), hist.end(), 0);
            const int T = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
                int64_t* hs = hist.data() + (size_t)t * nd;
                for (int64_t i = lo; i < hi; i++) hs[((b.pair_hap[src[i]] - h0) >> sh) & (nd - 1)]++;
            });
            int64_t run = 0;
            for (int d = 0; d < nd; d++)
                for (int t = 0; t < T; t++) { int64_t& c = hist[(size_t)t * nd + d]; const int64_t v = c; c = run; run += v; }
            int* dst = bufs[cur];
            parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
                int64_t* pos = hist.data() + (size_t)t * nd;
                for (int64_t i = lo; i < hi; i++) { const int p = src[i]; dst[pos[((b.pair_hap[p] - h0) >> sh) & (nd - 1)]++] = p; }
            });
            src = dst;
            cur ^= 1;
        }
        return;
    }
    std::vector<std::vector<int>> hist(BATCHER_THREADS);
    const int T = parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& hs = hist[t];
        hs.assign((size_t)nh, 0);
        for (int64_t i = lo; i < hi; i++) hs[b.pair_hap[ids[i]] - h0]++;
    });
    int64_t run = 0;
    for (int64_t h = 0; h < nh; h++)
        for (int t = 0; t < T; t++) { const int c = hist[t][h]; hist[t][h] = (int)run; run += c; }
    parallel_chunks(n, 1 << 17, [&](int t, int64_t lo, int64_t hi) {
        std::vector<int>& pos = hist[t];
        for (int64_t i = lo; i < hi; i++) { const int p = ids[i]; out[pos[b.pair_hap[p] - h0]++] = p; }
    });
}

void plan_short(const HostBatchView& b, const uint8_t* is_short, int N2, int task_rows, ShortPlan* out) {
    std::vector<int> ids, sorted;  // the hot path's own sequence (phmm_api.cu, run_slice): ids of the short pairs, sorted by haplotype
    for (int64_t p = 0; p < b.n_pairs; p++)
        if (is_short[p]) ids.push_back((int)p);
    sort_ids_by_hap(b, ids.data(), (int64_t)ids.size(), &sorted);
    plan_tasks(b, sorted.data(), (int64_t)sorted.size(), 0, N2, task_rows, out);
}

// Tasks and warps for a haplotype-major list of n short pairs (`sorted`: caller pair indices).  table_base: what is
// subtracted from a read's absolute table position (the slice's table starts at its first read).
void plan_tasks(const HostBatchView& b, const int* sorted, int64_t n_sel, int64_t table_base, int N2, int task_rows, ShortPlan* out) {
    out->warp_first.clear();  // tasks and the sorted arrays keep their size: they are overwritten in full
    out->cells = 0; out->padded_cells = 0; out->max_read_len = 0;
    if (n_sel == 0) { out->tasks.clear(); out->srt_out.clear(); out->srt_ent.clear(); out->warp_first.push_back(0); return; }
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
    std::vector<ShortTask>& tasks = out->tmp_tasks;
    {
        std::vector<ShortTask>* part = out->tmp_cut;
        for (int t = 0; t < BATCHER_THREADS; t++) part[t].clear();
        int64_t pcells[BATCHER_THREADS] = {0};
        int pmax[BATCHER_THREADS] = {0};
        const int T2 = parallel_chunks(n_sel, 1 << 15, [&](int t, int64_t lo, int64_t hi) {
            auto hap_at = [&](int64_t q) { return b.pair_hap[sorted[q]]; };
            while (lo > 0 && lo < n_sel && hap_at(lo) == hap_at(lo - 1)) lo++;  // this run belongs to the chunk before
            while (hi > 0 && hi < n_sel && hap_at(hi) == hap_at(hi - 1)) hi++;
            std::vector<ShortTask>& tv = part[t];
            tv.reserve((size_t)std::max<int64_t>(hi - lo, 0) + 1);  // (at most one task per pair; untouched pages cost nothing)
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
        size_t nt = 0, at[BATCHER_THREADS + 1];
        for (int t = 0; t < T2; t++) { at[t] = nt; nt += part[t].size(); }
        if (tasks.size() != nt) tasks.resize(nt);
        {
            std::vector<std::thread> th;
            auto cp = [&](int t) { if (!part[t].empty()) memcpy(tasks.data() + at[t], part[t].data(), part[t].size() * sizeof(ShortTask)); };
            for (int t = 1; t < T2; t++) th.emplace_back(cp, t);
            cp(0);
            for (auto& x : th) x.join();
        }
        for (int t = 0; t < T2; t++) {
            out->cells += pcells[t];
            if (pmax[t] > out->max_read_len) out->max_read_len = pmax[t];
        }
    }
    // ---- 3. pack tasks into warps: duration classes (longest first), lanes bin-packed largest-fit.  Every thread packs a
    //         contiguous share of the task list on its own (its own counting sort by class and lane count; the open bin
    //         carries over from a class to the next shorter one); the threads' warps are then merged class by class, so that
    //         the launch order is still longest first.  (Until round 2 the classes were dealt to the threads: a batch of
    //         millions of equal tasks -- one class -- was packed by one thread.)
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
    typedef ShortPlan::PackPart Part;
    const int64_t nt = (int64_t)tasks.size();
    int TP = (int)std::min<int64_t>(BATCHER_THREADS, std::max<int64_t>(1, nt / (1 << 14)));
    {
        const unsigned hw = std::thread::hardware_concurrency();
        if (hw > 0 && (unsigned)TP > hw) TP = (int)hw;
    }
    Part* part = out->tmp_pack;
    auto pack_share = [&](int t) {
        Part& P = part[(size_t)t];
        const int64_t lo = nt * t / TP, hi = nt * (t + 1) / TP, n = hi - lo;
        P.tasks.clear(); P.warp_end.clear(); P.padded = 0;
        P.tasks.reserve((size_t)n);
        P.warp_end.reserve((size_t)n / 2 + 1);
        P.warps_after.assign((size_t)NCLS + 1, 0);
        // counting sort of the share's task ids by bucket = cls * 33 + lanes
        std::vector<int>&bstart = P.bstart, &tb = P.tb, &ids = P.ids, &avail = P.avail;
        bstart.assign((size_t)NCLS * 33 + 1, 0);
        if (tb.size() < (size_t)n) { tb.resize((size_t)n); ids.resize((size_t)n); }
        int last_ents = -1, last_cls = 0;
        for (int64_t i = 0; i < n; i++) {
            const ShortTask& tk = tasks[(size_t)(lo + i)];
            if (tk.ents != last_ents) { last_ents = tk.ents; last_cls = cls_of(tk); }  // (neighbours often have equal durations)
            tb[(size_t)i] = last_cls * 33 + lanes_of(tk);
            bstart[(size_t)tb[(size_t)i] + 1]++;
        }
        for (size_t i = 0; i + 1 < bstart.size(); i++) bstart[i + 1] += bstart[i];
        avail.assign(bstart.begin(), bstart.end() - 1);  // next unused id per bucket
        {
            std::vector<int> pos(avail);
            for (int64_t i = 0; i < n; i++) ids[(size_t)pos[(size_t)tb[(size_t)i]]++] = (int)i;
        }
        int cap = 32, bin_steps = 0;
        auto close_bin = [&]() {
            if (cap < 32) {
                P.warp_end.push_back((int)P.tasks.size());
                P.padded += (int64_t)bin_steps * 32 * N2;
            }
            cap = 32; bin_steps = 0;
        };
        for (int c = NCLS - 1; c >= 0; c--) {
            uint64_t nonempty = 0;  // bit g <=> bucket (c, g) still has tasks
            for (int g = 1; g <= 32; g++)
                if (avail[(size_t)c * 33 + g] < bstart[(size_t)c * 33 + g + 1]) nonempty |= 1ull << g;
            uint64_t best_mask = 0;  // best[q] = most lanes of a q-lane gap that lane counts of best_mask can fill (unbounded knapsack)
            int best[33];
            while (nonempty) {
                if (cap == 32 && (nonempty & (nonempty - 1)) == 0) {  // one lane count left in this class, a fresh bin: whole warps at once
                    const int g = __builtin_ctzll(nonempty), per = 32 / g;
                    const size_t bk = (size_t)c * 33 + g;
                    const int full = (bstart[bk + 1] - avail[bk]) / per;
                    for (int w = 0; w < full; w++) {
                        int steps = 0;
                        for (int j = 0; j < per; j++) {
                            const ShortTask& tk = tasks[(size_t)(lo + ids[(size_t)avail[bk]++])];
                            P.tasks.push_back(tk);
                            steps = std::max(steps, tk.ents + 2 * g - 1);
                        }
                        P.warp_end.push_back((int)P.tasks.size());
                        P.padded += (int64_t)steps * 32 * N2;
                    }
                    if (avail[bk] == bstart[bk + 1]) { nonempty = 0; break; }
                }
                const uint64_t fit = nonempty & ((2ull << cap) - 1);  // lane counts <= cap
                if (!fit) { close_bin(); continue; }  // nothing of this class fits the open bin
                if (best_mask != nonempty) {
                    best_mask = nonempty;
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
                const size_t bk = (size_t)c * 33 + g;
                const ShortTask& tk = tasks[(size_t)(lo + ids[(size_t)avail[bk]++])];
                if (avail[bk] == bstart[bk + 1]) nonempty &= ~(1ull << g);
                P.tasks.push_back(tk);
                cap -= g;
                bin_steps = std::max(bin_steps, tk.ents + 2 * g - 1);
                if (cap == 0) close_bin();
            }
            if (c == 0) close_bin();
            P.warps_after[(size_t)c] = (int)P.warp_end.size();
        }
    };
    {
        std::vector<std::thread> th;
        for (int t = 1; t < TP; t++) th.emplace_back(pack_share, t);
        pack_share(0);
        for (auto& x : th) x.join();
    }
    // ---- merge: for every class, longest first, the warps every thread closed in it
    int64_t n_warps = 0;
    for (int t = 0; t < TP; t++) { n_warps += (int64_t)part[(size_t)t].warp_end.size(); out->padded_cells += part[(size_t)t].padded; }
    if (out->tasks.size() != (size_t)nt) out->tasks.resize((size_t)nt);
    out->warp_first.assign((size_t)n_warps + 1, 0);
    std::vector<int64_t> seg_w((size_t)TP * (NCLS + 1), 0), seg_t((size_t)TP * (NCLS + 1), 0);  // output offsets of segment (t, c)
    {
        int64_t w = 0, k = 0;
        for (int c = NCLS - 1; c >= 0; c--)
            for (int t = 0; t < TP; t++) {
                const Part& P = part[(size_t)t];
                const int w0 = P.warps_after[(size_t)c + 1], w1 = P.warps_after[(size_t)c];
                seg_w[(size_t)t * (NCLS + 1) + c] = w; seg_t[(size_t)t * (NCLS + 1) + c] = k;
                if (w1 > w0) { w += w1 - w0; k += P.warp_end[(size_t)w1 - 1] - (w0 > 0 ? P.warp_end[(size_t)w0 - 1] : 0); }
            }
    }
    auto merge_share = [&](int t) {
        const Part& P = part[(size_t)t];
        for (int c = NCLS - 1; c >= 0; c--) {
            const int w0 = P.warps_after[(size_t)c + 1], w1 = P.warps_after[(size_t)c];
            if (w1 <= w0) continue;
            const int k0 = w0 > 0 ? P.warp_end[(size_t)w0 - 1] : 0, k1 = P.warp_end[(size_t)w1 - 1];
            const int64_t wo = seg_w[(size_t)t * (NCLS + 1) + c], ko = seg_t[(size_t)t * (NCLS + 1) + c];
            memcpy(out->tasks.data() + ko, P.tasks.data() + k0, (size_t)(k1 - k0) * sizeof(ShortTask));
            for (int w = w0; w < w1; w++) out->warp_first[(size_t)(wo + (w - w0)) + 1] = (int)(ko + (P.warp_end[(size_t)w] - k0));
        }
    };
    {
        std::vector<std::thread> th;
        for (int t = 1; t < TP; t++) th.emplace_back(merge_share, t);
        merge_share(0);
        for (auto& x : th) x.join();
    }
}

}  // namespace phmm
