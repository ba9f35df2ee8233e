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
    for (int64_t p = 0; p < b.n_pairs; p++) {
        const int64_t r = b.pair_read[p], h = b.pair_hap[p];
        if (r < 0 || r >= b.n_reads || h < 0 || h >= b.n_haps) return PHMM_E_OFFSETS;
        if (b.read_off[r + 1] == b.read_off[r] || b.hap_off[h + 1] == b.hap_off[h]) return PHMM_E_EMPTY;
    }
    return PHMM_OK;
}

void plan_short(const HostBatchView& b, const uint8_t* is_short, int N2, int task_rows, ShortPlan* out) {
    out->tasks.clear(); out->warp_first.clear(); out->srt_read.clear(); out->srt_out.clear(); out->srt_ent.clear();
    out->cells = 0; out->padded_cells = 0; out->max_read_len = 0;
    const int64_t np = b.n_pairs;
    // ---- 1. stable counting sort of the selected pairs by haplotype
    std::vector<int> cnt((size_t)b.n_haps + 1, 0);
    int64_t n_sel = 0;
    for (int64_t p = 0; p < np; p++)
        if (is_short[p]) { cnt[b.pair_hap[p] + 1]++; n_sel++; }
    if (n_sel == 0) { out->warp_first.push_back(0); return; }
    for (int64_t h = 0; h < b.n_haps; h++) cnt[h + 1] += cnt[h];
    out->srt_read.resize((size_t)n_sel);
    out->srt_out.resize((size_t)n_sel);
    out->srt_ent.resize((size_t)n_sel * 2);
    {
        std::vector<int> pos(cnt.begin(), cnt.end() - 1);
        for (int64_t p = 0; p < np; p++)
            if (is_short[p]) {
                const int q = pos[b.pair_hap[p]]++;
                const int r = b.pair_read[p];
                out->srt_read[q] = r;
                out->srt_out[q] = (int)p;
                out->srt_ent[2 * (size_t)q] = (int)(TABLE_ZERO_RUN + b.read_off[r] + (int64_t)TABLE_EXTRA_ROWS * r);
                out->srt_ent[2 * (size_t)q + 1] = (int)(b.read_off[r + 1] - b.read_off[r]) + TABLE_EXTRA_ROWS;
            }
    }
    // ---- 2. cut each haplotype's run of reads into tasks of about task_rows read rows
    std::vector<ShortTask> tasks;
    tasks.reserve((size_t)(n_sel / 4 + 16));
    for (int64_t h = 0; h < b.n_haps; h++) {
        const int lo = cnt[h], hi = cnt[h + 1];
        if (lo == hi) continue;
        const int64_t k = b.hap_off[h + 1] - b.hap_off[h];
        ShortTask t = {(int)h, lo, 0, 0};
        for (int q = lo; q < hi; q++) {
            const int r = out->srt_read[q];
            const int l = (int)(b.read_off[r + 1] - b.read_off[r]);
            out->cells += (int64_t)l * k;
            if (l > out->max_read_len) out->max_read_len = l;
            t.n_pairs++;
            t.rows += l;
            if (t.rows >= task_rows) {
                tasks.push_back(t);
                t.pair_first = q + 1; t.n_pairs = 0; t.rows = 0;
            }
        }
        if (t.n_pairs > 0) tasks.push_back(t);
    }
    // ---- 3. pack tasks into warps: duration classes (longest first), lanes bin-packed largest-fit
    const int NCLS = 8 * 40;  // class = floor(8 * log2(duration)), duration < 2^40
    auto cls_of = [&](const ShortTask& t) {
        const double d = (double)(t.rows + TABLE_EXTRA_ROWS * t.n_pairs);
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
    for (size_t i = 0; i < tasks.size(); i++) {
        tb[i] = cls_of(tasks[i]) * 33 + lanes_of(tasks[i]);
        bstart[tb[i] + 1]++;
    }
    for (size_t i = 0; i + 1 < bstart.size(); i++) bstart[i + 1] += bstart[i];
    std::vector<int> ids(tasks.size());
    {
        std::vector<int> pos(bstart.begin(), bstart.end() - 1);
        for (size_t i = 0; i < tasks.size(); i++) ids[pos[tb[i]]++] = (int)i;
    }
    std::vector<int> avail(bstart.begin(), bstart.end() - 1);  // next unused id per bucket
    out->tasks.reserve(tasks.size());
    out->warp_first.reserve(tasks.size() / 2 + 2);
    out->warp_first.push_back(0);
    int cap = 32, bin_steps = 0;
    auto close_bin = [&]() {
        if (cap < 32) {
            out->warp_first.push_back((int)out->tasks.size());
            out->padded_cells += (int64_t)bin_steps * 32 * N2;
        }
        cap = 32; bin_steps = 0;
    };
    for (int c = NCLS - 1; c >= 0; c--) {
        for (;;) {
            int g = cap;
            for (; g >= 1; g--)
                if (avail[c * 33 + g] < bstart[c * 33 + g + 1]) break;
            if (g < 1) {
                // nothing of this class fits the open bin: is anything of this class left at all?
                bool any = false;
                for (int gg = cap + 1; gg <= 32 && !any; gg++) any = avail[c * 33 + gg] < bstart[c * 33 + gg + 1];
                if (!any) break;  // class exhausted: carry the open bin over to the next (shorter) class
                close_bin();
                continue;
            }
            const ShortTask& t = tasks[ids[avail[c * 33 + g]++]];
            out->tasks.push_back(t);
            cap -= g;
            bin_steps = std::max(bin_steps, t.rows + TABLE_EXTRA_ROWS * t.n_pairs + 2 * g - 1);
            if (cap == 0) close_bin();
        }
    }
    close_bin();
}

}  // namespace phmm
