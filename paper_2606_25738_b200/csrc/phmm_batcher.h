// Host-side batcher ("pairs are batched according to their
// lengths and run on dedicated kernels").  Pure host C++; no CUDA types.
//
// Short pairs (haplotype fits one warp) are grouped BY HAPLOTYPE: a "task" is a run of reads that
// are all aligned against the same haplotype by one group of g = ceil(k / columns-per-lane)
// consecutive lanes, the reads streaming through the lanes back to back, so the systolic
// fill/drain (2g steps) is paid once per task instead of once per pair.  Tasks are then packed
// into 32-lane warps: tasks of similar duration share a warp (all groups of a warp run the same
// number of steps) and the lane counts are bin-packed (largest-fit-first).
#pragma once
#include <stdint.h>
#include <vector>

#include "phmm_kernels.h"

#include <algorithm>
#include <thread>

namespace phmm {

// fn(t, begin, end) over [0, n) in contiguous chunks on up to BATCHER_THREADS threads (the caller's included)
constexpr int BATCHER_THREADS = 16;
template <typename F> inline int parallel_chunks(int64_t n, int64_t min_chunk, F fn) {
    int T = (int)std::min<int64_t>(BATCHER_THREADS, std::max<int64_t>(1, n / min_chunk));
    const unsigned hw = std::thread::hardware_concurrency();
    if (hw > 0 && (unsigned)T > hw) T = (int)hw;
    const int64_t per = (n + T - 1) / T;
    std::vector<std::thread> th;
    for (int t = 1; t < T; t++) th.emplace_back([=]() { fn(t, std::min(n, t * per), std::min(n, (t + 1) * per)); });
    fn(0, 0, std::min(n, per));
    for (auto& x : th) x.join();
    return T;
}



struct HostBatchView {
    int64_t n_reads, n_haps, n_pairs;
    const int64_t *read_off, *hap_off;
    const int32_t *pair_read, *pair_hap;
};

struct ShortPlan {
    std::vector<ShortTask> tasks;   // ordered by warp
    std::vector<int> warp_first;    // n_warps + 1
    std::vector<int> srt_ent;       // 2 ints per sorted pair: first table entry of its read's run, entries of the run (table_run_len)
    std::vector<int> srt_out;       // caller's pair index per sorted pair
    int64_t cells = 0;              // real cells of the short pairs
    int64_t padded_cells = 0;       // lane-cells swept: sum over warps of steps * 32 lanes * columns-per-lane
    int max_read_len = 0;
    // scratch of plan_tasks, kept between calls so that a steady stream of equal-sized batches touches no fresh memory
    struct PackPart {
        std::vector<ShortTask> tasks;   // in packing order
        std::vector<int> warp_end;      // one past the last task of each warp
        std::vector<int> warps_after;   // [c]: warps closed once the classes >= c are done
        std::vector<int> tb, ids, bstart, avail;
        int64_t padded = 0;
    };
    std::vector<ShortTask> tmp_tasks;
    std::vector<ShortTask> tmp_cut[BATCHER_THREADS];
    PackPart tmp_pack[BATCHER_THREADS];
};

// is_short[p] != 0 selects the pairs to plan.  cols_per_lane = 2*NV of the kernel.
void plan_short(const HostBatchView& b, const uint8_t* is_short, int cols_per_lane, int task_rows, ShortPlan* out);
// The three stages of plan_short, for batches that are processed in slices of reads (phmm_api.cu):
int slice_reads(const HostBatchView& b, int64_t max_table_bytes, int min_slices, std::vector<int64_t>* bound);
void bucket_pairs_by_slice(const HostBatchView& b, const uint8_t* read_slice, int n_slices, std::vector<int>* out,
                           std::vector<int64_t>* slice_first);
void sort_ids_by_hap(const HostBatchView& b, const int* ids, int64_t n, std::vector<int>* sorted);
void plan_tasks(const HostBatchView& b, const int* sorted, int64_t n_sel, int64_t table_base, int cols_per_lane, int task_rows,
                ShortPlan* out);

// Validation of offsets / indices / lengths; returns a PHMM_E_* code or 0.
int validate_batch(const HostBatchView& b);

}  // namespace phmm
