// Internal host-side interface between the API / batcher (api.cpp-ish code in phmm_api.cu) and the
// kernels.  Plain structs of device pointers; nothing here crosses the C ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace phmm {

#ifndef SHORT_NV_
#define SHORT_NV_ 16  // (8 for the columns-per-thread sweep of profiles/r2_gn_sweep.md)
#endif
constexpr int SHORT_NV = SHORT_NV_;        // columns per virtual lane, fp32 short and long kernels
constexpr int SHORT_N2 = 2 * SHORT_NV;    // columns per CUDA lane
constexpr int SHORT_MAX_K = 32 * SHORT_N2;  // 1024: widest haplotype one warp covers
constexpr int CHAIN_NV_F32 = 16;
#ifndef CHAIN_NV_F64_
#define CHAIN_NV_F64_ 8
#endif
constexpr int CHAIN_NV_F64 = CHAIN_NV_F64_;
#ifndef SHORT_WPC_
#define SHORT_WPC_ 4
#endif
constexpr int SHORT_WARPS_PER_CTA = SHORT_WPC_;
constexpr int TABLE_ZERO_RUN = 256;       // all-zero entries at the start of the row-constant table (idle lanes read them)
constexpr int TABLE_EXTRA_ROWS = 3;       // short path: run-in entry in front of, sum and flush entries behind every read's rows (phmm_rowconst.cuh)
// Table positions of the short path.  Every read's run starts at an EVEN entry and has an even length (padded with one
// more all-zero entry where l + 3 is odd), so that the parity of a lane's table position equals the parity of its step:
// the kernel's step loop is unrolled by two and the odd step's entry sits 16 slots behind the even one's, always in
// the same 32-entry block, with no address arithmetic and no run switch in between (phmm_short.cu).
constexpr int TABLE_SLOTS_PER_READ = 4;   // table entries reserved per read beyond its rows
inline __host__ __device__ int64_t table_run_start(int64_t read_off_r, int64_t r) {
    const int64_t b = TABLE_ZERO_RUN + read_off_r + TABLE_SLOTS_PER_READ * r;
    return b + (b & 1);
}
inline __host__ __device__ int table_run_len(int l) { return (l + TABLE_EXTRA_ROWS + 1) & ~1; }
static_assert(TABLE_ZERO_RUN % 2 == 0, "idle lanes walk the zero run two entries per loop iteration");
constexpr int CHAIN_EXTRA_ROWS = 3;       // chain kernel: the same stream

// PHMM_FP32_RESCUE: short-class pairs whose haplotype nearly fills a strip of the long kernel (> 7/8 of the short/long cut) and
// whose read has this many rows or more go through the long kernel as one-strip items: a related read loses 0.2-0.8 bits per
// row, so from here on a growing share would underflow the unrescaled fp32 kernel and be recomputed in fp64 (27 % of the
// 1024 x 1024 pairs of the paper's sweep shape), while a full strip of the long kernel runs at its full rate and never underflows.
constexpr int TALL_MIN_ROWS = 768;
inline __host__ __device__ bool long_class(int64_t k, int64_t l, int long_k, int tall_k) {
    return k > long_k || l > 4096 || (tall_k > 0 && k > tall_k && l >= TALL_MIN_ROWS);
}

struct DevBatch {  // device mirrors of the batch
    const uint8_t *read_bases, *qual_base, *qual_ins, *qual_del, *qual_gcp, *hap_bases;
    const int64_t *read_off, *hap_off;  // device copies of the host offset arrays
    int64_t n_reads, n_haps;
    int n_wild;          // phmm_options.n_is_wildcard: an N (read or haplotype) matches every base
    int64_t table_base;  // absolute table position (table_run_start) of the zero run of the table in use: a slice of reads has its own
};

// ---- fp64 recomputation of short pairs (phmm_rescue.cu)
#ifndef RESCUE_NV_
#define RESCUE_NV_ 32
#endif
constexpr int RESCUE_NV = RESCUE_NV_;           // columns per lane
constexpr int RESCUE_MAX_K = 32 * RESCUE_NV;    // widest haplotype one warp covers in fp64
constexpr int RESCUE_MAX_L = 4096;              // = the short class.  Unrescaled fp64 holds ~600 unrelated rows (3.3 bits lost per row) but
                                                // thousands of related ones; a result below 1e-290 is passed on to the rescaled chain kernel,
                                                // and above it the flushed cells weigh < 2^-36 of the sum

// Device-side binning of the pairs to recompute: bucket = (lane-group size g = ceil(k / RESCUE_NV), read-length class l >> 3),
// g-major, so that the pairs sharing a warp (same g) also have similar lengths and finish together.
constexpr int RESCUE_LCLS = RESCUE_MAX_L / 8 + 1;   // read-length classes
constexpr int RESCUE_NB = 33 * RESCUE_LCLS;         // buckets
enum { RQ_TICKET = RESCUE_NB, RQ_NQUEUE = RESCUE_NB + 1, RQ_FALLBACK = RESCUE_NB + 2, RQ_INTS = RESCUE_NB + 16 };
struct RescueQueue {
    int4* queue;      // (pair, bucket, ticket within the bucket, -)
    int* cnt;         // RQ_INTS ints, zeroed per call: [0..RESCUE_NB) items per bucket, [RQ_TICKET] warp ticket of the kernel,
                      // [RQ_NQUEUE] items in queue, [RQ_FALLBACK] pairs passed on to the chain kernel
};
#ifdef __CUDACC__
__device__ __forceinline__ void rescue_push(const RescueQueue& rq, int pair, int k, int l) {
    const int g = (k + RESCUE_NV - 1) / RESCUE_NV;
    const int bk = g * RESCUE_LCLS + (l >> 3);
    const int n = atomicAdd(rq.cnt + bk, 1);
    const int i = atomicAdd(rq.cnt + RQ_NQUEUE, 1);
    rq.queue[i] = make_int4(pair, bk, n, 0);
}
#endif

struct ShortTask {  // one lane group's work: several reads streamed against one haplotype
    int hap, pair_first, n_pairs, rows;  // rows = sum of the read lengths (reset rows not counted)
    int ents;                            // table entries of its stream = sum of table_run_len(l)
};

struct ShortLaunch {
    const float* table;        // 16 floats (64 bytes) per entry; see k_table_f32 for the layout
    const ShortTask* tasks;    // ordered by warp
    const int* warp_first;     // n_warps+1: first task of each warp
    int n_warps;
    const int2* srt_ent;       // (first table entry, number of entries = table_run_len(read length)) of each sorted pair
    const int* srt_out;        // caller's pair index of each sorted pair
    double* out;
    uint8_t* flags;
    float rescue_thr;          // scaled sums below this (or non-finite) are queued for fp64
    RescueQueue rescue;        // underflowed pairs with k <= RESCUE_MAX_K and l <= RESCUE_MAX_L: sub-warp fp64 kernel
    const int* pair_read;      // device copy of the caller's pair list (the queue is binned by read length)
    int* rescue_count;         // the others: device counter and
    int* rescue_list;          // caller pair indices for the rescaled chain kernel
};

struct ChainItem {  // one strip (32 lanes x 2NV columns) of one pair, run concurrently with its neighbours
    int pair;        // caller's pair index
    int strip;       // strip number, 0 = leftmost
    int prog0;       // index of the pair's first progress counter (one per strip boundary)
    int pad;
    int64_t buf0;    // index (in boundary blocks) of the pair's first boundary buffer
};

struct ChainLaunch {
    const ChainItem* items;    // device; or, with items_are_pairs, a plain int array of caller pair indices
                               // (each such pair is run by one warp, its strips in sequence)
    const int* n_items;        // device (may be produced by an earlier kernel)
    int* ticket;               // device, zeroed before the launch
    const int* pair_read;      // device copies of the caller's pair list
    const int* pair_hap;
    const double* lut;         // 256 entries 10^(-q/10)
    void* boundary;            // concurrent strips: boundary buffers; sequential: 2 x scratch_blocks per warp of the grid
    int64_t scratch_blocks;
    int* progress;             // concurrent strips: rows published per boundary
    double* out;
    uint8_t* flags;
    uint8_t flag_bits;         // written to flags[pair]
    int log2C;                 // scale constant C = 2^log2C of Eq.1 (0 for the rescaled kernels)
    int long_k;                // items_are_pairs: pairs with a haplotype longer than this (or a read over 4096) also get PHMM_FLAG_LONG
    int tall_k;                // ... and so do pairs with a haplotype longer than this and a read of TALL_MIN_ROWS or more (0: rule off)
};

struct LongLaunch {  // fp32 long path (phmm_long.cu): strips of 32 lanes x 32 columns, table-driven like the short kernel
    const float* table;        // the row-constant table of k_table_f32 (must cover the reads of every long pair)
    const ChainItem* items;    // strip-major; buf0 = index of the pair's first boundary record
    const int* n_items;
    int* ticket;               // zeroed before the launch
    const int* pair_read;
    const int* pair_hap;
    float4* records;           // per pair and strip boundary: l + 3 records {s, T, exponent, -}
    float4* totals;            // per progress counter: the Eq.4 total of the strips up to this one {lo, hi of a double, exponent, -}
    int* progress;             // per pair and strip: entries published (l + 4 once the total is there); zeroed before the launch
    double* out;
    uint8_t* flags;
    uint8_t flag_bits;
    int publish;               // entries per progress publication: a power of two >= 16
    int* fallback_count;       // pairs whose fp32 result is not a normal positive number: list for the fp64 chain kernel
    int* fallback_list;
    const uint8_t* risk;       // per read, by launch_read_risk: 255 = fp32's per-lane range may not do (straight to fp64), else the read's smallest GCP quality
};
cudaError_t launch_read_risk(const DevBatch& b, int qual_offset, int64_t r0, int64_t r1, uint8_t* risk, cudaStream_t st);
cudaError_t launch_long_f32(const DevBatch& b, const LongLaunch& p, int grid_ctas, cudaStream_t st);
int long_ctas_per_sm();
int long_warps_per_cta();

constexpr int RESCUE_PLAN_INTS = 68 + RESCUE_NB;  // [0..33] first warp of bucket g, [34..67] first list slot of bucket g, [68..) first slot of each (g, length class) bucket
struct RescueLaunch {
    RescueQueue queue;
    int max_queue;             // upper bound of the queue length (grid of the scatter kernel)
    const int* enqueue_pairs;  // PHMM_FP64 mode: device list of pairs to queue first (else nullptr)
    int n_enqueue;
    int* plan;                 // RESCUE_PLAN_INTS ints of scratch
    int* sorted;               // max_queue ints of scratch
    const void* table;         // PHMM_FP32_RESCUE: the fp32 row-constant table of the short path (the recomputation runs in
                               // double on the fp32-rounded constants: it needs the range, not the precision);
    int table_f64;             // PHMM_FP64: the table of launch_table_f64 (constants in double)
    const int* pair_read;
    const int* pair_hap;
    const double* lut;
    double* out;
    uint8_t* flags;
    uint8_t flag_bits;
    int* fallback_count;       // pairs the unrescaled fp64 pass could not represent: queued for the chain kernel
    int* fallback_list;
};
cudaError_t launch_rescue_f64(const DevBatch& b, const RescueLaunch& r, int grid_ctas, cudaStream_t st);
int rescue_ctas_per_sm();
// PHMM_FP64: the row-constant table in double for the sub-warp kernel (64 bytes per entry, field-major blocks of 32 entries)
cudaError_t launch_table_f64(const DevBatch& b, const double* lut, double* table, int64_t r0, int64_t r1, int max_read_len, cudaStream_t st);

cudaError_t launch_lut_table(const DevBatch& b, const double* lut, float* table, int64_t r0, int64_t r1, int max_read_len, cudaStream_t st);
cudaError_t launch_short_f32(const DevBatch& b, const ShortLaunch& p, cudaStream_t st);
// debug pass (phmm_options.validate): *d_err |= 1 bad base, 2 quality below the offset, 4 iota + delta >= 1
cudaError_t launch_validate(const DevBatch& b, const double* lut, int64_t read_lo, int64_t read_hi, int64_t hap_lo, int64_t hap_hi, int qual_offset, int* d_err, cudaStream_t st);
// rescue_from_list: items are taken from p.items[...] as plain pair indices in `rescue_list` form
cudaError_t launch_chain(const DevBatch& b, const ChainLaunch& p, bool fp64, bool items_are_pairs, int grid_ctas,
                         cudaStream_t st);
int chain_ctas_per_sm(bool fp64);
int chain_warps_per_cta(bool fp64);
size_t chain_block_bytes(bool fp64);  // bytes of one 32-row boundary block
int chain_strip_cols(bool fp64);      // haplotype columns covered by one strip (fp32 long kernel: SHORT_MAX_K)
// PHMM_FP64 long pairs as concurrent strips (phmm_long64.cu): ChainLaunch as for the chain kernel (items, progress, boundary
// blocks of long64_block_bytes()), constants from the double table of launch_table_f64
cudaError_t launch_long_f64(const DevBatch& b, const ChainLaunch& p, const double* table, int grid_ctas, cudaStream_t st);
int long64_ctas_per_sm();
size_t long64_block_bytes();
int long64_strip_cols();

}  // namespace phmm
