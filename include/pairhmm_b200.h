/*
 * pairhmm_b200.h -- C ABI of libpairhmm_b200.so: batch PairHMM forward on one NVIDIA B200 (sm_100a).
 *
 * What the library computes (reference/PAPER.md = arxiv/paper_2606_25738, "Endeavor"):
 *   for every (read, haplotype) pair of a batch, the PairHMM forward likelihood
 *       L = sum_{j=1..k} ( M_{l,j} + I_{l,j} ) / C                        (Eq.4)
 *   of the three-state recurrence (Eq.2) started from Eq.1 with the
 *   emission prior of Eq.3 and per-read-position transition probabilities derived
 *   from the insertion / deletion / gap-continuation qualities (Listing 2
 *   :293-295).  The kernels evaluate the paper's row-wise reformulation (Eq.6-7, PAPER.md:99-121,
 *   D eliminated / carried as a running weighted sum) as a skewed systolic wavefront; the result
 *   is the same number.  Output is log10 L (the paper returns the raw scaled sum).
 *
 * Conventions
 *   - "host" / "device" below says where a pointer must live.  Device buffers are allocated by
 *     the caller (e.g. through PyTorch); the library only reads inputs and writes the outputs.
 *   - Bases are compared literally (Eq.3: r_i == h_j) over the alphabet A, C, G, T, N: an N matches an N and nothing
 *     else (reading G17; phmm_options.n_is_wildcard makes it match everything).  Any other byte is treated
 *     as N; phmm_options.validate rejects it.
 *   - Qualities are RAW Phred bytes 0..93 (NOT ASCII+33 unless phmm_options.qual_offset says so; reading G5):
 *        eps = 10^(-Qbase/10), iota = 10^(-Qins/10), delta = 10^(-Qdel/10), gamma = 10^(-Qgcp/10);
 *        T_MM = 1-iota-delta, T_MI = iota, T_MD = delta, T_II = T_DD = gamma, T_IM = T_DM = 1-gamma,
 *     all taken at the read position (row) of the cell being written.  Precondition: iota+delta < 1.
 *   - All calls are thread-compatible per context (one context = one caller at a time).  Calls on different streams
 *     of one context are ordered by the library (they share the context's workspaces).
 *   - Every function returns PHMM_OK (0) or a negative PHMM_E_* code; nothing throws or aborts.
 *     A call that fails argument validation writes nothing.
 */
#ifndef PAIRHMM_B200_H
#define PAIRHMM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PHMM_VERSION 1

/* error codes */
#define PHMM_OK 0
#define PHMM_E_ARG (-1)          /* null pointer, negative size, unknown precision */
#define PHMM_E_OFFSETS (-2)      /* offsets not monotone, or a pair index out of range */
#define PHMM_E_EMPTY (-3)        /* a pair references a read or haplotype of length 0 */
#define PHMM_E_TOOLONG (-4)      /* a sequence exceeds PHMM_MAX_LEN */
#define PHMM_E_CUDA (-5)         /* a CUDA runtime call failed (see phmm_last_cuda_error) */
#define PHMM_E_NOMEM (-6)        /* host or device allocation failed */
#define PHMM_E_UNSUPPORTED (-7)  /* device is not sm_100, or option not supported */

#define PHMM_MAX_LEN (1 << 24)   /* longest read / haplotype accepted, in bases */

/* precision modes of phmm_forward_batch */
#define PHMM_FP32_RESCUE 0 /* fp32 recurrence; pairs whose fp32 result underflows are redone in fp64 */
#define PHMM_FP64 1        /* fp64 recurrence for every pair */

/* bits of the per-pair output flags */
#define PHMM_FLAG_RESCUED 1u /* PHMM_FP32_RESCUE only: pair was recomputed in fp64 */
#define PHMM_FLAG_LONG 2u    /* pair went through the multi-warp / multi-CTA rescaled wavefront path */
#define PHMM_FLAG_RANGE 4u   /* phmm_forward_batch_noalloc only: the likelihood left the range of unscaled double (value unusable) */

typedef struct phmm_ctx phmm_ctx; /* opaque; owns workspaces, internal streams, the last stats */

/* Tunables; zero-initialise and set `size = sizeof(phmm_options)`, fields left 0 take defaults. */
typedef struct phmm_options {
    uint32_t size;
    /* fp32 rescue criterion (reading G16): the fp32 pass runs with scale constant
     * C = 2^120; a pair is redone in fp64 iff its scaled sum is not finite or is
     * < 2^rescue_log2_threshold.  Default -90  (<=> L < 2^-210 ~ 10^-63.2). */
    int32_t rescue_log2_threshold;
    /* haplotypes longer than this many bases (or reads longer than 4096) use the long, rescaled multi-strip path;
     * default and maximum 1024 (= 32 lanes x 32 columns, what one warp of the short kernel covers).  In PHMM_FP32_RESCUE
     * pairs with a haplotype over 7/8 of it and a read of 768 bases or more take that path too (as one strip): such reads
     * increasingly underflow the unrescaled fp32 kernel.  Either way the pair carries PHMM_FLAG_LONG. */
    int32_t long_min_hap_len;
    /* target number of read rows per short-path task (a task streams several reads of one
     * haplotype through one lane group); 0 = chosen per batch between 1024 and 8192 so that the
     * GPU still gets several waves of warps */
    int32_t task_rows;
    /* workspace budget, in bytes, of the row-constant table (64 bytes per read base + 256 per read).  A batch that
     * needs more is processed in slices of reads inside the call (phmm_stats.n_slices), each with a table within the
     * budget; PHMM_E_NOMEM only if a single read does not fit.  Default 4 GiB, minimum 4 MiB. */
    int64_t max_table_bytes;
    /* non-zero: bracket every kernel family of a call with CUDA events on the caller's stream; the
     * durations appear in phmm_stats.ms_* (phmm_get_stats synchronises the last event).  Default 0. */
    int32_t profile_events;
    /* non-zero: before anything is launched, one device pass checks the payload's preconditions -- every base is one of
     * A C G T N, every quality byte is >= qual_offset, and iota + delta < 1 on every read position -- and the call returns
     * PHMM_E_ARG, having written nothing, if one is violated (it synchronises the stream once).  Default 0: the payload
     * is trusted (SURVEY.md section 8(b) "Errors"). */
    int32_t validate;
    /* Compatibility semantics (none of them changes a config of
     * BASELINE.json, all default to 0 = the literal reading of Eq.3 on raw Phred bytes):
     *   qual_offset     subtracted from every quality byte before use (33 for FASTQ / ASCII-encoded qualities, PAPER.md:76
     *                   "Q - 33"); bytes below it count as quality 0
     *   min_base_qual   base qualities below this value (after the offset) are raised to it (a quality floor)
     *   n_is_wildcard   non-zero: an N in the read or in the haplotype matches every base (prior 1 - eps), instead of
     *                   matching only another N */
    int32_t qual_offset;
    int32_t min_base_qual;
    int32_t n_is_wildcard;
} phmm_options;

/* One batch, CSR layout, natural order (a read, a haplotype and four
 * read-length quality strings per pair; here reads and haplotypes are stored once and pairs
 * reference them by index). */
typedef struct phmm_batch {
    int64_t n_reads, n_haps, n_pairs;
    const int64_t* h_read_off;   /* host,   n_reads+1: byte offset of each read in the d_* read arrays */
    const int64_t* h_hap_off;    /* host,   n_haps+1 : byte offset of each haplotype in d_hap_bases */
    const uint8_t* d_read_bases; /* device, h_read_off[n_reads] bytes */
    const uint8_t* d_qual_base;  /* device, same length: raw Phred base qualities */
    const uint8_t* d_qual_ins;   /* device, same length: insertion gap-open qualities */
    const uint8_t* d_qual_del;   /* device, same length: deletion gap-open qualities */
    const uint8_t* d_qual_gcp;   /* device, same length: gap-continuation qualities */
    const uint8_t* d_hap_bases;  /* device, h_hap_off[n_haps] bytes */
    const int32_t* h_pair_read;  /* host,   n_pairs: read index of each pair */
    const int32_t* h_pair_hap;   /* host,   n_pairs: haplotype index of each pair */
} phmm_batch;

/* Counters of the most recent phmm_forward_batch / phmm_forward_batch_host on a context. */
typedef struct phmm_stats {
    int64_t n_pairs;
    int64_t cells;              /* sum over pairs of read_len * hap_len (the TCUPS numerator) */
    int64_t n_short_pairs;      /* pairs run by the sub-warp systolic kernel */
    int64_t n_long_pairs;       /* pairs run by the CTA-chain wavefront kernel */
    int64_t n_rescued;          /* PHMM_FP32_RESCUE: pairs recomputed in fp64 (valid after the stream is synchronised) */
    int64_t short_cells;        /* real cells of the short-path pairs */
    int64_t short_padded_cells; /* lane-cells the short kernel actually swept (padding, fill/drain included) */
    int64_t n_kernel_launches;  /* kernels enqueued by the call */
    int64_t table_bytes;        /* row-constant table size of the call */
    double host_batch_ms;       /* host time spent in the batcher */
    int32_t n_short_warps;      /* warp tasks of the short kernel */
    int32_t n_slices;           /* slices of reads the call was processed in (phmm_options.max_table_bytes) */
    /* device time per kernel family, milliseconds, CUDA events on the caller's stream; filled only
     * with phmm_options.profile_events (else 0).  ms_short is the sub-warp systolic fp32 kernel, ms_table
     * the row-constant prologue, ms_rescue the fp64 (rescue / PHMM_FP64 short) chain launch, ms_long
     * the concurrent-strip wavefront launch. */
    double ms_table, ms_short, ms_rescue, ms_long;
} phmm_stats;

/* Create a context on CUDA device `device`.  opt may be NULL.  Fails with PHMM_E_UNSUPPORTED on a
 * device whose compute capability is not 10.x. */
int phmm_create(phmm_ctx** ctx, int device, const phmm_options* opt);
int phmm_destroy(phmm_ctx* ctx);

/* log10 likelihood of every pair of `b`, in the caller's pair order.
 *   precision    PHMM_FP32_RESCUE or PHMM_FP64
 *   d_out_log10  device, n_pairs doubles (written)
 *   d_out_flags  device, n_pairs bytes (written; may be NULL)
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream).  The call enqueues all device work on
 *                it (internally forked streams are joined back) and returns without synchronising
 *                the device; outputs are valid once the caller has synchronised `cuda_stream`.
 * The host batcher ("batched according to their lengths") runs inside the call.
 * For valid input every output is finite. */
int phmm_forward_batch(phmm_ctx* ctx, const phmm_batch* b, int precision, double* d_out_log10,
                       uint8_t* d_out_flags, void* cuda_stream);

/* Same computation with ALL buffers on the host (the d_* members of `b` are host pointers, out
 * pointers are host): the library copies the payload to the device, runs phmm_forward_batch, copies
 * the results back and synchronises.  This is the end-to-end entry ("with transfer").
 * The reads are processed in slices (at least one per 48 MB of read payload, and as many as the table budget asks for):
 * the copy of a slice's reads and its host plan run under the kernels of the slice before; results and flags are the
 * same as for one call with device buffers.  phmm_get_stats afterwards reports the sums over the slices.  The device work
 * runs on a stream of the context, not on the caller's. */
int phmm_forward_batch_host(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out_log10,
                            uint8_t* h_out_flags);

/* The streaming form of phmm_forward_batch_host (the "with transfer" convention; SURVEY.md section 8(f)
 * item 2): enqueues the copies in, the kernels and the copies out of one batch and returns with a ticket; the results are
 * in h_out_log10 / h_out_flags once phmm_wait_host(ctx, ticket) has returned.  Up to two calls are in flight per context:
 * a third call first waits for the oldest one.  With a second call submitted before the first is waited for, the copies
 * and the host plan of one batch run under the kernels of the batch before it (the context keeps two device copies of
 * payload and outputs); the reads of a call are then not sliced unless the table budget asks for it.
 *   - Every host array of `b` (offsets, pair lists and the payload), h_out_log10 and h_out_flags must stay valid and
 *     unchanged / unread until the ticket has been waited for.  The payload and the output arrays should be pinned
 *     (cudaHostAlloc / cudaHostRegister) memory: with pageable memory the copies are staged by the driver and the call does
 *     not return before they are done, so nothing overlaps (the results are the same).
 *   - Results, flags and error codes are those of phmm_forward_batch_host.  An error is reported by the call that finds it
 *     (arguments, offsets, allocation: the submitting call, which then leaves nothing in flight for its ticket).
 *   - phmm_get_stats reports the batch of the most recently waited ticket (per-family kernel times: of the most recently
 *     submitted call that has completed).
 *   - phmm_wait_host on a ticket that has already been waited for (or whose set a later call has taken over, which
 *     implies it completed) returns PHMM_OK at once.  One caller thread at a time per context, as for every entry. */
int phmm_forward_batch_host_async(phmm_ctx* ctx, const phmm_batch* b, int precision, double* h_out_log10,
                                  uint8_t* h_out_flags, int* ticket);
int phmm_wait_host(phmm_ctx* ctx, int ticket);

/* Statistics of the most recent call on the context.  Waits for that call's device work to complete (the rescue count and
 * the per-family times are only known then), on whatever stream the call was issued. */
int phmm_get_stats(phmm_ctx* ctx, phmm_stats* out);
const char* phmm_strerror(int code);
/* cudaError_t value of the last failing CUDA call on this context (0 if none). */
int phmm_last_cuda_error(phmm_ctx* ctx);

/* Measured non-tensor arithmetic peak of the device, used as roofline denominator (BASELINE.json
 * north_star: "fraction of the FP32 (and FP64) non-tensor roofline").  kind: 0 = scalar FFMA,
 * 1 = packed FFMA2 (fma.rn.f32x2), 2 = DFMA.  Writes TFLOP/s (2 flops per lane-FMA) of a kernel of
 * independent FMA chains, best of `reps` launches, timed with CUDA events. */
int phmm_measure_peak(int device, int kind, int reps, double* out_tflops);

/* Host batcher only (no device is touched): the work plan the short path
 * would use for the short-class pairs of `b` in PHMM_FP32_RESCUE: haplotype length <= long_min_hap_len (0 = default 1024), read
 * length <= 4096, and not both haplotype > 7/8 of the cut and read >= 768 (phmm_options.long_min_hap_len).  Only the host arrays of `b` are read (offsets, pair list).  Outputs, all host, caller-owned:
 *   plan_counts[4]   = { n_warps, n_tasks, n_sorted_pairs, columns per lane }
 *   warp_first       n_warps + 1 ints: first task of each warp              (capacity cap_warps + 1)
 *   tasks            4 ints per task: haplotype, first sorted pair, number of pairs, read rows (capacity 4 * cap_tasks)
 *   sorted_pair      caller's pair index of each sorted pair                 (capacity cap_pairs)
 * Any output pointer may be NULL (then only plan_counts is written).  Returns PHMM_E_NOMEM if a capacity
 * is too small, validation errors as phmm_forward_batch.  For tests and for sizing workspaces. */
int phmm_plan_host(const phmm_batch* b, int long_min_hap_len, int task_rows, int64_t* plan_counts, int32_t* warp_first,
                   int64_t cap_warps, int32_t* tasks, int64_t cap_tasks, int32_t* sorted_pair, int64_t cap_pairs);

/* Host batcher only (no device is touched): how phmm_forward_batch would cut the reads of `b` into slices for a table budget
 * of max_table_bytes (0 = default 4 GiB) and at least min_slices slices.  Only the host arrays of `b` are read.
 *   n_slices     number of slices (written)
 *   read_first   n_slices + 1 read indices: slice s covers the reads [read_first[s], read_first[s+1])   (may be NULL)
 *   pair_count   pairs of each slice (a pair belongs to the slice of its read)                           (may be NULL)
 *   cap_slices   capacity of pair_count (read_first needs cap_slices + 1); PHMM_E_NOMEM if too small */
int phmm_plan_slices_host(const phmm_batch* b, int64_t max_table_bytes, int min_slices, int64_t* n_slices,
                          int64_t* read_first, int64_t* pair_count, int64_t cap_slices);

/* ---- An entry point that allocates nothing (no cudaMalloc / cudaFree, no context): for callers under CUDA graph capture,
 * serving loops and harnesses that forbid allocation.  It computes what phmm_forward_batch(..., PHMM_FP64, ...) computes
 * for SHORT-CLASS pairs only -- every pair's haplotype <= 1024 bases and read <= 4096 -- with default options (raw Phred
 * qualities, literal N), in unscaled double (Eq.1-4 with C = 2^1000): the same kernel arithmetic as the library's fp64
 * sub-warp kernel.  Its scratch (the quality tables and the row-constant table, 64 bytes per read row) is a file-scope
 * device array of PHMM_NOALLOC_SCRATCH_BYTES that every GPU loading the library holds until exit; a batch fits if
 * sum over reads of (length + 4) + 258 <= phmm_noalloc_limits()' max_table_entries (131008).
 *   b             as for phmm_forward_batch: host offsets and pair lists (read for validation and sizing), device payload
 *   d_read_off, d_hap_off, d_pair_read, d_pair_hap   device copies of b's four host arrays (the caller's, n+1 / n_pairs long)
 *   d_out_log10   device, n_pairs doubles (written)
 *   d_out_flags   device, n_pairs bytes (written; may be NULL): 0, or PHMM_FLAG_RANGE where L < 1e-290 * 2^-1000 (about
 *                 10^-591: e.g. unrelated reads over ~600 bases) -- use phmm_forward_batch for such pairs
 * Returns PHMM_E_TOOLONG, having launched nothing, if a sequence or the batch exceeds the limits above; validation errors
 * as phmm_forward_batch.  Asynchronous on cuda_stream.  Every call shares the one scratch array: calls that overlap on
 * the GPU (different streams without a dependency, or two processes' worth of threads) race -- serialise them.  The
 * first call on a device does a one-time set-up (cudaGetSymbolAddress, a 4 KB synchronous copy); call
 * phmm_noalloc_setup(device) beforehand where that must not happen inside the call (graph capture). */
#define PHMM_NOALLOC_SCRATCH_BYTES (8u << 20)
int phmm_noalloc_setup(int device);
int phmm_noalloc_limits(int64_t* max_table_entries, int32_t* max_hap_len, int32_t* max_read_len);
int phmm_forward_batch_noalloc(int device, const phmm_batch* b, const int64_t* d_read_off, const int64_t* d_hap_off,
                               const int32_t* d_pair_read, const int32_t* d_pair_hap, double* d_out_log10,
                               uint8_t* d_out_flags, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PAIRHMM_B200_H */
