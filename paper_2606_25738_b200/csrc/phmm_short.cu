// Short-pair path: row-constant table prologue + the sub-warp systolic fp32 kernel.
//
// Hot path rows of SURVEY.md section 8(a): a1 (quality -> row constants: table kernel), a2 (haplotype
// staging: match words / fp16 base codes in registers), a3/a4 (row updates), a5 (lane-to-lane carry: 2 shuffles
// per row), a9 (final reduction, log10), a10 (underflow detection -> rescue queue).
#include "phmm_engine.cuh"
#include "phmm_kernels.h"
#include "phmm_rowconst.cuh"
#include "phmm_table.cuh"
#include <type_traits>

// Tunables, each with the measurement that chose it (configs[1], in-kernel TCUPS)
#ifndef SHORT_L2_PREFETCH
#define SHORT_L2_PREFETCH 1  // table loads carry the L2 256-byte prefetch hint: +0.6 %
#endif
#ifndef SHORT_L2_LINE_PREFETCH
#define SHORT_L2_LINE_PREFETCH 0  // entries ahead (0 = off)
#endif
#ifndef SHORT_MIN_CTAS
#define SHORT_MIN_CTAS 3  // resident CTAs per SM the register allocation is held to (3 x 128 threads -> <= 168 registers); 4 x 128 registers spills: 3.17 vs 3.36 TCUPS
#endif

namespace phmm {

// ------------------------------------------------------------------ a1: row-constant table
// Each 64-byte table entry holds the constants of entry e (for the .x half) and of entry e-1 (for .y; zero
// for e = 0), already paired the way FFMA2 wants them:
//   float4 0: gamma.x gamma.y A.x A.y | 1: C.x C.y G.x G.y | 2: pm.x px.x pm.y px.y | 3: word 0 0 0
// word = entry_word16 of e | entry_word16 of e-1 << 16 (phmm_rowconst.cuh): what HSETP2 compares with the per-column
// codes in the high bytes, the meta bytes in the low ones.
// The table starts with TABLE_ZERO_RUN all-zero entries (what idle lanes fetch); read r's run starts at
// entry table_run_start(read_off[r], r) (even; phmm_kernels.h).  Constants are formed in double from the
// 10^(-q/10) table and rounded once ("q32" table; Listing 2 :293-295 for which
// qualities enter which transition).  One warp per read and chunk of 1024 entries (blockIdx.y = chunk).
// Memory layout: the entries are permuted inside blocks of 32 so that the lanes of a warp, which read entries
// two apart (lane L's .x half is 2L entries behind lane 0's), touch consecutive 16-byte slots: block = 2 KB =
// 4 chunk planes (the four float4 of an entry) x 2 parities x 16 slots.  A lane-strided LDG.128 then costs
// ~4 L1 wavefronts instead of 32 (ncu: l1tex throughput 90 % -> see profiles/).
constexpr int TABLE_CHUNK_ENTRIES = 1024;
__global__ void __launch_bounds__(256) k_table_f32(DevBatch b, const double* __restrict__ lut, float* __restrict__ table, int64_t r0, int64_t r1) {
    const int64_t r = r0 + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (r >= r1) return;
    const int lane = threadIdx.x & 31;
    const int64_t off = b.read_off[r];
    const int l = (int)(b.read_off[r + 1] - off);
    float4* dst = reinterpret_cast<float4*>(table);
    const int64_t first = table_run_start(off, r) - b.table_base;
    const int e_hi = min(table_run_len(l), ((int)blockIdx.y + 1) * TABLE_CHUNK_ENTRIES);
    for (int e = (int)blockIdx.y * TABLE_CHUNK_ENTRIES + lane; e < e_hi; e += 32) {  // (an entry behind the flush entry is all zero too)
        const RowC x = row_constants(b, lut, off, l, e, true), y = row_constants(b, lut, off, l, e - 1, true);
        float4* d = dst + table_slot(first + e);
        d[0 * TABLE_CHUNK_STRIDE] = make_float4((float)x.gam, (float)y.gam, (float)x.A, (float)y.A);
        d[1 * TABLE_CHUNK_STRIDE] = make_float4((float)x.C, (float)y.C, (float)x.G, (float)y.G);
        d[2 * TABLE_CHUNK_STRIDE] = make_float4((float)x.pm, (float)x.px, (float)y.pm, (float)y.px);
        d[3 * TABLE_CHUNK_STRIDE] = make_float4(__uint_as_float(entry_word16(x) | (entry_word16(y) << 16)), 0.f, 0.f, 0.f);
    }
}

cudaError_t launch_lut_table(const DevBatch& b, const double* lut, float* table, int64_t r0, int64_t r1, int max_read_len, cudaStream_t st) {
    if (r1 <= r0) return cudaSuccess;
    const int wpb = 8;
    int64_t grid = (r1 - r0 + wpb - 1) / wpb;
    const int chunks = (table_run_len(max_read_len) + TABLE_CHUNK_ENTRIES - 1) / TABLE_CHUNK_ENTRIES;
    // the zero run (whole 32-entry blocks) that idle lanes walk: cleared on every call, whatever the batch size
    cudaError_t e = cudaMemsetAsync(table, 0, (size_t)TABLE_ZERO_RUN * 64, st);
    if (e != cudaSuccess) return e;
    k_table_f32<<<dim3((unsigned)grid, (unsigned)chunks), wpb * 32, 0, st>>>(b, lut, table, r0, r1);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ the short kernel
// Per lane, the .x half walks its task's stream of table entries (run of read 1, run of read 2, ...) starting
// 2*lg steps after the group's first lane.  While it waits, and after its stream has ended, a lane walks the
// zero run at the start of the table (all-zero constants decay T and J to 0), so the fetch needs no special
// cases.  Entries are loaded one step ahead into two alternating register sets (the step loop is unrolled by two, so
// no register is ever copied).
struct Cursor {
    int pos, end;        // next entry to fetch, one past the last entry of the current run
    int npos, nend;      // the run after it: the next read of the task, or the zero run
    int q;               // reads of the task already handed to (npos, nend)
};

// HS = false (match words instead of fp16 column codes) only under phmm_options.n_is_wildcard, where a haplotype N has to
// match every read base -- something one fp16 equality cannot say
template <int NV, bool HS>
__global__ void __launch_bounds__(SHORT_WARPS_PER_CTA * 32, SHORT_MIN_CTAS) k_short_f32(DevBatch b, ShortLaunch p) {
    typedef Lane2<float, NV, HS> L;  // HSETP2 predicates (2.78 vs 2.60 TCUPS with bit tests), Eq.4 through the s chain
    constexpr int N2 = 2 * NV;
    const int warp = blockIdx.x * SHORT_WARPS_PER_CTA + (threadIdx.x >> 5);
    if (warp >= p.n_warps) return;
    const int lane = threadIdx.x & 31;

    // ---- which task does this lane belong to?  tasks of a warp occupy consecutive lane ranges
    const int t0 = p.warp_first[warp], nt = p.warp_first[warp + 1] - t0;
    ShortTask tk = {0, 0, 0, 0, 0};
    int k = 0, g = 0;
    if (lane < nt) {
        tk = p.tasks[t0 + lane];
        k = (int)(b.hap_off[tk.hap + 1] - b.hap_off[tk.hap]);
        g = (k + N2 - 1) / N2;
    }
    int start = g;  // inclusive scan -> exclusive start
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int v = __shfl_up_sync(PHMM_FULL, start, o);
        if (lane >= o) start += v;
    }
    start -= g;
    int ti = -1;
    for (int i = 0; i < nt; i++) {
        int s = __shfl_sync(PHMM_FULL, start, i);
        int gi = __shfl_sync(PHMM_FULL, g, i);
        if (lane >= s && lane < s + gi) ti = i;
    }
    const int src = ti < 0 ? 0 : ti;
    const int m_hap = __shfl_sync(PHMM_FULL, tk.hap, src), m_first = __shfl_sync(PHMM_FULL, tk.pair_first, src);
    int m_np = __shfl_sync(PHMM_FULL, tk.n_pairs, src), m_ents = __shfl_sync(PHMM_FULL, tk.ents, src);
    int m_k = __shfl_sync(PHMM_FULL, k, src);
    const int m_start = __shfl_sync(PHMM_FULL, start, src), m_g = __shfl_sync(PHMM_FULL, g, src);
    if (ti < 0) { m_np = 0; m_ents = 0; m_k = 0; }
    const int lg = ti < 0 ? 0 : lane - m_start;
    const bool is_first = (ti < 0) || lg == 0;
    const bool is_last = (ti >= 0) && lg == m_g - 1;
    const uint32_t sum_bit = is_last ? (META_SUM << 16) : 0u;
    const bool full_last = m_k == m_g * N2;  // no column behind the haplotype's last one

    // ---- number of steps of this warp: the last lane's .y half finishes the last entry of its stream
    int steps = (ti < 0) ? 0 : m_ents + 2 * m_g - 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) steps = max(steps, __shfl_xor_sync(PHMM_FULL, steps, o));

    L ln;
    ln.init();
    ln.load_hap(b.hap_bases + (ti < 0 ? 0 : b.hap_off[m_hap]), m_k, lg * N2, b.n_wild != 0);
    const float Cok = (float)(ldexp(1.0, 120) / (double)(m_k > 0 ? m_k : 1));  // Eq.1: C/k with C = 2^120

    const float4* tab = reinterpret_cast<const float4*>(p.table);
    const int2* ent = p.srt_ent + m_first;
    Cursor c;
    c.q = 0;
    auto load_next = [&]() {
        c.npos = 0; c.nend = TABLE_ZERO_RUN;
        if (c.q < m_np) {
            const int2 e = __ldg(ent + c.q);
            c.q++;
            c.npos = e.x; c.nend = e.x + e.y;
        }
    };
    c.pos = TABLE_ZERO_RUN - 2 * lg; c.end = TABLE_ZERO_RUN;  // 2*lg idle steps before the stream starts
    load_next();
    // dep: the word of the entry the CURRENT step works on.  Its top bit is never set, but the address now depends on
    // it, which keeps the loads behind the wait for that entry (see the step loop).
    // Runs start at even entries and have even lengths, so a lane's position is even at the loop's even steps: only
    // those look at the cursor and form an address; the odd step's entry is the next one of the same 32-entry block,
    // 16 slots (256 bytes) further on.
    const float4* e_even = tab;
    auto load_entry = [&](RawEntry& r, const float4* e) {
#if SHORT_L2_PREFETCH
        r.a = ldg_pf(e);
        r.b = ldg_pf(e + TABLE_CHUNK_STRIDE);
        r.c = ldg_pf(e + 2 * TABLE_CHUNK_STRIDE);
        r.w = ldg_pf_u32(reinterpret_cast<const uint32_t*>(e + 3 * TABLE_CHUNK_STRIDE));
#else
        r.a = __ldg(e);
        r.b = __ldg(e + TABLE_CHUNK_STRIDE);
        r.c = __ldg(e + 2 * TABLE_CHUNK_STRIDE);
        r.w = __ldg(reinterpret_cast<const uint32_t*>(e + 3 * TABLE_CHUNK_STRIDE));
#endif
    };
    auto fetch_even = [&](RawEntry& r, uint32_t dep) {
        if (c.pos == c.end) { c.pos = c.npos; c.end = c.nend; load_next(); }
        e_even = tab + ((((int64_t)(c.pos >> 5)) << 7) + (int64_t)(((c.pos >> 1) & 15) + (dep >> 31)));  // table_slot of an even position
#if SHORT_L2_LINE_PREFETCH
        // the group's first lane asks L2 for one 128-byte table line PF entries ahead per two steps: the 8 lines (4 chunk
        // planes x 2 parities) of a 16-entry half block over 16 entries.  Past the end of a run this runs into the next
        // read's entries, which the task usually streams next (reads of a haplotype are adjacent in the pair list).
        if (is_first) {
            const int t = c.pos + SHORT_L2_LINE_PREFETCH, q = (c.pos >> 1) & 7;
            const float4* pf = tab + ((((int64_t)(t >> 5)) << 7) + (int64_t)((q >> 1) * TABLE_CHUNK_STRIDE + (q & 1) * 16 + ((t >> 4) & 1) * 8));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(pf));
        }
#endif
        c.pos += 2;
        load_entry(r, e_even);
    };
    auto fetch_odd = [&](RawEntry& r, uint32_t dep) { load_entry(r, e_even + (16 + (dep >> 31))); };

    int nout = 0;
    const double LOG10_2 = 0.30102999566398119521;
    auto one_step = [&](const RawEntry& r) {
        Entry2<float> E;
        E.gam = make_float2(r.a.x, r.a.y); E.A = make_float2(r.a.z, r.a.w);
        E.C = make_float2(r.b.x, r.b.y); E.G = make_float2(r.b.z, r.b.w);
        E.pmx = r.c.x; E.pxx = r.c.y; E.pmy = r.c.z; E.pxy = r.c.w;
        E.metaX = r.w & 0xffu; E.metaY = (r.w >> 16) & 0xffu;
        E.r2 = r.w & 0xff00ff00u;
        // what the left neighbour's .y half handed out in its last step; a haplotype that fills its last lane completely
        // has its last column's M+I there when the sum entry arrives, not in a T of its own
        const float prevT = ln.outT.y;
        float inS = __shfl_up_sync(PHMM_FULL, ln.outS.y, 1);
        float inT = __shfl_up_sync(PHMM_FULL, prevT, 1);
        if (is_first) {  // column-0 boundary, Eq.1
            const bool f = (E.metaX & META_FIRST) != 0;
            inS = f ? Cok : 0.f;
            inT = E.C.x * inS;
        }
        ln.step(E, inS, inT);
        if (r.w & sum_bit) {  // the group's last lane, its .y half on the sum entry: s has collected M_l + I_l of every column (Eq.4)
            const float sg = full_last ? ln.outS.y + prevT : ln.outS.y;
            const int pair = p.srt_out[m_first + nout];
            nout++;
            if (isfinite(sg) && sg >= p.rescue_thr) {
                p.out[pair] = log10((double)sg) - 120.0 * LOG10_2;
                if (p.flags) p.flags[pair] = 0;
            } else if (m_k <= RESCUE_MAX_K) {  // (every short-class read has l <= RESCUE_MAX_L)
                const int rr = p.pair_read[pair];
                rescue_push(p.rescue, pair, m_k, (int)(b.read_off[rr + 1] - b.read_off[rr]));  // a10: unrescaled fp64 sub-warp kernel
            } else {
                const int idx = atomicAdd(p.rescue_count, 1);  // rescaled fp64 chain kernel
                p.rescue_list[idx] = pair;
            }
        }
    };
    // ptxas tracks every table load with ONE scoreboard, so the first use of a loaded entry waits for all loads in
    // flight, the newest included (seen in the SASS control codes; with three register sets and two steps of fetch-ahead
    // one step in three stalled for a full memory latency: 10 % of the stall samples).  Each step therefore makes the
    // address of the next entry depend on its own entry's word (loaded one step ago), so the loads are issued BEHIND the
    // wait and the wait never covers loads younger than a whole step: 3.31 -> 3.36 TCUPS, 4 fewer registers.
    RawEntry eA, eB;
    fetch_even(eA, 0u);
    for (int s = 0; s < steps; s += 2) {  // an odd step count runs one extra all-idle step, which is harmless
        fetch_odd(eB, eA.w);
        one_step(eA);
        fetch_even(eA, eB.w);
        one_step(eB);
    }
}

cudaError_t launch_short_f32(const DevBatch& b, const ShortLaunch& p, cudaStream_t st) {
    if (p.n_warps == 0) return cudaSuccess;
    const int grid = (p.n_warps + SHORT_WARPS_PER_CTA - 1) / SHORT_WARPS_PER_CTA;
    if (b.n_wild) k_short_f32<SHORT_NV, false><<<grid, SHORT_WARPS_PER_CTA * 32, 0, st>>>(b, p);
    else k_short_f32<SHORT_NV, true><<<grid, SHORT_WARPS_PER_CTA * 32, 0, st>>>(b, p);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ debug pass: preconditions of the payload
__global__ void k_validate(DevBatch b, const double* __restrict__ lut, int64_t read_lo, int64_t read_hi, int64_t hap_lo, int64_t hap_hi,
                           int qual_offset, int* err) {
    int bad = 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    auto base_ok = [](uint8_t c) { return c == 'A' || c == 'C' || c == 'G' || c == 'T' || c == 'N'; };
    for (int64_t i = read_lo + i0; i < read_hi; i += stride) {
        if (!base_ok(b.read_bases[i])) bad |= 1;
        const int qb = b.qual_base[i], qi = b.qual_ins[i], qd = b.qual_del[i], qg = b.qual_gcp[i];
        if (qb < qual_offset || qi < qual_offset || qd < qual_offset || qg < qual_offset) bad |= 2;
        if (!(lut[qi] + lut[qd] < 1.0)) bad |= 4;  // T_MM = 1 - iota - delta must stay positive (reading G18)
    }
    for (int64_t i = hap_lo + i0; i < hap_hi; i += stride)
        if (!base_ok(b.hap_bases[i])) bad |= 1;
    if (bad) atomicOr(err, bad);
}

cudaError_t launch_validate(const DevBatch& b, const double* lut, int64_t read_lo, int64_t read_hi, int64_t hap_lo, int64_t hap_hi,
                            int qual_offset, int* d_err, cudaStream_t st) {
    k_validate<<<592, 256, 0, st>>>(b, lut, read_lo, read_hi, hap_lo, hap_hi, qual_offset, d_err);
    return cudaGetLastError();
}

}  // namespace phmm
