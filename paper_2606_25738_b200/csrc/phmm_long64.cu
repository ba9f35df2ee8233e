// PHMM_FP64 long path: table-driven strips in double with per-thread block exponents.
//
// SURVEY.md section 8(a) rows a4, a5, a7 (cross-CTA carry: the paper's lock-step Eq.11, as a skewed
// wavefront), a8 (rescaling, absent from the paper: reading G15), a9.
//
// One warp = one strip of 32 lanes x 32 haplotype columns of one long pair; the strips of all pairs are taken by ticket in
// strip-major order (a strip's producer holds an earlier ticket: forward progress without co-residency assumptions) and
// chained left to right through 32-entry boundary blocks in global memory, published with st.release and awaited with
// relaxed polls and strong (L2) loads of the block, as in phmm_long.cu -- the hand-off of the chain kernel (phmm_chain.cu),
// which this kernel replaces for the concurrent strips; the chain kernel stays the sequential fallback.  The engine is the one of the fp64 sub-warp kernel (phmm_rescue.cu): the T/J
// form of phmm_engine.cuh in double, one lane = 32 columns, lane L one stream entry behind lane L-1, row constants from the
// double table of k_table_f64 one step ahead, the strip's first lane prefetching the table into L2.  Against the chain
// kernel (two 8-column halves per thread, constants formed in the loop, 19 instructions per cell) that is 9 instructions
// per cell with the fp64 pipe as the binding unit.
//
// Rescaling is the chain kernel's, unchanged in its arithmetic: true value = stored value * 2^ex with one integer ex per
// THREAD (its 32 columns of T and J and what it hands to the right).  Every 16 steps a thread takes the maximum of what it
// holds and, if that left the window 2^(0 +- 400), multiplies everything by the power of two that brings it back to 2^0
// (exact, except that values more than the format's range below the thread maximum flush to zero: G15's documented limit).
// The two values crossing a lane or strip boundary per step come with the producer's ex and are converted by one exact
// multiply; if they would not fit (above 2^600 at this thread's exponent), the consumer first moves its own exponent up.
#include "phmm_common.cuh"
#include "phmm_kernels.h"

namespace phmm {

#ifndef LONG64_MIN_CTAS
#define LONG64_MIN_CTAS 8  // one-warp CTAs, 255 registers: 8 warps per SM
#endif

namespace {

constexpr int L64_NV = 32;
constexpr int L64_TGT = 0, L64_WIN = 400, L64_UP = 600;

struct Rec64 {  // boundary block of 32 stream entries, SoA
    double S[32], Tn[32];
    int ex[32];
};

__device__ __forceinline__ int ld_relaxed64(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release64(int* p, int v) {  // MEMBAR + strong store, no L1 invalidation
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ double ld_strong_f64(const double* p) {  // served by L2: never a stale L1 line
    double v;
    asm volatile("ld.relaxed.gpu.global.f64 %0, [%1];" : "=d"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ int ld_strong_s32(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

struct Raw64 { double gam, A, C, G, pm, px; uint32_t w; };

}  // namespace

__global__ void __launch_bounds__(32, LONG64_MIN_CTAS) k_long_f64(DevBatch b, ChainLaunch p, const double* __restrict__ table) {
    constexpr int NV = L64_NV;
    __shared__ Rec64 RI, RO;
    const int lane = threadIdx.x;
    const double LOG10_2 = 0.30102999566398119521;
    const int n_items = *p.n_items;

    for (;;) {
        int ticket = 0;
        if (lane == 0) ticket = atomicAdd(p.ticket, 1);
        ticket = __shfl_sync(PHMM_FULL, ticket, 0);
        if (ticket >= n_items) break;
        const ChainItem it = p.items[ticket];
        const int pair = it.pair, strip = it.strip;
        const int r = p.pair_read[pair], h = p.pair_hap[pair];
        const int64_t ro = b.read_off[r], ho = b.hap_off[h];
        const int l = (int)(b.read_off[r + 1] - ro), k = (int)(b.hap_off[h + 1] - ho);
        const int n_ent = l + 2;  // run-in entry, rows 1..l, sum entry
        const int nstrips = (k + 32 * NV - 1) / (32 * NV);
        const int k_last = k - (nstrips - 1) * 32 * NV;  // real columns of the last strip
        const int out_lane = (k_last - 1) / NV;          // Eq.4 is taken at the lane that holds the haplotype's last column
        const bool full_last = (k_last % NV) == 0;
        const int nblk = (l + CHAIN_EXTRA_ROWS + 31) / 32;  // boundary blocks per buffer (the host's count)
        const int run0 = (int)(table_run_start(ro, r) - b.table_base);
        const double Cok = ldexp(1.0, p.log2C) / (double)k;
        Rec64* bufbase = reinterpret_cast<Rec64*>(p.boundary);
        const Rec64* inb = bufbase + it.buf0 + (int64_t)(strip - 1) * nblk;
        Rec64* outb = bufbase + it.buf0 + (int64_t)strip * nblk;
        const int* inprog = p.progress + it.prog0 + strip - 1;
        int* outprog = p.progress + it.prog0 + strip;
        const bool has_in = strip > 0, has_out = strip + 1 < nstrips;
        // the step at which this lane processes the sum entry (entry l + 1): e = s - lane
        const int out_step = (!has_out && lane == out_lane) ? l + 1 + lane : -1;

        // ---- haplotype columns of this lane: one match word per base code, [4] = N; [5] = what "matches" the sum entry
        // (prior pm = 0): the columns more than one behind the haplotype's last (phmm_engine.cuh)
        const int j0 = (strip * 32 + lane) * NV;
        const int nv = min(max(k - j0, 0), NV);
        uint32_t hm[6] = {0u, 0u, 0u, 0u, 0u, 0u};
        for (int x = 0; x < nv; x++) {
            const int c = base_code(b.hap_bases[ho + j0 + x]);
#pragma unroll
            for (int q = 0; q < 5; q++) hm[q] |= ((c == q || (b.n_wild && c == 4)) ? 1u : 0u) << x;
        }
#pragma unroll
        for (int x = 0; x < NV; x++) hm[5] |= (j0 + x > k ? 1u : 0u) << x;

        double T[NV], J[NV];
#pragma unroll
        for (int x = 0; x < NV; x++) { T[x] = 0.0; J[x] = 0.0; }
        double outS = 0.0, outT = 0.0;
        int ex = 0;        // true value = stored value * 2^ex, one exponent per thread
        bool zero = true;  // this thread holds nothing but zeros

        auto scale_all = [&](int d) {  // *= 2^d
            d = max(-Fx<double>::CLAMP, min(Fx<double>::CLAMP, d));
            const int hh = d / 2;
            const double f1 = Fx<double>::exp2i(hh), f2 = Fx<double>::exp2i(d - hh);
#pragma unroll
            for (int x = 0; x < NV; x++) { T[x] = T[x] * f1 * f2; J[x] = J[x] * f1 * f2; }
            outS = outS * f1 * f2;
            outT = outT * f1 * f2;
        };
        // entry e of the read's run (e < 0 or e >= n_ent: an all-zero entry of the table's zero run)
        auto fetch = [&](Raw64& re, int e) {
            const int pos = ((unsigned)e < (unsigned)n_ent) ? run0 + e : 0;
            const double* q = table + (((int64_t)(pos >> 5)) << 8) + (pos & 31);
            re.gam = __ldg(q); re.A = __ldg(q + 32); re.C = __ldg(q + 64); re.G = __ldg(q + 96);
            re.pm = __ldg(q + 128); re.px = __ldg(q + 160);
            re.w = __ldg(reinterpret_cast<const uint32_t*>(q - (pos & 31) + 192) + (pos & 31));
        };
        Raw64 ea, eb;
        fetch(ea, -lane);
        __syncwarp();
        int seen = 0;  // entries the producer is known to have published
        // One step; `even`: s is even (an event every 16 steps and a new incoming block every 32 can only fall on those).
        // The loop below runs the steps in pairs with the two entry buffers swapped, so that no register is ever copied.
        auto body = [&](const bool even, const int s, const Raw64& cur, Raw64& nxt) {
            if (even && (s & 15) == 0) {
                // ---- incoming boundary block for entries s..s+31 (lane 0 consumes entry s at step s)
                if ((s & 31) == 0 && has_in && s < n_ent) {
                    __syncwarp();
                    const int need = min(s + 32, n_ent);
                    while (seen < need) {  // relaxed polls, and only while the producer is not known to be far enough
                        seen = ld_relaxed64(inprog);
                        if (seen < need) __nanosleep(64);
                    }
                    const Rec64* src = inb + (s >> 5);
                    RI.S[lane] = ld_strong_f64(src->S + lane); RI.Tn[lane] = ld_strong_f64(src->Tn + lane);
                    RI.ex[lane] = ld_strong_s32(src->ex + lane);
                }
                // ---- a8: block-floating event of this thread.  Everything held is >= 0, so the largest high word is the
                // high word of the maximum.
                int hi = max(__double2hiint(outS), __double2hiint(outT));
#pragma unroll
                for (int x = 0; x < NV; x++) hi = max(hi, max(__double2hiint(T[x]), __double2hiint(J[x])));
                const int eb_ = (hi >> 20) & 0x7ff;
                if (eb_ > 0) {
                    const int e = eb_ - 1023;
                    if (e > L64_TGT + L64_WIN || e < L64_TGT - L64_WIN) {
                        scale_all(L64_TGT - e);
                        ex += e - L64_TGT;
                    }
                    zero = false;
                } else {
                    zero = true;  // nothing held (or only subnormals): the exponent is free, adopt the next incoming one
                }
                __syncwarp();
            }
            fetch(nxt, s + 1 - lane);
            if (lane == 0) {  // the strip's leading lane asks L2 for the block 24 entries ahead, one of its 16 lines per step
                const int pos = run0 + s + 24;
                const char* q = reinterpret_cast<const char*>(table) + (((int64_t)(pos >> 5)) << 11) + ((s & 15) << 7);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(q));
            }
            const double gam = cur.gam, A = cur.A, C = cur.C, G = cur.G, pm = cur.pm, px = cur.px;
            const uint32_t meta = cur.w & 0xffu;
            const uint32_t code = meta & META_CODE_MASK;
            const uint32_t m01 = (code & 1u) ? hm[1] : hm[0], m23 = (code & 1u) ? hm[3] : hm[2];
            uint32_t mw = (code & 4u) ? hm[4] : ((code & 2u) ? m23 : m01);
            mw = (meta & META_SUM) ? hm[5] : mw;
            // ---- left boundary: neighbour lane (shuffle), first strip (Eq.1 injection, reading G1) or boundary block
            const double prevT = outT;
            double inS = __shfl_up_sync(PHMM_FULL, outS, 1), inT = __shfl_up_sync(PHMM_FULL, prevT, 1);
            int exL = __shfl_up_sync(PHMM_FULL, ex, 1);
            {  // (selects instead of branches: the scheduler can then move engine work of this step above the exchange)
                const int q = s & 31;
                const bool ok = s < n_ent;
                const double fS = (meta & META_FIRST) ? Cok : 0.0;  // only the run-in entry injects, at exponent 0
                const double bS = has_in ? (ok ? RI.S[q] : 0.0) : fS;
                const double bT = has_in ? (ok ? RI.Tn[q] : 0.0) : C * fS;
                const int bE = has_in ? (ok ? RI.ex[q] : ex) : 0;
                inS = lane == 0 ? bS : inS; inT = lane == 0 ? bT : inT; exL = lane == 0 ? bE : exL;
            }
            // ---- bring the incoming values to this thread's exponent (exact power-of-two multiplies)
            {
                const double mi = fmax(inS, inT);
                const bool pos = mi > 0.0;
                ex = (zero && pos) ? exL : ex;  // nothing held: adopt the incoming exponent
                zero = zero && !pos;
                if (!zero && pos && Fx<double>::ilogb(mi) + exL - ex > L64_TGT + L64_UP) {
                    const int up = Fx<double>::ilogb(mi) + exL - ex - L64_TGT;  // they would not fit: move this thread up first
                    scale_all(-up);
                    ex += up;
                }
                // two factors, so that any shift is exact as long as the result is representable (|d| may exceed 1022)
                const int d = max(-Fx<double>::CLAMP, min(Fx<double>::CLAMP, exL - ex));
                const int hh = d / 2;
                const double f1 = Fx<double>::exp2i(hh), f2 = Fx<double>::exp2i(d - hh);
                inS = inS * f1 * f2; inT = inT * f1 * f2;
            }
            const double prevT2 = outT;  // at this thread's current exponent (every rescaling of this step is done)
            // ---- one systolic step (phmm_engine.cuh, in double: 4 FMA + 1 MUL per cell)
            double sr = inS;
            double U = ((mw & 1u) ? pm : px) * T[0];
            T[0] = inT;
#pragma unroll
            for (int x = 0; x < NV; x++) {
                double Un = U;
                if (x + 1 < NV) Un = ((mw & (1u << (x + 1))) ? pm : px) * T[x + 1];
                const double Wv = fma(A, U, J[x]);
                const double Tn = fma(C, sr, Wv);
                J[x] = fma(G, J[x], U);
                sr = fma(gam, sr, U);
                if (x + 1 < NV) T[x + 1] = Tn; else outT = Tn;
                U = Un;
            }
            outS = sr;
            // ---- right boundary of the strip: lane 31 has just finished entry s - 31
            const int eo = s - 31;
            if (lane == 31) {  // (before entry 0 and behind the last one: slots that are rewritten / no longer read)
                const int q = eo & 31;
                RO.S[q] = outS; RO.Tn[q] = outT; RO.ex[q] = ex;
            }
            if (has_out && eo >= 0 && eo < n_ent) {
                if ((eo & 31) == 31 || eo == n_ent - 1) {
                    __syncwarp();
                    Rec64* dst = outb + (eo >> 5);
                    dst->S[lane] = RO.S[lane]; dst->Tn[lane] = RO.Tn[lane];
                    dst->ex[lane] = RO.ex[lane];
                    __syncwarp();
                    if (lane == 0) st_release64(outprog, eo + 1);
                    __syncwarp();
                }
            }
            if (s == out_step) {  // this lane has just done the sum entry: s has collected Eq.4; log10 in double
                // M+I of column j reaches the chain through the T of column j+1; a haplotype that fills its last lane has
                // the last one in what this lane handed out one step ago instead
                const double sum = full_last ? outS + prevT2 : outS;
                p.out[pair] = log10(sum) + ((double)ex - (double)p.log2C) * LOG10_2;
                if (p.flags) p.flags[pair] = p.flag_bits;
            }
        };
        const int steps = (n_ent + 31 + 1) & ~1;  // (a step behind the last one meets only zero entries)
        for (int s = 0; s < steps; s += 2) {
            body(true, s, ea, eb);
            body(false, s + 1, eb, ea);
        }
        __syncwarp();
    }
}

cudaError_t launch_long_f64(const DevBatch& b, const ChainLaunch& p, const double* table, int grid_ctas, cudaStream_t st) {
    if (grid_ctas <= 0) return cudaSuccess;
    k_long_f64<<<grid_ctas, 32, 0, st>>>(b, p, table);
    return cudaGetLastError();
}

int long64_ctas_per_sm() {
    int n = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_long_f64, 32, 0);
    return n > 0 ? n : 1;
}
size_t long64_block_bytes() { return sizeof(Rec64); }
int long64_strip_cols() { return 32 * L64_NV; }

}  // namespace phmm
