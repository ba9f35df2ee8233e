// Long-pair fp32 path: one warp = one strip of 32 lanes x 32 haplotype columns of one pair, the strips of a pair chained
// left to right through boundary records in global memory (the multi-block row-parallel wavefront of BASELINE.json
// north_star; the paper's lock-step carries Eq.10/11, become a skewed wavefront with a
// two-value handoff per read row).  SURVEY.md section 8(a) rows a4-a9 for haplotypes over 1024 bases or reads over 4096.
//
// The recurrence step, the table of per-row constants and the way entries are fetched are exactly the short kernel's
// (phmm_engine.cuh, phmm_table.cuh, phmm_short.cu): a strip is a lane group of 32 lanes streaming ONE read.  What this
// kernel adds:
//
// Rescaling (a8, reading G15; the paper has none).  Block floating point per LANE: true value = stored value * 2^ex, one
// integer ex for everything a thread holds.  Exponents change only at "events", every 16 steps, for all lanes of the warp
// at once; between two events a lane converts the two values it receives per step from its left neighbour with ONE cached
// power-of-two factor f_in = 2^(ex_left - ex) (two multiplies per step; no branch, no exponent arithmetic in the step).
// At an event every lane
//   1. takes the maximum m of what it holds and proposes ex' = ex + ilogb(m) - TGT (its maximum back to 2^TGT);
//   2. is held to ex'_L >= max over the lanes m < L of ex'_m - KTOT (a prefix maximum: 5 shuffles), and lane 0 to the
//      exponents of the 16 boundary records it is about to consume.  Values move only right and down and only shrink in
//      true magnitude, so whatever reaches a lane in the next 16 steps is stored at or below 2^(TGT+KTOT) there, over
//      any number of hops: no overflow, no per-step check;
//   3. multiplies its state by 2^(ex - ex') (exact; what falls below the format's range was more than 2^-(126+TGT) below
//      the lane's own maximum or 2^-(126+TGT+KTOT) below the maximum of a lane to its left: G15's documented limit) and
//      recomputes f_in.
// A result that is not a normal positive number (or a NaN anywhere in a lane's share of Eq.4) sends the pair to the
// fp64 chain kernel (phmm_chain.cu): the same cascade as fp32 -> fp64 for short pairs.
//
// Eq.4.  The short kernel lets the running sum s collect M_l + I_l across the whole lane group on the "sum entry".  Here
// the lanes of a group do not share an exponent and s does not decay on that entry, so each lane takes only its OWN sum
// (the incoming s is cut to 0 on the sum entry) at its own exponent; the 32 (sum, exponent) pairs are combined once per
// strip, and the strips of a pair pass the running total along their chain (one (sum, exponent) slot per strip).
//
// Handoff between strips (a6/a7).  Lane 31 stores one 16-byte record {s, T, ex, -} per stream entry and publishes a
// progress counter every `publish` entries (st.release.gpu: MEMBAR + strong store, no L1 invalidation).  The consumer's
// lanes 0-15 poll that counter with relaxed loads only when the producer was not known to be finished, and read the
// records with strong (L2) loads: nothing here invalidates L1, which holds the table windows of every warp of the SM
// (an acquire load or __threadfence would: CCTL.IVALL).  Items are taken by ticket in strip-major order, so a strip's
// producer always holds an earlier ticket: forward progress without co-residency assumptions.
#include "phmm_engine.cuh"
#include "phmm_kernels.h"
#include "phmm_table.cuh"

namespace phmm {

#ifndef LONG_MIN_CTAS
#define LONG_MIN_CTAS 3
#endif
constexpr int LONG_WPC = 4;       // warps per CTA
constexpr int LONG_TGT = 0;       // a lane's maximum is brought back to 2^TGT at every event (0: the shift 2^(TGT - ilogb) is always one factor)
constexpr int LONG_KTOT = 90;     // a lane's exponent is at most this much below that of any lane to its left
constexpr int LONG_EVERY = 16;    // steps between two events
constexpr int LONG_FLOOR = -(1 << 28);  // "no proposal" (a lane that holds nothing but zeros)

__device__ __forceinline__ int ld_relaxed_gpu(const int* p) {
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ float4 ld_strong_f4(const float4* p) {  // served by L2: never a stale L1 line
    float4 v;
    asm volatile("ld.relaxed.gpu.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_strong_f4(float4* p, float4 v) {
    asm volatile("st.relaxed.gpu.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
// 2^e for any e: 0 below the normal range, 2^127 above
__device__ __forceinline__ float pow2f(int e) { return Fx<float>::exp2i(e); }
// v * 2^d for |d| up to 252, exact unless the result leaves the format
__device__ __forceinline__ float scale2(float v, int d) {
    d = max(-252, min(252, d));
    const int h = d / 2;
    return v * pow2f(h) * pow2f(d - h);
}

#ifdef LONG_DEBUG
__device__ float g_dbg[1 << 16];
extern "C" int phmm_debug_read(float* dst, int n) { return (int)cudaMemcpyFromSymbol(dst, g_dbg, (size_t)n * 4); }
#endif

struct LongSmem {
    float4 ring[4 * 128];    // 4 table blocks of 32 entries (2 KB each, in the table's own layout)
    float2 rin[LONG_EVERY];  // the boundary values lane 0 consumes in the next 16 steps, already at its exponent
};

template <int NV>
__global__ void __launch_bounds__(LONG_WPC * 32, LONG_MIN_CTAS) k_long_f32(DevBatch b, LongLaunch p) {
    typedef Lane2<float, NV, true> L;
    constexpr int N2 = 2 * NV;
    constexpr int STRIP = 32 * N2;
    __shared__ __align__(16) LongSmem sm_all[LONG_WPC];
    __shared__ __align__(16) float4 sm_zero[128];  // an all-zero table block
    LongSmem& sm = sm_all[threadIdx.x >> 5];
    for (int i = threadIdx.x; i < 128; i += blockDim.x) sm_zero[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const double LOG10_2 = 0.30102999566398119521;
    const int n_items = *p.n_items;
    const float4* tab = reinterpret_cast<const float4*>(p.table);

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
        const int n_ent = l + TABLE_EXTRA_ROWS;        // run-in entry, rows 1..l, sum entry, flush entry
        const int run0 = (int)table_run_start(ro, r), run_len = table_run_len(l);
        const int nstrips = (k + STRIP - 1) / STRIP;
        const bool has_in = strip > 0, has_out = strip + 1 < nstrips;
        const int k_loc = min(k - strip * STRIP, STRIP);          // real columns of this strip
        const int out_lane = (k_loc - 1) / N2;                      // the lane that holds the strip's last real column
        const float4* inrec = p.records + it.buf0 + (int64_t)(strip - 1) * n_ent;
        float4* outrec = p.records + it.buf0 + (int64_t)strip * n_ent;
        const int* inprog = p.progress + it.prog0 + strip - 1;
        int* outprog = p.progress + it.prog0 + strip;
        const bool store_out = has_out && lane == 31;
        const float Cok = (float)(1.0 / (double)k);                // Eq.1 with C = 1 (the exponents do the scaling)

        L ln;
        ln.init();
        ln.load_hap(b.hap_bases + ho, k, (strip * 32 + lane) * N2);
        int ex = 0;            // true value = stored value * 2^ex
        float f_in = 1.f;      // 2^(ex of the left neighbour - ex)
        int seen = 0;          // entries the producer strip is known to have published
        float fin_m = 0.f;     // this lane's share of Eq.4 and its exponent
        int fin_e = LONG_FLOOR;

        // ---- fetch.  The table blocks (32 entries = 2 KB, phmm_table.cuh) the warp is walking live in a ring of 4 blocks in
        // shared memory, filled by cp.async one block (32 steps) ahead of lane 0: the step never waits for L2 or DRAM.
        // Lane L's .x half is at table position run0 + s - 2L at step s; before its stream starts and after it has ended a
        // lane reads the all-zero block instead.  Block B sits in ring slot B & 3: when lane 0 enters block B, lane 31 (62
        // entries behind) is in block B-2, so slot (B+1) & 3 = (B-3) & 3 is free for block B+1.
        const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(sm.ring);
        const uint32_t zero_s = (uint32_t)__cvta_generic_to_shared(sm_zero);
        auto fill = [&](int blk) {
            const char* g = reinterpret_cast<const char*>(tab) + ((int64_t)blk << 11) + lane * 16;
            const uint32_t d = ring_s + ((blk & 3) << 11) + lane * 16;
#pragma unroll
            for (int j = 0; j < 4; j++)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + j * 512), "l"(g + j * 512) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        auto fill_wait = [&]() {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
        };
        uint32_t e_even = zero_s;  // shared-memory address of chunk 0 of the even entry
        auto load_entry = [&](RawEntry& re, uint32_t e) {
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(re.a.x), "=f"(re.a.y), "=f"(re.a.z), "=f"(re.a.w) : "r"(e));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+512];" : "=f"(re.b.x), "=f"(re.b.y), "=f"(re.b.z), "=f"(re.b.w) : "r"(e));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+1024];" : "=f"(re.c.x), "=f"(re.c.y), "=f"(re.c.z), "=f"(re.c.w) : "r"(e));
            asm volatile("ld.shared.b32 %0, [%1+1536];" : "=r"(re.w) : "r"(e));
        };
        auto fetch_even = [&](RawEntry& re, int s) {  // the entry of (even) step s
            const int v = s - 2 * lane;
            const int pos = run0 + v;
            e_even = (unsigned)v < (unsigned)run_len ? ring_s + (((pos >> 5) & 3) << 11) + (((pos >> 1) & 15) << 4) : zero_s;
            load_entry(re, e_even);
        };
        auto fetch_odd = [&](RawEntry& re) { load_entry(re, e_even + 256); };  // (runs have even lengths: same block, same range)
        fill(run0 >> 5);
        fill((run0 >> 5) + 1);
        fill_wait();

        // ---- an event: new exponents for all lanes, the next 16 boundary records for lane 0
        auto event = [&](int s) {
            // what lane 31 has stored so far becomes visible to the next strip (release: MEMBAR + strong store)
            if (store_out && s > 63 && (s & (p.publish - 1)) == 0) st_release_gpu(outprog, min(s - 63, n_ent));
            float4 rec = make_float4(0.f, 0.f, 0.f, 0.f);
            int bmax = LONG_FLOOR;
            if (has_in && s < n_ent) {  // (warp-uniform)
                const int need = min(s + LONG_EVERY, n_ent);
                if (need > seen) {  // (the producer is usually far ahead: one look every few hundred steps)
                    int v = ld_relaxed_gpu(inprog);
                    while (v < need) { __nanosleep(100); v = ld_relaxed_gpu(inprog); }
                    seen = v;
                }
                if (lane < LONG_EVERY && s + lane < n_ent) rec = ld_strong_f4(inrec + s + lane);
                const float mi = fmaxf(rec.x, rec.y);
                bmax = mi > 0.f ? __float_as_int(rec.z) + Fx<float>::ilogb(mi) : LONG_FLOOR;
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) bmax = max(bmax, __shfl_xor_sync(PHMM_FULL, bmax, o));
                bmax = __shfl_sync(PHMM_FULL, bmax, 0);
            }
            // 1. own proposal (none for a lane that holds nothing)
            float m = fmax3(ln.outS.x, ln.outS.y, fmaxf(ln.outT.x, ln.outT.y));
#pragma unroll
            for (int x = 0; x < NV; x++) m = fmax3(m, fmaxf(ln.Tt[x].x, ln.Tt[x].y), fmaxf(ln.J[x].x, ln.J[x].y));
            int c = m > 0.f ? ex + Fx<float>::ilogb(m) - LONG_TGT : LONG_FLOOR;
            // 2. ex'_L = max(c_L, max over m < L of c_m - KTOT), the boundary records counting as a lane to the left of lane
            //    0: nothing that can reach lane L (values only move right and down, and only shrink in true magnitude) is
            //    stored above 2^(TGT+KTOT) there -- whatever the hop count
            const int bsrc = bmax > LONG_FLOOR ? bmax - LONG_TGT : LONG_FLOOR;
            int pm = lane == 0 ? max(c, bsrc) : c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(PHMM_FULL, pm, o);
                if (lane >= o) pm = max(pm, t);
            }
            pm = __shfl_up_sync(PHMM_FULL, pm, 1);
            if (lane == 0) pm = bsrc;
            if (pm > LONG_FLOOR) c = max(c, pm - LONG_KTOT);
            const int exn = c < LONG_FLOOR / 2 ? ex : c;  // nothing held, nothing to the left: keep the exponent
            // 3. rescale the state: d <= TGT - ilogb(m) <= 127 when something is held, any d when nothing is
            const int d = m > 0.f ? ex - exn : 0;
            const int ex_new = exn;
            const float f = pow2f(d);  // 0 for d < -126: everything held is negligible against what is about to arrive
            const float2 F = make_float2(f, f);
#pragma unroll
            for (int x = 0; x < NV; x++) { ln.Tt[x] = __fmul2_rn(ln.Tt[x], F); ln.J[x] = __fmul2_rn(ln.J[x], F); }
            ln.outS = __fmul2_rn(ln.outS, F);
            ln.outT = __fmul2_rn(ln.outT, F);
            ex = ex_new;
#ifdef LONG_DEBUG
            if (pair == 0 && s / 16 < 60) {
                float* q = g_dbg + ((strip * 60 + s / 16) * 32 + lane) * 4;
                q[0] = m; q[1] = (float)ex; q[2] = f; q[3] = (float)c;
            }
#endif
            const int exl = __shfl_up_sync(PHMM_FULL, ex, 1);
            f_in = pow2f(exl - ex);  // (exl - ex <= KTOT by construction; lane 0 does not use it)
            // 4. lane 0's next 16 boundary values at its new exponent
            if (has_in) {
                const int ex0 = __shfl_sync(PHMM_FULL, ex, 0);
                __syncwarp();
                if (lane < LONG_EVERY) {
                    const int dd = __float_as_int(rec.z) - ex0;
                    sm.rin[lane] = make_float2(scale2(rec.x, dd), scale2(rec.y, dd));
                }
                __syncwarp();
            }
        };

        const uint32_t sum_y = META_SUM << 16;
        auto one_step = [&](const RawEntry& re, int s) {
            Entry2<float> E;
            E.gam = make_float2(re.a.x, re.a.y); E.A = make_float2(re.a.z, re.a.w);
            E.C = make_float2(re.b.x, re.b.y); E.G = make_float2(re.b.z, re.b.w);
            E.pmx = re.c.x; E.pxx = re.c.y; E.pmy = re.c.z; E.pxy = re.c.w;
            E.metaX = re.w & 0xffu; E.metaY = (re.w >> 16) & 0xffu;
            E.r2 = re.w & 0xff00ff00u;
            const float prevT = ln.outT.y;
            float inS = __shfl_up_sync(PHMM_FULL, ln.outS.y, 1) * f_in;
            float inT = __shfl_up_sync(PHMM_FULL, prevT, 1) * f_in;
            if (lane == 0) {
                if (has_in) {
                    const float2 v = sm.rin[s & (LONG_EVERY - 1)];
                    inS = v.x; inT = v.y;
                } else {  // column-0 boundary, Eq.1 (reading G1): only the run-in entry injects, at exponent 0
                    inS = (E.metaX & META_FIRST) ? Cok : 0.f;
                    inT = E.C.x * inS;
                }
            }
            if (E.metaX & META_SUM) inS = 0.f;  // Eq.4: every lane sums its own columns only
            ln.step(E, inS, inT);
            if (re.w & sum_y) {  // this lane's .y half has just finished the sum entry: its share of Eq.4
                if (lane <= out_lane) {
                    // M+I of column j reaches the sum through the T of column j+1; a strip whose last real column is the last
                    // column of its lane has that one in what the lane handed out one step ago
                    const bool full = !has_out && lane == out_lane && (k_loc % N2) == 0;  // (else the next strip counts it)
                    fin_m = full ? ln.outS.y + prevT : ln.outS.y;
                    fin_e = ex;
                }
            }
            // ---- right boundary: lane 31's .y half has just finished entry s - 63
            // (published at the next event, or with the Eq.4 total behind the loop)
            if (store_out && (unsigned)(s - 63) < (unsigned)n_ent)
                st_strong_f4(outrec + (s - 63), make_float4(ln.outS.y, ln.outT.y, __int_as_float(ex), 0.f));
        };

        RawEntry eA, eB;
        fetch_even(eA, 0);
        const int steps = run_len + 64;  // even; lane 31's .y half finishes entry run_len - 1 >= n_ent - 1 at step run_len + 62
        for (int s = 0; s < steps; s += 2) {
            if ((s & (LONG_EVERY - 1)) == 0) event(s);
            if (((run0 + s + 2) & 31) == 0) {  // lane 0's next fetch enters a new block (now complete): the one after it starts its way in
                fill_wait();
                fill(((run0 + s + 2) >> 5) + 1);
            }
            fetch_odd(eB);
            one_step(eA, s);
            fetch_even(eA, s + 2);
            one_step(eB, s + 1);
        }

        // ---- Eq.4: combine the lanes' shares, then the strips' (each strip waits for the total of the strips to its left)
        int em = fin_m > 0.f ? fin_e + Fx<float>::ilogb(fin_m) : LONG_FLOOR;  // exponent of the largest share
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) em = max(em, __shfl_xor_sync(PHMM_FULL, em, o));
        // in units of 2^em; a share that is neither zero nor a positive number (NaN: an overflow upstream) poisons the total
        double tot = fin_m > 0.f ? ldexp((double)fin_m, max(fin_e - em, -1000)) : (fin_m == 0.f ? 0.0 : (double)fin_m);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(PHMM_FULL, tot, o);
        if (lane == 31) {  // (the lane that published the records, so the progress counter has one writer)
            double acc = tot;
            int acc_e = em;
            if (has_in) {  // total of the strips to the left: (double mantissa, exponent), published behind the last record
                int v = seen;
                while (v < n_ent + 1) { v = ld_relaxed_gpu(inprog); if (v < n_ent + 1) __nanosleep(100); }
                const float4 t = ld_strong_f4(p.totals + it.prog0 + strip - 1);
                const double lm = __hiloint2double(__float_as_int(t.y), __float_as_int(t.x));
                const int le = __float_as_int(t.z);
                if (!(lm >= 0.0) || !(acc >= 0.0)) acc = lm + acc;  // NaN stays NaN
                else if (lm > 0.0) {
                    if (!(acc > 0.0)) { acc = lm; acc_e = le; }
                    else if (le >= acc_e) { acc = lm + ldexp(acc, max(acc_e - le, -2000)); acc_e = le; }
                    else acc += ldexp(lm, max(le - acc_e, -2000));
                }
            }
            if (has_out) {
                st_strong_f4(p.totals + it.prog0 + strip,
                             make_float4(__int_as_float(__double2loint(acc)), __int_as_float(__double2hiint(acc)), __int_as_float(acc_e), 0.f));
                st_release_gpu(outprog, n_ent + 1);
            } else if (acc > 0.0 && acc < 1e300) {  // (finite and positive; acc is a sum of normal floats)
                p.out[pair] = log10(acc) + (double)acc_e * LOG10_2;
                if (p.flags) p.flags[pair] = p.flag_bits;
            } else {  // overflow or a vanished sum: the fp64 chain kernel recomputes the pair
#ifdef LONG_DEBUG
                p.out[pair] = acc != acc ? -1e9 : (acc >= 1e300 ? -2e9 : (acc == 0.0 ? -3e9 : -4e9));
                if (p.flags) p.flags[pair] = 64;
#else
                const int idx = atomicAdd(p.fallback_count, 1);
                p.fallback_list[idx] = pair;
#endif
            }
        }
        __syncwarp();
    }
}

cudaError_t launch_long_f32(const DevBatch& b, const LongLaunch& p, int grid_ctas, cudaStream_t st) {
    if (grid_ctas <= 0) return cudaSuccess;
    k_long_f32<SHORT_NV><<<grid_ctas, LONG_WPC * 32, 0, st>>>(b, p);
    return cudaGetLastError();
}

int long_ctas_per_sm() {
    int n = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_long_f32<SHORT_NV>, LONG_WPC * 32, 0);
    return n > 0 ? n : 1;
}
int long_warps_per_cta() { return LONG_WPC; }

}  // namespace phmm
