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
//   2. is held to ex'_L >= max over the lanes m < L of ex'_m - KTOT - (L - 1 - m) HOP (a max-plus prefix scan: 5 shuffles),
//      HOP = what the running sum loses crossing a lane, and lane 0 to the exponents of the 16 boundary records it is about
//      to consume.  Values move only right and down and only shrink in true magnitude, so whatever reaches a lane in the
//      next 16 steps is stored at or below 2^(TGT+KTOT) there, over any number of hops: no overflow, no per-step check;
//   3. multiplies its state by 2^(ex - ex') (exact; what falls below the format's range was more than 2^-(126+TGT) below
//      the lane's own maximum or 2^-(126+TGT+KTOT+(L-1-m) HOP) below the maximum of lane m to its left: G15's limit --
//      less than what that maximum's path would pay to get there, see the event) and recomputes f_in.
// A result that is not a normal positive number (or a NaN anywhere in a lane's share of Eq.4) sends the pair to the
// fp64 chain kernel (phmm_chain.cu): the same cascade as fp32 -> fp64 for short pairs.  So does a lane whose maximum falls
// by more than 2^LONG_DROP between two events, and so does the input guard k_read_risk at the end of this file, which
// states when 166 bits of range below a lane's maximum are enough.
//
// Eq.4.  The short kernel lets the running sum s collect M_l + I_l across the whole lane group on the "sum entry".  Here
// the lanes of a group do not share an exponent and s does not decay on that entry, so each lane takes only its OWN sum
// (the incoming s is cut to 0 on the sum entry) at its own exponent; the 32 (sum, exponent) pairs are combined once per
// strip, and the strips of a pair pass the running total along their chain (one (sum, exponent) slot per strip).
//
// Handoff between strips (a6/a7).  One 16-byte record {s, T, ex, -} per stream entry from lane 31, and a
// progress counter every `publish` entries (st.release.gpu: MEMBAR + strong store, no L1 invalidation).  The records are
// staged in shared memory and flushed, 16 at a time, at the events.  The consumer's lanes 0-15 poll that counter with relaxed
// loads only when the producer was not known to be far enough, and read the records with strong (L2) loads.  Items are taken by ticket in strip-major order, so a strip's
// producer always holds an earlier ticket: forward progress without co-residency assumptions.
#include "phmm_engine.cuh"
#include "phmm_kernels.h"
#include "phmm_table.cuh"

namespace phmm {

#ifndef LONG_MIN_CTAS
#define LONG_MIN_CTAS 3
#endif
constexpr int LONG_WPC = 4;       // warps per CTA
#ifndef LONG_HOPNUM_
#define LONG_HOPNUM_ 85  // 0.332 x 256
#endif
#ifndef LONG_TGT_
#define LONG_TGT_ 40
#endif
constexpr int LONG_TGT = LONG_TGT_;      // a lane's maximum is brought back to 2^TGT at every event: 166 bits of range below it
#ifndef LONG_KTOT_
#define LONG_KTOT_ 80
#endif
constexpr int LONG_KTOT = LONG_KTOT_;     // a lane's exponent is at most this much below that of any lane to its left
#ifndef LONG_EVERY_
#define LONG_EVERY_ 16
#endif
constexpr int LONG_EVERY = LONG_EVERY_;    // steps between two events
#ifndef LONG_DROP_
#define LONG_DROP_ 126
#endif
constexpr int LONG_DROP = LONG_DROP_;    // a lane's own maximum may fall by 2^LONG_DROP between two events before the pair is sent to fp64
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


// Shared memory of one warp.  The ring holds the 4 table blocks (32 entries = 2 KB each) the warp is walking, re-laid so
// that a lane's fetch address advances by 16 bytes per two steps and wraps inside a 1 KB window: chunk plane c (the c-th
// float4 of an entry) at c * 2048, the odd entries 1024 bytes behind the even ones, entry pos at ((pos >> 1) & 63) * 16.
struct LongSmem {
    float4 ring[4 * 128];
    float4 rraw[LONG_EVERY];  // the boundary records of the NEXT event, copied in (cp.async) during the steps before it
    float2 rin[LONG_EVERY];   // boundary values lane 0 consumes in the next 16 steps, already at its exponent
    float2 rout[LONG_EVERY];  // what lane 31 handed out in the last 16 steps (flushed to the records at the next event)
    float2 fin[32];           // per lane: its share of Eq.4 and the exponent it is stored at
    uint8_t own[32];          // per lane: see the event
    int lossy;
};

template <int NV, bool HS>  // HS = false only under phmm_options.n_is_wildcard (phmm_short.cu)
__global__ void __launch_bounds__(LONG_WPC * 32, LONG_MIN_CTAS) k_long_f32(DevBatch b, LongLaunch p) {
    typedef Lane2<float, NV, HS> L;
    constexpr int N2 = 2 * NV;
    constexpr int STRIP = 32 * N2;
    __shared__ __align__(128) LongSmem sm_all[LONG_WPC];
    __shared__ __align__(16) float4 sm_zero[512];  // all-zero entries for lanes outside their stream (same offsets as the ring)
    LongSmem& sm = sm_all[threadIdx.x >> 5];
    for (int i = threadIdx.x; i < 512; i += blockDim.x) sm_zero[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const double LOG10_2 = 0.30102999566398119521;
    const int n_items = *p.n_items;
    const char* tab = reinterpret_cast<const char*>(p.table);
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(sm.ring);
    const uint32_t zero_s = (uint32_t)__cvta_generic_to_shared(sm_zero);
    const uint32_t rin_s = (uint32_t)__cvta_generic_to_shared(sm.rin);  // rout follows at +128

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
        const int run0 = (int)(table_run_start(ro, r) - b.table_base), run_len = table_run_len(l);
        const int nstrips = (k + STRIP - 1) / STRIP;
        const bool has_in = strip > 0, has_out = strip + 1 < nstrips;
        const int risk = p.risk[r];  // k_read_risk: 255 = fp32's range per lane may not do for this read, else its smallest GCP quality
        const int hop = (risk * 32 * LONG_HOPNUM_) >> 8;  // bits the running sum loses per lane it crosses: 32 columns x 0.332 GCP_min (rounded down)
        const int hcs = ((risk * LONG_HOPNUM_) >> 8) << 23;  // the same per column (rounded down), as a step of the fp32 exponent field
        if (risk == 255) {  // the pair's last strip hands it to fp64
            if (!has_out && lane == 0) {
                const int idx = atomicAdd(p.fallback_count, 1);
                p.fallback_list[idx] = pair;
            }
            continue;
        }

        L ln;
        ln.init();
        ln.load_hap(b.hap_bases + ho, k, (strip * 32 + lane) * N2, b.n_wild != 0);
        int ex = 0;            // true value = stored value * 2^ex
        float f_in = 1.f;      // 2^(ex of the left neighbour - ex)
        int seen = 0;          // entries the producer strip is known to have published
        int pre = -1;          // first entry of the boundary records that are on their way into sm.rraw (-1: none)
        // sm.own[lane]: at the last event this lane's exponent was set by its own maximum (stored maximum = 2^TGT);
        // sm.lossy: some lane's maximum then fell by more than 2^LONG_DROP within one interval (see the event)
        sm.own[lane] = 0;
        if (lane == 0) sm.lossy = 0;
        sm.fin[lane] = make_float2(0.f, 0.f);

        // ---- fetch.  The table blocks live in the ring, filled by cp.async one block (32 steps) ahead of lane 0: the step
        // never waits for L2 or DRAM.  Lane L's .x half is at table position run0 + v, v = s - 2L, at step s; outside
        // [0, run_len) it reads all-zero entries.  Block B sits in ring slot B & 3: when lane 0 enters block B, lane 31 (62
        // entries behind) is in block B-2, so slot (B+1) & 3 = (B-3) & 3 is free for block B+1.
        auto fill = [&](int blk) {
            const char* g = tab + ((int64_t)blk << 11) + lane * 16;
            const uint32_t d = ring_s + ((lane >> 4) << 10) + ((blk & 3) << 8) + ((lane & 15) << 4);
#pragma unroll
            for (int j = 0; j < 4; j++)  // chunk plane j: 512 bytes of the table block, parity halves 256 bytes each
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d + j * 2048), "l"(g + j * 512) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        auto fill_wait = [&]() {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncwarp();
        };
        auto load_entry = [&](RawEntry& re, uint32_t e) {
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(re.a.x), "=f"(re.a.y), "=f"(re.a.z), "=f"(re.a.w) : "r"(e));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+2048];" : "=f"(re.b.x), "=f"(re.b.y), "=f"(re.b.z), "=f"(re.b.w) : "r"(e));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+4096];" : "=f"(re.c.x), "=f"(re.c.y), "=f"(re.c.z), "=f"(re.c.w) : "r"(e));
            asm volatile("ld.shared.b32 %0, [%1+6144];" : "=r"(re.w) : "r"(e));
        };
        int v = -2 * lane;                                          // stream index of the next even entry to fetch
        uint32_t off = (uint32_t)(((run0 >> 1) - lane) & 63) << 4;  // its offset in the ring's 1 KB window
        uint32_t e_even = zero_s;
        auto fetch_even = [&](RawEntry& re) {
            e_even = (unsigned)v < (unsigned)run_len ? ring_s + off : zero_s;
            v += 2;
            off = (off + 16) & 1023;
            load_entry(re, e_even);
        };
        auto fetch_odd = [&](RawEntry& re) { load_entry(re, e_even + 1024); };  // (runs have even lengths: same range)
        fill(run0 >> 5);
        fill((run0 >> 5) + 1);
        fill_wait();

        // ---- an event (every 16 steps): flush what lane 31 handed out, new exponents for all lanes, the next 16 boundary
        //      records for lane 0.  `last`: behind the loop, only the flush.
        auto event = [&](int s, bool last) {
            // 0. records of the steps s-16 .. s-1 (entries s-79 .. s-64), at the exponent lane 31 had during those steps
            if (has_out) {  // (warp-uniform)
                const int exo = __shfl_sync(PHMM_FULL, ex, 31);
                __syncwarp();
                const int eo = s - 79 + lane;
                if (lane < LONG_EVERY && (unsigned)eo < (unsigned)n_ent) {
                    const float2 o = sm.rout[lane];
                    st_strong_f4(p.records + it.buf0 + (int64_t)strip * n_ent + eo, make_float4(o.x, o.y, __int_as_float(exo), 0.f));
                }
                __syncwarp();
                if (lane == 0 && !last && s > 63 && (s & (p.publish - 1)) == 0)
                    st_release_gpu(p.progress + it.prog0 + strip, min(s - 63, n_ent));  // release: MEMBAR + strong store
            }
            if (last) return;
            // 1. the boundary records lane 0 consumes in the steps s .. s+15 (their loads fly while the maximum is taken)
            float4 rec = make_float4(0.f, 0.f, 0.f, 0.f);
            const bool in_now = has_in && s < n_ent;  // (warp-uniform)
            if (in_now) {
                const int need = min(s + LONG_EVERY, n_ent);
                if (need > seen) {  // (the producer is usually far ahead: one look every few hundred steps)
                    const int* inprog = p.progress + it.prog0 + strip - 1;
                    int q = ld_relaxed_gpu(inprog);
                    while (q < need) { __nanosleep(100); q = ld_relaxed_gpu(inprog); }
                    seen = q;
                }
                const float4* src = p.records + it.buf0 + (int64_t)(strip - 1) * n_ent;
                if (pre == s) {  // copied in during the last 16 steps
                    asm volatile("cp.async.wait_group 0;" ::: "memory");
                    if (lane < LONG_EVERY && s + lane < n_ent) rec = sm.rraw[lane];
                } else if (lane < LONG_EVERY && s + lane < n_ent) {
                    rec = ld_strong_f4(src + s + lane);
                }
                // the records of the next event, if the producer has them already (it usually has): no L2 round trip then
                const int s2 = s + LONG_EVERY;
                pre = -1;
                if (s2 < n_ent && seen >= min(s2 + LONG_EVERY, n_ent)) {
                    if (lane < LONG_EVERY && s2 + lane < n_ent)
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(&sm.rraw[lane])), "l"(src + s2 + lane) : "memory");
                    asm volatile("cp.async.commit_group;" ::: "memory");
                    pre = s2;
                }
            }
            // 2. own proposal (none for a lane that holds nothing) and what can LEAVE this lane on its right within the next 16
            // steps: the .y half (columns 16..31) as it stands; a value in column x < 16 moves at most 16 columns along
            // diagonals in 16 rows and has to be deleted across the other 16 - x (gamma_max per column; charged per group of
            // four columns, at the group's last).  All values are >= 0, so float order is integer order and a power of two is a
            // step of the exponent field.  (Proposing the lane maximum instead, as until late in round 2, charges a lane
            // whose large values sit at its left edge -- every lane of a deletion corridor -- 32 columns = 106 bits too little,
            // and the lanes to its right were pushed up until the cells at their own right edge, 103 bits below their maximum,
            // fell off fp32's range: M states inside a long deletion that split it in two, worth 0.6 % of the likelihood of a
            // two-stretch read.)
            static_assert(NV % 4 == 0, "the exit bound below groups the columns of the .x half by four");
            constexpr int NG = NV / 4;
            const int hcs_now = s < 64 + LONG_EVERY ? 0 : hcs;  // (no loss per column while the run-in entry is in the strip, see hop_now)
            int gy0 = max(__float_as_int(ln.outS.y), __float_as_int(ln.outT.y)), gy1 = max(__float_as_int(ln.outS.x), __float_as_int(ln.outT.x));
            int gx[NG];
#pragma unroll
            for (int q = 0; q < NG; q++) {
                gx[q] = max(__float_as_int(ln.Tt[4 * q].x), __float_as_int(ln.J[4 * q].x));
#pragma unroll
                for (int x = 4 * q + 1; x < 4 * q + 4; x++) gx[q] = max(gx[q], max(__float_as_int(ln.Tt[x].x), __float_as_int(ln.J[x].x)));
            }
#pragma unroll
            for (int x = 0; x < NV; x += 2) {
                gy0 = max(gy0, max(__float_as_int(ln.Tt[x].y), __float_as_int(ln.J[x].y)));
                gy1 = max(gy1, max(__float_as_int(ln.Tt[x + 1].y), __float_as_int(ln.J[x + 1].y)));
            }
            const int gy = max(gy0, gy1);
            int mall = gy, mo = gy;
#pragma unroll
            for (int q = 0; q < NG; q++) {  // the group's last column, 4q + 3, is 2NV - 4q - 3 columns from the lane's right edge: 16 of them may be diagonal
                const int del = 2 * NV - 19 - 4 * q;
                mall = max(mall, gx[q]);
                mo = max(mo, gx[q] - (del > 0 ? del : 0) * hcs_now);
            }
            const float m = __int_as_float(mall);
            int c = m > 0.f ? ex + max(Fx<float>::ilogb(m) - LONG_TGT, -127) : LONG_FLOOR;  // (the shift 2^(ex - ex') stays one factor)
            const int cout = mo >= 0x00800000 ? ex + (mo >> 23) - 127 - LONG_TGT : LONG_FLOOR;
            // Soundness of the 16-step interval: a lane whose own maximum stood at 2^TGT one event ago and has dropped by more
            // than LONG_DROP bits since (it takes gap-continuation qualities above 20, i.e. more than ~7 bits lost per row on every
            // path) may have flushed values that were NOT negligible (less than 166 - LONG_DROP bits below that maximum): the pair is
            // recomputed by the fp64 chain kernel.  Only while the lane is inside the read's rows and holds real columns.
            {
                const int e = s - 2 * lane;
                const int lane_hi = (min(k - strip * STRIP, STRIP) - 1) / N2;  // lanes that hold real columns
                if (sm.own[lane] && lane <= lane_hi && e - LONG_EVERY >= 1 && e + 1 <= l && !(m > 0.f && Fx<float>::ilogb(m) >= LONG_TGT - LONG_DROP))
                    sm.lossy = 1;
            }
            int bmax = LONG_FLOOR;
            if (in_now) {
                const float mi = fmaxf(rec.x, rec.y);
                bmax = mi > 0.f ? __float_as_int(rec.z) + Fx<float>::ilogb(mi) : LONG_FLOOR;
#pragma unroll
                for (int o = 8; o > 0; o >>= 1) bmax = max(bmax, __shfl_xor_sync(PHMM_FULL, bmax, o));
                bmax = __shfl_sync(PHMM_FULL, bmax, 0);
            }
            // 3. ex'_L = max(c_L, max over the 8 lanes m < L of o_m - KTOT - (L - 1 - m) HOP), o_m = the exponent of what can
            //    leave lane m (above), the boundary records counting as a lane to the left of lane 0.  What lane m holds can
            //    reach lane L within the next 16 steps only through the running sum, which loses HOP = 32 log2(1 / gamma_max)
            //    bits per full lane it crosses (a deletion per column), and crossing a lane takes two steps: nothing that
            //    reaches lane L before the next event is stored above 2^(TGT+KTOT) there -- up to the 16 columns a value
            //    may cover along diagonals instead, which a stretch that starts abruptly could turn into an overflow: inf and
            //    NaN persist into Eq.4's total and send the pair to fp64 (below).  And what is flushed in lane L -- a cell more
            //    than 2^-(126+TGT+KTOT) 2^-((L-1-m) HOP) below what leaves lane m -- is negligible against lane m's own
            //    continuation into lane L.  (A constraint without the HOP term, as first written, flushes the start of a
            //    second matching stretch a few hundred columns to the right of the first one: reads with a long deletion against
            //    the haplotype came out too small by up to 240 in log10; with the HOP term but the lane MAXIMUM as o_m, over the
            //    whole prefix of lanes instead of 8, the far ends of the lanes inside such a deletion were flushed: 0.6 %.)
            const int bsrc = bmax > LONG_FLOOR ? bmax - LONG_TGT : LONG_FLOOR;
            // (the run-in entry -- row 0 of Eq.1 -- carries C/k through every column undiminished, gamma := 1: no HOP until it
            // has left the strip's last lane, at step 63)
            const int hop_now = s < 64 + LONG_EVERY ? 0 : hop;
            // (a window of 8 lanes: crossing a lane takes two steps, so nothing further to the left arrives before the next event)
            int pm = cout;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                const int t = __shfl_up_sync(PHMM_FULL, pm, o) - o * hop_now;
                if (lane >= o) pm = max(pm, t);
            }
            pm = __shfl_up_sync(PHMM_FULL, pm, 1);
            if (lane == 0) pm = LONG_FLOOR;
            if (lane < 8) pm = max(pm, bsrc - lane * hop_now);
            if (pm > LONG_FLOOR / 2) c = max(c, pm - LONG_KTOT);
            const int exn = c < LONG_FLOOR / 2 ? ex : c;  // nothing held, nothing to the left: keep the exponent
            sm.own[lane] = m > 0.f && exn == ex + Fx<float>::ilogb(m) - LONG_TGT;  // (a clamped proposal does not count)
            // 4. rescale the state: d <= 127 when something is held (the proposal is clamped), any d when nothing is
            const float f = pow2f(m > 0.f ? ex - exn : 0);  // 0 for d < -126: what is held is negligible against what arrives
            const float2 F = make_float2(f, f);
#pragma unroll
            for (int x = 0; x < NV; x++) { ln.Tt[x] = __fmul2_rn(ln.Tt[x], F); ln.J[x] = __fmul2_rn(ln.J[x], F); }
            ln.outS = __fmul2_rn(ln.outS, F);
            ln.outT = __fmul2_rn(ln.outT, F);
            ex = exn;
            const int exl = __shfl_up_sync(PHMM_FULL, ex, 1);
            f_in = pow2f(exl - ex);  // (exl - ex <= KTOT by construction; lane 0 does not use it)
            // 5. lane 0's next 16 boundary values at its new exponent; in the first strip: Eq.1 (reading G1), the run-in
            //    entry injects s = C/k = 1/k and T = g_1 C/k at exponent 0, every other entry nothing
            {
                const int ex0 = __shfl_sync(PHMM_FULL, ex, 0);
                if (lane < LONG_EVERY) {
                    float2 o = make_float2(0.f, 0.f);
                    if (has_in) {
                        const int dd = __float_as_int(rec.z) - ex0;
                        o = make_float2(scale2(rec.x, dd), scale2(rec.y, dd));
                    } else if (s == 0 && lane == 0) {
                        const float Cok = __frcp_rn((float)k);  // (k < 2^24: the correctly rounded 1/k)
                        float g1;  // C of the run-in entry = g_1: chunk plane 1, first float of the entry at run0
                        asm volatile("ld.shared.f32 %0, [%1+2048];" : "=f"(g1) : "r"(ring_s + ((uint32_t)((run0 >> 1) & 63) << 4)));
                        o = make_float2(Cok, g1 * Cok);
                    }
                    sm.rin[lane] = o;
                }
                __syncwarp();
            }
        };

        const uint32_t sum_y = META_SUM << 16;
        const bool lane0 = lane == 0, lane31 = lane == 31;
        auto one_step = [&](const RawEntry& re, uint32_t slot) {  // slot: shared-memory address of rin[step & 15]
            Entry2<float> E;
            E.gam = make_float2(re.a.x, re.a.y); E.A = make_float2(re.a.z, re.a.w);
            E.C = make_float2(re.b.x, re.b.y); E.G = make_float2(re.b.z, re.b.w);
            E.pmx = re.c.x; E.pxx = re.c.y; E.pmy = re.c.z; E.pxy = re.c.w;
            E.metaX = re.w & 0xffu; E.metaY = (re.w >> 16) & 0xffu;
            E.r2 = re.w & 0xff00ff00u;
            const float prevT = ln.outT.y;
            float2 bin;
            asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(bin.x), "=f"(bin.y) : "r"(slot));
            float inS = __shfl_up_sync(PHMM_FULL, ln.outS.y, 1) * f_in;
            float inT = __shfl_up_sync(PHMM_FULL, prevT, 1) * f_in;
            inS = lane0 ? bin.x : inS;
            inT = lane0 ? bin.y : inT;
            if (E.metaX & META_SUM) inS = 0.f;  // Eq.4: every lane sums its own columns only
            ln.step(E, inS, inT);
            if (re.w & sum_y) {  // this lane's .y half has just finished the sum entry: its share of Eq.4
                // M+I of column j reaches the sum through the T of column j+1; a strip whose last real column is the last
                // column of its lane has that one in what the lane handed out one step ago (unless the next strip counts it)
                const int k_loc = min(k - strip * STRIP, STRIP), out_lane = (k_loc - 1) / N2;
                if (lane <= out_lane) {
                    const bool full = !has_out && lane == out_lane && (k_loc % N2) == 0;
                    sm.fin[lane] = make_float2(full ? ln.outS.y + prevT : ln.outS.y, __int_as_float(ex));
                }
            }
            if (lane31) {  // right boundary of the strip: staged, flushed to the records at the next event
                asm volatile("st.shared.f32 [%0+128], %1;" ::"r"(slot), "f"(ln.outS.y) : "memory");
                asm volatile("st.shared.f32 [%0+132], %1;" ::"r"(slot), "f"(ln.outT.y) : "memory");
            }
        };

        RawEntry eA, eB;
        fetch_even(eA);
        // lane 31's .y half finishes entry run_len - 1 >= n_ent - 1 at step run_len + 62; a multiple of 16 steps
        const int steps = (run_len + 64 + 15) & ~15;
        for (int s = 0; s < steps; s += 2) {
            const bool ev = (s & (LONG_EVERY - 1)) == 0, fl = ((run0 + s + 2) & 31) == 0;
            if (ev | fl) {  // (one branch per two steps)
                if (ev) event(s, false);
                if (fl) {  // lane 0's next fetch enters a new block (now complete): the one after it starts its way in
                    fill_wait();
                    fill(((run0 + s + 2) >> 5) + 1);
                }
            }
            const uint32_t slot = rin_s + ((s & (LONG_EVERY - 2)) << 3);
            fetch_odd(eB);
            one_step(eA, slot);
            fetch_even(eA);
            one_step(eB, slot + 8);
        }
        event(steps, true);

        // ---- Eq.4: combine the lanes' shares, then the strips' (each strip waits for the total of the strips to its left)
        const float2 fin = sm.fin[lane];
        __syncwarp();
        const float fin_m = sm.lossy ? __int_as_float(0x7fc00000) : fin.x;  // (NaN poisons the total)
        const int fin_e = __float_as_int(fin.y);
        int em = fin_m > 0.f ? fin_e + Fx<float>::ilogb(fin_m) : LONG_FLOOR;  // exponent of the largest share
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) em = max(em, __shfl_xor_sync(PHMM_FULL, em, o));
        // in units of 2^em; a share that is neither zero nor a positive number (NaN: an overflow upstream) poisons the total
        double tot = fin_m > 0.f ? ldexp((double)fin_m, max(fin_e - em, -1000)) : (fin_m == 0.f ? 0.0 : (double)fin_m);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(PHMM_FULL, tot, o);
        if (lane == 0) {  // (the lane that publishes the progress counter)
            double acc = tot;
            int acc_e = em;
            if (has_in) {  // total of the strips to the left: (double mantissa, exponent), published behind the last record
                const int* inprog = p.progress + it.prog0 + strip - 1;
                int q = seen;
                while (q < n_ent + 1) { q = ld_relaxed_gpu(inprog); if (q < n_ent + 1) __nanosleep(100); }
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
                st_release_gpu(p.progress + it.prog0 + strip, n_ent + 1);
            } else if (acc > 0.0 && acc < 1e300) {  // (finite and positive; acc is a sum of normal floats)
                p.out[pair] = log10(acc) + (double)acc_e * LOG10_2;
                if (p.flags) p.flags[pair] = p.flag_bits;
            } else {  // overflow or a vanished sum: the fp64 chain kernel recomputes the pair
                const int idx = atomicAdd(p.fallback_count, 1);
                p.fallback_list[idx] = pair;
            }
        }
        __syncwarp();
    }
}

// ---- input guard of the fp32 long kernel.  Inside one lane (32 columns, 2 rows) everything shares one exponent, 166 bits of
// range below the lane's maximum A.  A cell B of the same lane that is flushed can never matter later if A's path can reach B's
// continuation for less than those 166 bits: either by deleting up to 31 columns in B's row (cost 31 x 0.332 x GCP of the row +
// the gap-open cost) or by inserting up to 32 rows (0.332 x the sum of their GCP qualities + the open cost).  At GCP 10 both
// bridges cost ~125 bits: 40 bits of margin, what is flushed weighs < 2^-40.  A read with any GCP quality above 10 is marked
// and k_long_f32 hands its pairs to the fp64 chain kernel.  (Found by fuzzing with per-base GCP between 3 and 40: results
// off by up to 0.6 in log10 with no non-finite value to detect.)  Second condition, the padding columns of the haplotype's
// last lane: mismatch diagonals seeded by the real columns keep running there at the cost of a mismatch per row
// (0.332 Qbase + 1.585 bits) while the real cells, once their diagonals have run off the haplotype's end, pay a gap
// continuation per row (0.332 GCP): where base qualities stay below ~5 for long, the padding outgrows the real cells and
// takes the lane's exponent with it.  A read whose best stretch of rows gains the padding more than 60 bits is marked too.
// One warp per read; every lane scans a contiguous share of the rows, the shares are combined (maximum subarray).
__global__ void k_read_risk(DevBatch b, int qual_offset, int64_t r0, int64_t r1, uint8_t* __restrict__ risk) {
    const int64_t r = r0 + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (r >= r1) return;
    const int lane = threadIdx.x & 31;
    const int64_t off = b.read_off[r];
    const int l = (int)(b.read_off[r + 1] - off);
    const int seg = (l + 31) / 32, lo = min(l, lane * seg), hi = min(l, lo + seg);
    bool bad = false;
    int gmin = 255;
    // maximum-subarray summary of this lane's rows: total, best prefix, best suffix, best
    float tot = 0.f, pre = 0.f, suf = 0.f, best = 0.f;
    for (int i = lo; i < hi; i++) {
        const int g = max((int)b.qual_gcp[off + i] - qual_offset, 0), q = max((int)b.qual_base[off + i] - qual_offset, 0);
        if (g > 10) bad = true;
        gmin = min(gmin, g);
        const float v = 0.332f * (float)(g - q) - 1.585f;
        tot += v;
        pre = fmaxf(pre, tot);
        suf = fmaxf(suf + v, 0.f);
        best = fmaxf(best, suf);
    }
    for (int o = 1; o < 32; o <<= 1) {  // inclusive scan of the summaries, left to right
        const float t2 = __shfl_up_sync(PHMM_FULL, tot, o), p2 = __shfl_up_sync(PHMM_FULL, pre, o);
        const float s2 = __shfl_up_sync(PHMM_FULL, suf, o), b2 = __shfl_up_sync(PHMM_FULL, best, o);
        if (lane >= o) {  // (left = the shuffled one, right = this lane's)
            best = fmaxf(fmaxf(best, b2), s2 + pre);
            pre = fmaxf(p2, t2 + pre);
            suf = fmaxf(suf, s2 + tot);
            tot = t2 + tot;
        }
    }
    if (best > 60.f) bad = true;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) gmin = min(gmin, __shfl_xor_sync(PHMM_FULL, gmin, o));
    bad = __any_sync(PHMM_FULL, bad);
    if (lane == 0) risk[r] = bad ? 255 : (uint8_t)gmin;  // (gmin <= 10 where not marked)
}

cudaError_t launch_read_risk(const DevBatch& b, int qual_offset, int64_t r0, int64_t r1, uint8_t* risk, cudaStream_t st) {
    if (r1 <= r0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(risk + r0, 0, (size_t)(r1 - r0), st);
    if (e != cudaSuccess) return e;
    k_read_risk<<<(unsigned)((r1 - r0 + 7) / 8), 256, 0, st>>>(b, qual_offset, r0, r1, risk);
    return cudaGetLastError();
}

cudaError_t launch_long_f32(const DevBatch& b, const LongLaunch& p, int grid_ctas, cudaStream_t st) {
    if (grid_ctas <= 0) return cudaSuccess;
    if (b.n_wild) k_long_f32<SHORT_NV, false><<<grid_ctas, LONG_WPC * 32, 0, st>>>(b, p);
    else k_long_f32<SHORT_NV, true><<<grid_ctas, LONG_WPC * 32, 0, st>>>(b, p);
    return cudaGetLastError();
}

int long_ctas_per_sm() {
    int n = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_long_f32<SHORT_NV, true>, LONG_WPC * 32, 0);
    return n > 0 ? n : 1;
}
int long_warps_per_cta() { return LONG_WPC; }

}  // namespace phmm
