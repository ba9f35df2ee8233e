// fp64 recomputation of short pairs (PHMM_FP64 mode for short pairs):
// device-side binning of the pairs by lane-group size, then a sub-warp systolic kernel in double.
//
// One thread = ONE virtual lane of RESCUE_NV haplotype columns (fp64 has no packed form, so nothing is
// gained by two halves per thread); lane L of a group runs one stream entry (read row) behind lane L-1.
// A group works on one pair; a warp holds floor(32/g) groups of the same size g = ceil(k / RESCUE_NV).
// Which pairs land here is only known on the device (the fp32 kernel's underflow test), so the queue is
// binned there: the producer takes a ticket in its size bucket, k_rescue_plan turns the 33 bucket counts
// into warp and list offsets, k_rescue_scatter orders the queue by bucket, and the persistent kernel
// k_rescue_f64 hands out whole warps by ticket.
//
// Arithmetic: the plain (unscaled-I) row-wise form of Eq.6-7 with the row constants formed on the fly
// from the quality bytes -- no division, no table:
//     M      = p_{i,x} * T[x]                                 (Eq.3 select)            MUL
//     s'     = gamma_i * s + M                                S_{i,x}, the serial chain  FMA
//     T[x+1] = a_{i+1} M + g_{i+1} I[x] + c_{i+1} s           c_{i+1} = g_{i+1} d_i     MUL + 2 FMA
//     I[x]   = iota_{i+1} M + gamma_{i+1} I[x]                                           MUL + FMA
// = 7 DP instructions per cell.  Entry 0 is the run-in row (p = 0, gamma_0 := 1, d_0 := 1; the first
// lane injects s = C/k: Eq.1 under reading G1); behind the last row a' = g' = c' := 0 and iota' =
// gamma' := 1, which leaves I[x] = M_l + I_l, the summand of Eq.4.  Scale constant C = 2^1000
// (PAPER.md:61 uses 2^1020; 20 bits of head room because with per-base qualities L is bounded by a
// small constant, not by 1: SURVEY 8(c) item 3).  A result that is still not a normal finite number
// goes on to the rescaled chain kernel.
#include "phmm_common.cuh"
#include "phmm_kernels.h"
#include "phmm_table.cuh"

namespace phmm {

constexpr int RESCUE_WARPS = 4;
#ifndef RESCUE_MIN_CTAS
#define RESCUE_MIN_CTAS 2
#endif
constexpr int RESCUE_LOG2C = 1000;

// ---- binning
// counters (RescueQueue::cnt): [0..RESCUE_NB) items per (g, length class) bucket, g-major; RQ_TICKET, RQ_NQUEUE, RQ_FALLBACK
// plan (ints): [0..33] first warp of lane-group size g (exclusive prefix; [33] = total warps), [34..67] first list slot of
// size g, [68 + bucket] first list slot of each bucket.  One block of 1024 threads.
__global__ void __launch_bounds__(1024) k_rescue_plan(const int* __restrict__ cnt, int* __restrict__ plan) {
    __shared__ int s_part[1024];
    __shared__ int s_g[34];
    constexpr int PER = (RESCUE_NB + 1023) / 1024;
    const int t = threadIdx.x, lo = t * PER, hi = min(lo + PER, RESCUE_NB);
    int sum = 0;
    for (int i = lo; i < hi; i++) sum += cnt[i];
    s_part[t] = sum;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {  // inclusive scan of the partial sums
        const int v = t >= o ? s_part[t - o] : 0;
        __syncthreads();
        s_part[t] += v;
        __syncthreads();
    }
    int run = s_part[t] - sum;
    for (int i = lo; i < hi; i++) { plan[68 + i] = run; run += cnt[i]; }
    __syncthreads();
    if (t <= 33) s_g[t] = t <= 32 ? plan[68 + t * RESCUE_LCLS] : s_part[1023];  // first slot of size g; total
    __syncthreads();
    if (t == 0) {
        int w = 0;
        for (int g = 0; g <= 32; g++) {
            plan[g] = w; plan[34 + g] = s_g[g];
            const int c = s_g[g + 1] - s_g[g];
            if (g >= 1) w += (c + (32 / g) - 1) / (32 / g);
        }
        plan[33] = w; plan[34 + 33] = s_g[33];
    }
}

__global__ void k_rescue_scatter(const int4* __restrict__ queue, const int* __restrict__ cnt, const int* __restrict__ plan,
                                 int* __restrict__ sorted) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cnt[RQ_NQUEUE]) return;
    const int4 q = queue[i];  // pair, bucket, ticket within the bucket
    sorted[plan[68 + q.y] + q.z] = q.x;
}

// PHMM_FP64 mode: every short pair is queued (no fp32 pass ran)
__global__ void k_rescue_enqueue(DevBatch b, RescueQueue rq, const int* __restrict__ pairs, int n, const int* __restrict__ pair_read,
                                 const int* __restrict__ pair_hap) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int pair = pairs[i];
    const int r = pair_read[pair], h = pair_hap[pair];
    rescue_push(rq, pair, (int)(b.hap_off[h + 1] - b.hap_off[h]), (int)(b.read_off[r + 1] - b.read_off[r]));
}

// ---- the kernel
struct RescueArgs {
    const int* sorted;       // pairs ordered by bucket
    const int* plan;         // see k_rescue_plan
    int* ticket;
    const int* pair_read;
    const int* pair_hap;
    const double* lut;       // 256 entries 10^(-q/10)
    double* out;
    uint8_t* flags;
    uint8_t flag_bits;
    int* fallback_count;     // results that are not normal finite numbers: queue for the rescaled chain kernel
    int* fallback_list;
    int* fallback_stat;      // number of such pairs (statistics only)
};

__global__ void __launch_bounds__(RESCUE_WARPS * 32, RESCUE_MIN_CTAS) k_rescue_f64(DevBatch b, RescueArgs p) {
    constexpr int NV = RESCUE_NV;
    __shared__ double s_lut[512];  // [0..255] gap qualities, [256..511] base qualities (phmm_rowconst.cuh)
    __shared__ int s_plan[68];
    for (int i = threadIdx.x; i < 512; i += blockDim.x) s_lut[i] = p.lut[i];
    for (int i = threadIdx.x; i < 68; i += blockDim.x) s_plan[i] = p.plan[i];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int total_warps = s_plan[33];
    const double LOG10_2 = 0.30102999566398119521;

    for (;;) {
        int w = 0;
        if (lane == 0) w = atomicAdd(p.ticket, 1);
        w = __shfl_sync(PHMM_FULL, w, 0);
        if (w >= total_warps) break;
        int g = 1;
        while (g < 32 && w >= s_plan[g + 1]) g++;    // bucket of this warp (33 entries, warp-uniform)
        const int per = 32 / g;                       // pairs per warp
        const int grp = lane / g, lg = lane - grp * g;
        const int slot = (w - s_plan[g]) * per + grp;  // index within the bucket
        const bool active = grp < per && slot < s_plan[34 + g + 1] - s_plan[34 + g];
        int pair = -1, l = 0, k = 1;
        int64_t ro = 0, ho = 0;
        if (active) {
            pair = p.sorted[s_plan[34 + g] + slot];
            const int r = p.pair_read[pair], h = p.pair_hap[pair];
            ro = b.read_off[r]; ho = b.hap_off[h];
            l = (int)(b.read_off[r + 1] - ro); k = (int)(b.hap_off[h + 1] - ho);
        }
        int steps = active ? l + g : 0;  // entries 0..l, lane lg one entry behind lane lg-1
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) steps = max(steps, __shfl_xor_sync(PHMM_FULL, steps, o));

        // ---- haplotype columns of this lane: one match word per base (bit x <=> column x carries that base)
        const int j0 = lg * NV;
        const int nv = active ? min(max(k - j0, 0), NV) : 0;
        uint32_t hm[5] = {0u, 0u, 0u, 0u, 0u};  // one per base code; [4] = N (Eq.3 compares literally: N matches N only, reading G17)
        for (int x = 0; x < nv; x++) {
            const int c = base_code(b.hap_bases[ho + j0 + x]);
#pragma unroll
            for (int q = 0; q < 5; q++) hm[q] |= ((c == q || (b.n_wild && c == 4)) ? 1u : 0u) << x;
        }
        const double Cok = ldexp(1.0, RESCUE_LOG2C) / (double)k;

        double T[NV], I[NV];
#pragma unroll
        for (int x = 0; x < NV; x++) { T[x] = 0.0; I[x] = 0.0; }
        double outS = 0.0, outT = 0.0, sig = 0.0;
        double gam_own = 1.0, d_own = 1.0;  // gamma_i and d_i of the entry about to be processed (entry 0: both := 1)

        for (int s = 0; s < steps; s++) {
            const int e = s - lg;  // stream entry = read row (0 = run-in)
            const bool on = active && e >= 0 && e <= l;
            // ---- a1: row constants on the fly
            double pm = 0.0, px = 0.0, gam = 0.0, an = 0.0, gn = 0.0, cn = 0.0, in_ = 0.0, gan = 0.0;
            uint32_t mw = 0u;
            if (on) {
                gam = gam_own;
                if (e >= 1) {
                    const double eps = s_lut[256 + b.qual_base[ro + e - 1]];
                    const int code = base_code(b.read_bases[ro + e - 1]);
                    px = eps * (1.0 / 3.0);  // within 1 ulp of Eq.3's eps/3; a double division per step would cost ~10 % here
                    pm = 1.0 - eps;
                    if (b.n_wild && code == 4) px = pm;  // n_is_wildcard: a read N matches every column
                    const uint32_t m01 = (code & 1) ? hm[1] : hm[0], m23 = (code & 1) ? hm[3] : hm[2];
                    mw = (code & 4) ? hm[4] : (code & 2) ? m23 : m01;
                }
                if (e < l) {
                    const double io1 = s_lut[b.qual_ins[ro + e]], de1 = s_lut[b.qual_del[ro + e]], ga1 = s_lut[b.qual_gcp[ro + e]];
                    an = 1.0 - io1 - de1; gn = 1.0 - ga1; cn = gn * d_own; in_ = io1; gan = ga1;
                    gam_own = ga1; d_own = de1;
                } else {
                    in_ = 1.0; gan = 1.0;  // behind the last row: I[x] <- M_l + I_l (Eq.4 summand)
                }
            }
            // ---- left boundary
            double inS = __shfl_up_sync(PHMM_FULL, outS, 1), inT = __shfl_up_sync(PHMM_FULL, outT, 1);
            double inSig = __shfl_up_sync(PHMM_FULL, sig, 1);
            if (lg == 0) {  // column-0 boundary, Eq.1: only the run-in entry injects
                inS = (on && e == 0) ? Cok : 0.0;
                inT = cn * inS;
                inSig = 0.0;
            }
            double sr = inS;
            double M = ((mw & 1u) ? pm : px) * T[0];
            T[0] = inT;
#pragma unroll
            for (int x = 0; x < NV; x++) {
                double Mn = M;
                if (x + 1 < NV) Mn = ((mw & (1u << (x + 1))) ? pm : px) * T[x + 1];
                const double t2 = fma(gn, I[x], an * M);
                const double Tn = fma(cn, sr, t2);
                I[x] = fma(gan, I[x], in_ * M);
                sr = fma(gam, sr, M);
                if (x + 1 < NV) T[x + 1] = Tn; else outT = Tn;
                M = Mn;
            }
            outS = sr;
            if (on && e == l) {  // Eq.4
                double a = 0.0;
#pragma unroll
                for (int x = 0; x < NV; x++) a += (x < nv) ? I[x] : 0.0;
                sig = inSig + a;
                if (lg == g - 1) {
                    const double v = log10(sig) - (double)RESCUE_LOG2C * LOG10_2;
                    if (sig >= 1e-290 && sig < 1e300) {
                        p.out[pair] = v;
                        if (p.flags) p.flags[pair] = p.flag_bits;
                    } else {
                        const int idx = atomicAdd(p.fallback_count, 1);
                        p.fallback_list[idx] = pair;
                        atomicAdd(p.fallback_stat, 1);
                    }
                }
            }
        }
        __syncwarp();
    }
}

// ---- the table-driven kernel (PHMM_FP32_RESCUE: recomputation of what the fp32 kernel could not represent)
// The same T/J engine as the fp32 kernels (phmm_engine.cuh: 5 floating-point instructions per cell instead of 7) in double,
// one lane = RESCUE_NV columns, lane L one stream entry behind lane L-1, fed from the row-constant TABLE of the short
// path: the entries are loaded one step ahead and widened to double.  The constants are the fp32-rounded ones -- these
// pairs need fp64's range, not its precision: their results are part of the PHMM_FP32_RESCUE outputs, tolerance 1e-3
// (observed ~1e-6); PHMM_FP64 runs k_rescue_f64 above with constants formed in double.  Eq.4 comes out of the running
// sum on the table's sum entry exactly as in the short kernel; C = 2^1000.
struct RawT { float gam, A, C, G, pm, px; uint32_t w; };

__global__ void __launch_bounds__(RESCUE_WARPS * 32, RESCUE_MIN_CTAS) k_rescue_f64t(DevBatch b, RescueArgs p, const float* __restrict__ table) {
    constexpr int NV = RESCUE_NV;
    __shared__ int s_plan[68];
    for (int i = threadIdx.x; i < 68; i += blockDim.x) s_plan[i] = p.plan[i];
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int total_warps = s_plan[33];
    const double LOG10_2 = 0.30102999566398119521;

    for (;;) {
        int w = 0;
        if (lane == 0) w = atomicAdd(p.ticket, 1);
        w = __shfl_sync(PHMM_FULL, w, 0);
        if (w >= total_warps) break;
        int g = 1;
        while (g < 32 && w >= s_plan[g + 1]) g++;    // lane-group size of this warp (warp-uniform)
        const int per = 32 / g;                       // pairs per warp
        const int grp = lane / g, lg = lane - grp * g;
        const int slot = (w - s_plan[g]) * per + grp;  // index within the size's list (ordered by read length)
        const bool active = grp < per && slot < s_plan[34 + g + 1] - s_plan[34 + g];
        int pair = -1, l = 0, k = 1, run0 = 0;
        int64_t ho = 0;
        if (active) {
            pair = p.sorted[s_plan[34 + g] + slot];
            const int r = p.pair_read[pair], h = p.pair_hap[pair];
            const int64_t ro = b.read_off[r];
            ho = b.hap_off[h];
            l = (int)(b.read_off[r + 1] - ro); k = (int)(b.hap_off[h + 1] - ho);
            run0 = (int)(table_run_start(ro, r) - b.table_base);
        }
        const int n_ent = l + 2;  // run-in entry, rows 1..l, sum entry
        int steps = active ? n_ent + g - 1 : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) steps = max(steps, __shfl_xor_sync(PHMM_FULL, steps, o));

        // ---- haplotype columns of this lane: one match word per base code, [4] = N; [5] = what "matches" the sum entry
        // (prior pm = 0): the columns more than one behind the haplotype's last (phmm_engine.cuh)
        const int j0 = lg * NV;
        const int nv = active ? min(max(k - j0, 0), NV) : 0;
        uint32_t hm[6] = {0u, 0u, 0u, 0u, 0u, 0u};
        for (int x = 0; x < nv; x++) {
            const int c = base_code(b.hap_bases[ho + j0 + x]);
#pragma unroll
            for (int q = 0; q < 5; q++) hm[q] |= ((c == q || (b.n_wild && c == 4)) ? 1u : 0u) << x;
        }
#pragma unroll
        for (int x = 0; x < NV; x++) hm[5] |= (j0 + x > k ? 1u : 0u) << x;
        const bool is_last = active && lg == g - 1;
        const bool full_last = k == g * NV;
        const double Cok = ldexp(1.0, RESCUE_LOG2C) / (double)k;

        double T[NV], J[NV];
#pragma unroll
        for (int x = 0; x < NV; x++) { T[x] = 0.0; J[x] = 0.0; }
        double outS = 0.0, outT = 0.0;

        // entry e of the pair's run (e < 0 or e >= n_ent: an all-zero entry of the table's zero run)
        auto fetch = [&](RawT& re, int e) {
            const int pos = (active && (unsigned)e < (unsigned)n_ent) ? run0 + e : 0;
            const float* q = table + 4 * ((((int64_t)(pos >> 5)) << 7) + (int64_t)((pos & 1) * 16 + ((pos >> 1) & 15)));
            re.gam = __ldg(q); re.A = __ldg(q + 2);
            re.C = __ldg(q + 128); re.G = __ldg(q + 130);
            re.pm = __ldg(q + 256); re.px = __ldg(q + 257);
            re.w = __ldg(reinterpret_cast<const uint32_t*>(q + 384));
        };
        RawT cur, nxt;
        fetch(cur, -lg);
        for (int s = 0; s < steps; s++) {
            fetch(nxt, s + 1 - lg);
            if (lg == 0 && active) {  // the group's leading lane asks L2 for the entry 24 steps ahead (4 chunk planes)
                const int pos = run0 + s + 24;
                const float* q = table + 4 * ((((int64_t)(pos >> 5)) << 7) + (int64_t)((pos & 1) * 16 + ((pos >> 1) & 15)));
#pragma unroll
                for (int c = 0; c < 4; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(q + 128 * c));
            }
            const double gam = (double)cur.gam, A = (double)cur.A, C = (double)cur.C, G = (double)cur.G;
            const double pm = (double)cur.pm, px = (double)cur.px;
            const uint32_t meta = cur.w & 0xffu;
            const uint32_t code = meta & META_CODE_MASK;
            const uint32_t m01 = (code & 1u) ? hm[1] : hm[0], m23 = (code & 1u) ? hm[3] : hm[2];
            uint32_t mw = (code & 4u) ? hm[4] : ((code & 2u) ? m23 : m01);
            mw = (meta & META_SUM) ? hm[5] : mw;
            // ---- left boundary
            const double prevT = outT;
            double inS = __shfl_up_sync(PHMM_FULL, outS, 1), inT = __shfl_up_sync(PHMM_FULL, prevT, 1);
            if (lg == 0) {  // column-0 boundary, Eq.1 (reading G1): only the run-in entry injects
                inS = (meta & META_FIRST) ? Cok : 0.0;
                inT = C * inS;
            }
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
            if (is_last && (meta & META_SUM)) {  // Eq.4: the running sum has collected M_l + I_l of every column
                const double sig = full_last ? outS + prevT : outS;
                if (sig >= 1e-290 && sig < 1e300) {
                    p.out[pair] = log10(sig) - (double)RESCUE_LOG2C * LOG10_2;
                    if (p.flags) p.flags[pair] = p.flag_bits;
                } else {
                    const int idx = atomicAdd(p.fallback_count, 1);
                    p.fallback_list[idx] = pair;
                    atomicAdd(p.fallback_stat, 1);
                }
            }
            cur = nxt;
        }
        __syncwarp();
    }
}

int rescue_ctas_per_sm() {
    int n = 0, m = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_rescue_f64, RESCUE_WARPS * 32, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&m, k_rescue_f64t, RESCUE_WARPS * 32, 0);
    n = n > m ? n : m;
    return n > 0 ? n : 1;
}

cudaError_t launch_rescue_f64(const DevBatch& b, const RescueLaunch& r, int grid_ctas, cudaStream_t st) {
    RescueQueue rq = r.queue;
    if (r.enqueue_pairs && r.n_enqueue > 0)
        k_rescue_enqueue<<<(r.n_enqueue + 255) / 256, 256, 0, st>>>(b, rq, r.enqueue_pairs, r.n_enqueue, r.pair_read, r.pair_hap);
    k_rescue_plan<<<1, 1024, 0, st>>>(rq.cnt, r.plan);
    if (r.max_queue > 0) k_rescue_scatter<<<(r.max_queue + 255) / 256, 256, 0, st>>>(rq.queue, rq.cnt, r.plan, r.sorted);
    RescueArgs a;
    a.sorted = r.sorted; a.plan = r.plan; a.ticket = rq.cnt + RQ_TICKET;
    a.pair_read = r.pair_read; a.pair_hap = r.pair_hap; a.lut = r.lut; a.out = r.out; a.flags = r.flags; a.flag_bits = r.flag_bits;
    a.fallback_count = r.fallback_count; a.fallback_list = r.fallback_list; a.fallback_stat = rq.cnt + RQ_FALLBACK;
    if (r.table) k_rescue_f64t<<<grid_ctas, RESCUE_WARPS * 32, 0, st>>>(b, a, r.table);
    else k_rescue_f64<<<grid_ctas, RESCUE_WARPS * 32, 0, st>>>(b, a);
    return cudaGetLastError();
}

}  // namespace phmm
