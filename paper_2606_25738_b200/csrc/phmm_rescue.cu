// fp64 recomputation of short pairs (PHMM_FP64 mode for short pairs):
// device-side binning of the pairs by lane-group size and read length, then a sub-warp systolic kernel in double.
//
// One thread = ONE virtual lane of RESCUE_NV haplotype columns (fp64 has no packed form, so nothing is
// gained by two halves per thread); lane L of a group runs one stream entry (read row) behind lane L-1.
// A group works on one pair; a warp holds floor(32/g) groups of the same size g = ceil(k / RESCUE_NV).
// Which pairs land here is only known on the device (the fp32 kernel's underflow test), so the queue is
// binned there: the producer takes a ticket in its (size, length) bucket, k_rescue_plan turns the bucket counts
// into warp and list offsets, k_rescue_scatter orders the queue by bucket, and the persistent kernel
// k_rescue_f64t hands out whole warps by ticket.
//
// Arithmetic: the T/J form of phmm_engine.cuh (5 instructions per cell) in double on table entries fetched one step
// ahead -- the fp32 table of the short path under PHMM_FP32_RESCUE, a table in double under PHMM_FP64.  Scale constant
// C = 2^1000 (PAPER.md:61 uses 2^1020; 20 bits of head room because with per-base qualities L is bounded by a
// small constant, not by 1: SURVEY 8(c) item 3).  A result that is still not a normal finite number
// goes on to the rescaled chain kernel.  (Round 1's kernel formed the constants from the quality bytes in every lane
// and step, 7 instructions per cell: 0.94 TCUPS in PHMM_FP64 against 1.38 now, 8.1 ms against 4.9 for configs[1]'s rescue.)
#include "phmm_common.cuh"
#include "phmm_kernels.h"
#include "phmm_rowconst.cuh"
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
    double* out;
    uint8_t* flags;
    uint8_t flag_bits;
    int* fallback_count;     // results that are not normal finite numbers: queue for the rescaled chain kernel
    int* fallback_list;
    int* fallback_stat;      // number of such pairs (statistics only)
};

// ---- the table-driven kernel (PHMM_FP32_RESCUE: recomputation of what the fp32 kernel could not represent)
// The same T/J engine as the fp32 kernels (phmm_engine.cuh: 5 floating-point instructions per cell instead of 7) in double,
// one lane = RESCUE_NV columns, lane L one stream entry behind lane L-1, fed from the row-constant TABLE of the short
// path: the entries are loaded one step ahead and widened to double.  The constants are the fp32-rounded ones -- these
// pairs need fp64's range, not its precision: their results are part of the PHMM_FP32_RESCUE outputs, tolerance 1e-3
// (observed ~1e-6); PHMM_FP64 reads a table whose constants are formed and kept in double (k_table_f64).  Eq.4 comes out of the running
// sum on the table's sum entry exactly as in the short kernel; C = 2^1000.
// TT = float: the fp32 table of the short path (layout: phmm_table.cuh).  TT = double (PHMM_FP64): the table k_table_f64
// below writes, constants formed and kept in double: blocks of 32 entries x 64 bytes, field-major inside a block (six planes
// of 32 doubles: gamma, A, C, G, pm, px, then 32 words), so that the lanes of a group, which read consecutive entries, read
// consecutive doubles.
template <typename TT> struct RawT { TT gam, A, C, G, pm, px; uint32_t w; };

__global__ void __launch_bounds__(256) k_table_f64(DevBatch b, const double* __restrict__ lut, double* __restrict__ table, int64_t r0, int64_t r1) {
    const int64_t r = r0 + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (r >= r1) return;
    const int lane = threadIdx.x & 31;
    const int64_t off = b.read_off[r];
    const int l = (int)(b.read_off[r + 1] - off);
    const int64_t first = table_run_start(off, r) - b.table_base;
    const int e_hi = min(table_run_len(l), ((int)blockIdx.y + 1) * 1024);
    for (int e = (int)blockIdx.y * 1024 + lane; e < e_hi; e += 32) {
        const RowC x = row_constants(b, lut, off, l, e, true);
        const int64_t pos = first + e;
        double* d = table + ((pos >> 5) << 8) + (pos & 31);
        d[0] = x.gam; d[32] = x.A; d[64] = x.C; d[96] = x.G; d[128] = x.pm; d[160] = x.px;
        reinterpret_cast<uint32_t*>(table + ((pos >> 5) << 8) + 192)[pos & 31] = x.meta & 0xffu;
    }
}

cudaError_t launch_table_f64(const DevBatch& b, const double* lut, double* table, int64_t r0, int64_t r1, int max_read_len, cudaStream_t st) {
    if (r1 <= r0) return cudaSuccess;
    const int64_t grid = (r1 - r0 + 7) / 8;
    const int chunks = (table_run_len(max_read_len) + 1023) / 1024;
    cudaError_t e = cudaMemsetAsync(table, 0, (size_t)TABLE_ZERO_RUN * 64, st);  // the zero run: entries outside a lane's stream
    if (e != cudaSuccess) return e;
    k_table_f64<<<dim3((unsigned)grid, (unsigned)chunks), 256, 0, st>>>(b, lut, table, r0, r1);
    return cudaGetLastError();
}

template <typename TT>
__global__ void __launch_bounds__(RESCUE_WARPS * 32, RESCUE_MIN_CTAS) k_rescue_f64t(DevBatch b, RescueArgs p, const TT* __restrict__ table) {
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
        auto fetch = [&](RawT<TT>& re, int e) {
            const int pos = (active && (unsigned)e < (unsigned)n_ent) ? run0 + e : 0;
            if constexpr (sizeof(TT) == 4) {
                const float* q = reinterpret_cast<const float*>(table) + 4 * ((((int64_t)(pos >> 5)) << 7) + (int64_t)((pos & 1) * 16 + ((pos >> 1) & 15)));
                re.gam = __ldg(q); re.A = __ldg(q + 2);
                re.C = __ldg(q + 128); re.G = __ldg(q + 130);
                re.pm = __ldg(q + 256); re.px = __ldg(q + 257);
                re.w = __ldg(reinterpret_cast<const uint32_t*>(q + 384));
            } else {
                const double* q = reinterpret_cast<const double*>(table) + (((int64_t)(pos >> 5)) << 8) + (pos & 31);
                re.gam = __ldg(q); re.A = __ldg(q + 32); re.C = __ldg(q + 64); re.G = __ldg(q + 96);
                re.pm = __ldg(q + 128); re.px = __ldg(q + 160);
                re.w = __ldg(reinterpret_cast<const uint32_t*>(q - (pos & 31) + 192) + (pos & 31));
            }
        };
        RawT<TT> cur, nxt;
        fetch(cur, -lg);
        for (int s = 0; s < steps; s++) {
            fetch(nxt, s + 1 - lg);
            if (lg == 0 && active) {  // the group's leading lane asks L2 for the entry 24 steps ahead
                const int pos = run0 + s + 24;
                if constexpr (sizeof(TT) == 4) {  // 4 chunk planes
                    const float* q = reinterpret_cast<const float*>(table) + 4 * ((((int64_t)(pos >> 5)) << 7) + (int64_t)((pos & 1) * 16 + ((pos >> 1) & 15)));
#pragma unroll
                    for (int c = 0; c < 4; c++) asm volatile("prefetch.global.L2 [%0];" ::"l"(q + 128 * c));
                } else {  // one of the 16 lines of the block per step (each is reached 16 times before lane 0 gets there)
                    const char* q = reinterpret_cast<const char*>(table) + (((int64_t)(pos >> 5)) << 11) + ((s & 15) << 7);
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(q));
                }
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
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_rescue_f64t<double>, RESCUE_WARPS * 32, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&m, k_rescue_f64t<float>, RESCUE_WARPS * 32, 0);
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
    a.pair_read = r.pair_read; a.pair_hap = r.pair_hap; a.out = r.out; a.flags = r.flags; a.flag_bits = r.flag_bits;
    a.fallback_count = r.fallback_count; a.fallback_list = r.fallback_list; a.fallback_stat = rq.cnt + RQ_FALLBACK;
    if (r.table_f64) k_rescue_f64t<double><<<grid_ctas, RESCUE_WARPS * 32, 0, st>>>(b, a, (const double*)r.table);
    else k_rescue_f64t<float><<<grid_ctas, RESCUE_WARPS * 32, 0, st>>>(b, a, (const float*)r.table);
    return cudaGetLastError();
}

}  // namespace phmm
