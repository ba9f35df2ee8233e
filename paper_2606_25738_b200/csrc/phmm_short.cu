// Short-pair path: row-constant table prologue + the sub-warp systolic fp32 kernel.
//
// Hot path rows of SURVEY.md section 8(a): a1 (quality -> row constants: table kernel), a2 (haplotype
// staging: match bitmasks in registers), a3/a4 (row updates), a5 (lane-to-lane carry: 4 shuffles per
// row), a9 (final reduction, log10), a10 (underflow detection -> rescue queue).
#include "phmm_engine.cuh"
#include "phmm_kernels.h"

namespace phmm {

// ------------------------------------------------------------------ a1: row-constant table
// One warp per read; entry 0 = reset row, entries 1..l = read rows.  Constants are formed in double
// from the 10^(-q/10) table and rounded once to float ("q32" table; Listing 2
// :293-295 for which qualities enter which transition).
__global__ void __launch_bounds__(256) k_table_f32(DevBatch b, const double* __restrict__ lut, float* __restrict__ table) {
    const int64_t r = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (r >= b.n_reads) return;
    const int lane = threadIdx.x & 31;
    const int64_t off = b.read_off[r];
    const int l = (int)(b.read_off[r + 1] - off);
    float4* dst = reinterpret_cast<float4*>(table) + 2 * (off + r);
    for (int i = lane; i <= l; i += 32) {
        float4 A, B;
        if (i == 0) {
            A = make_float4(0.f, 0.f, 0.f, 0.f);
            B = make_float4(0.f, 0.f, 1.f, (float)META_RESET);
        } else {
            const double eps = lut[b.qual_base[off + i - 1]], io = lut[b.qual_ins[off + i - 1]];
            const double de = lut[b.qual_del[off + i - 1]], ga = lut[b.qual_gcp[off + i - 1]];
            const double g = 1.0 - ga;
            const double gn = (i < l) ? 1.0 - lut[b.qual_gcp[off + i]] : 1.0;
            const double dp = (i > 1) ? lut[b.qual_del[off + i - 2]] : 1.0;
            uint32_t meta = (uint32_t)base_code(b.read_bases[off + i - 1]) | (i == l ? META_LAST : 0u);
            A = make_float4((float)(1.0 - io - de), (float)(1.0 - eps), (float)(eps / 3.0), (float)(g * dp));
            B = make_float4((float)(gn * io), (float)(ga * gn / g), (float)ga, (float)meta);
        }
        dst[2 * i] = A;
        dst[2 * i + 1] = B;
    }
}

cudaError_t launch_lut_table(const DevBatch& b, const double* lut, float* table, cudaStream_t st) {
    if (b.n_reads == 0) return cudaSuccess;
    const int wpb = 8;
    int64_t grid = (b.n_reads + wpb - 1) / wpb;
    k_table_f32<<<(unsigned)grid, wpb * 32, 0, st>>>(b, lut, table);
    return cudaGetLastError();
}

// ------------------------------------------------------------------ the short kernel
template <int NV> struct Cursor {  // where a lane's .x half is in its task's stream of table entries
    const float4* cur;
    const float4* nxt;
    int rem, nxtRem, q, wait;
};

template <int NV>
__global__ void __launch_bounds__(SHORT_WARPS_PER_CTA * 32, 3) k_short_f32(DevBatch b, ShortLaunch p) {
    typedef Lane<float, NV, false> L;
    constexpr int N2 = 2 * NV;
    const int warp = blockIdx.x * SHORT_WARPS_PER_CTA + (threadIdx.x >> 5);
    if (warp >= p.n_warps) return;
    const int lane = threadIdx.x & 31;

    // ---- which task does this lane belong to?  tasks of a warp occupy consecutive lane ranges
    const int t0 = p.warp_first[warp], nt = p.warp_first[warp + 1] - t0;
    ShortTask tk = {0, 0, 0, 0};
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
    int m_np = __shfl_sync(PHMM_FULL, tk.n_pairs, src), m_rows = __shfl_sync(PHMM_FULL, tk.rows, src);
    int m_k = __shfl_sync(PHMM_FULL, k, src);
    const int m_start = __shfl_sync(PHMM_FULL, start, src), m_g = __shfl_sync(PHMM_FULL, g, src);
    if (ti < 0) { m_np = 0; m_rows = 0; m_k = 0; }
    const int lg = ti < 0 ? 0 : lane - m_start;
    const bool is_first = (ti < 0) || lg == 0;
    const bool is_last = (ti >= 0) && lg == m_g - 1;

    // ---- number of steps of this warp: the last lane's .y half finishes the last entry of its stream
    int steps = (ti < 0) ? 0 : m_rows + m_np + 2 * m_g - 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) steps = max(steps, __shfl_xor_sync(PHMM_FULL, steps, o));

    L ln;
    ln.init();
    ln.load_hap(b.hap_bases + (ti < 0 ? 0 : b.hap_off[m_hap]), m_k, lg * N2);
    const float Cok = (float)(ldexp(1.0, 120) / (double)(m_k > 0 ? m_k : 1));  // Eq.1: C/k with C = 2^120

    // ---- stream cursor of the .x half (entry for step s is fetched during step s-1)
    const float4* tab = reinterpret_cast<const float4*>(p.table);
    Cursor<NV> c;
    c.cur = tab; c.nxt = tab; c.rem = 0; c.nxtRem = 0; c.q = 0; c.wait = 2 * lg;
    auto load_next = [&]() {
        if (c.q < m_np) {
            const int r = p.srt_read[m_first + c.q];
            c.q++;
            const int64_t o = b.read_off[r];
            c.nxt = tab + 2 * (o + r);
            c.nxtRem = (int)(b.read_off[r + 1] - o) + 1;
        } else {
            c.nxtRem = 0;
        }
    };
    load_next();
    float4 eA = make_float4(0.f, 0.f, 0.f, 0.f), eB = make_float4(0.f, 0.f, 0.f, 0.f);
    auto fetch = [&]() {
        eA = make_float4(0.f, 0.f, 0.f, 0.f);
        eB = make_float4(0.f, 0.f, 0.f, 0.f);
        if (c.wait > 0) {
            c.wait--;
        } else {
            if (c.rem == 0) { c.cur = c.nxt; c.rem = c.nxtRem; load_next(); }
            if (c.rem > 0) {
                eA = __ldg(c.cur);
                eB = __ldg(c.cur + 1);
                c.cur += 2;
                c.rem--;
            }
        }
    };
    fetch();

    int nout = 0;
    const double LOG10_2 = 0.30102999566398119521;
    for (int s = 0; s < steps; s++) {
        RowConst<float> E;
        E.a = eA.x; E.pm = eA.y; E.px = eA.z; E.c = eA.w;
        E.gi = eB.x; E.gI = eB.y; E.gm = eB.z; E.meta = (uint32_t)eB.w;
        fetch();  // prefetch the next step's entry
        float lM = __shfl_up_sync(PHMM_FULL, ln.outM(), 1);
        float lI = __shfl_up_sync(PHMM_FULL, ln.outI(), 1);
        float lS = __shfl_up_sync(PHMM_FULL, ln.outS(), 1);
        float lSig = __shfl_up_sync(PHMM_FULL, ln.outSig(), 1);
        if (is_first) { lM = 0.f; lI = 0.f; lSig = 0.f; lS = (E.meta & META_RESET) ? Cok : 0.f; }
        ln.step(E, lM, lI, lS, lSig);
        if (is_last && (ln.metaY & META_LAST)) {
            const float sg = ln.outSig();
            const int pair = p.srt_out[m_first + nout];
            nout++;
            if (isfinite(sg) && sg >= p.rescue_thr) {
                p.out[pair] = log10((double)sg) - 120.0 * LOG10_2;
                if (p.flags) p.flags[pair] = 0;
            } else {
                const int idx = atomicAdd(p.rescue_count, 1);
                p.rescue_list[idx] = pair;
            }
        }
    }
}

cudaError_t launch_short_f32(const DevBatch& b, const ShortLaunch& p, cudaStream_t st) {
    if (p.n_warps == 0) return cudaSuccess;
    const int grid = (p.n_warps + SHORT_WARPS_PER_CTA - 1) / SHORT_WARPS_PER_CTA;
    k_short_f32<SHORT_NV><<<grid, SHORT_WARPS_PER_CTA * 32, 0, st>>>(b, p);
    return cudaGetLastError();
}

}  // namespace phmm
