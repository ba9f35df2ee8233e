// Generic rescaled path ("chain" kernel): one warp = one strip of 32 lanes x 2NV haplotype columns of
// one pair; the strips of a pair are chained left to right through boundary-column buffers in
// global memory (the last column's M, I', S, running final sum and block exponent for every read
// row), either concurrently (one strip per warp, progress counters; warps take strips in ticket
// order so a producer always holds an earlier ticket than its consumer => forward progress) or
// sequentially inside one warp (rescue of short pairs, fp64 mode).
//
// a1 (row constants, computed on the fly into a shared-memory ring), a4,
// a5, a6/a7 (cross-warp / cross-CTA carry -- the paper's Eq.10/11 lock-step carries, PAPER.md:263-267,
// :319-324, become a skewed wavefront with 32-row handoff blocks), a8 (rescaling), a9, a10 (fp64 rescue).
// Block-floating arithmetic: every thread keeps one integer exponent for all it holds; values
// crossing a thread boundary are converted exactly by a power of two.
#include "phmm_engine_v0.cuh"
#include "phmm_kernels.h"

namespace phmm {

constexpr int CHAIN_WARPS = 4;
constexpr int RING = 128;  // row-constant ring per warp (entries); must cover 62 rows of skew + two 32-row blocks

template <typename T> struct Rec {  // boundary block of 32 entries, SoA
    T M[32], I[32], S[32], Sig[32];
    int ex[32];
};

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

template <typename T, int NV>
__global__ void __launch_bounds__(CHAIN_WARPS * 32, (sizeof(T) == 4 ? 2 : 2))
k_chain(DevBatch b, ChainLaunch p, int items_are_pairs) {
    typedef LaneV0<T, NV, true> L;
    constexpr int N2 = 2 * NV;
    __shared__ T ring[CHAIN_WARPS][8][RING];        // row constants, SoA: [field][slot]
    __shared__ Rec<T> rin[CHAIN_WARPS], rout[CHAIN_WARPS];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gwarp = blockIdx.x * CHAIN_WARPS + w;
    T(*rg)[RING] = ring[w];
    Rec<T>& RI = rin[w];
    Rec<T>& RO = rout[w];
    const double LOG10_2 = 0.30102999566398119521;
    const int n_items = *p.n_items;

    for (;;) {
        int ticket = 0;
        if (lane == 0) ticket = atomicAdd(p.ticket, 1);
        ticket = __shfl_sync(PHMM_FULL, ticket, 0);
        if (ticket >= n_items) break;
        int pair, strip, prog0 = 0;
        int64_t buf0 = 0;
        if (items_are_pairs) {
            pair = reinterpret_cast<const int*>(p.items)[ticket];
            strip = -1;
        } else {
            ChainItem it = p.items[ticket];
            pair = it.pair; strip = it.strip; prog0 = it.prog0; buf0 = it.buf0;
        }
        const int r = p.pair_read[pair], h = p.pair_hap[pair];
        const int64_t ro = b.read_off[r], ho = b.hap_off[h];
        const int l = (int)(b.read_off[r + 1] - ro), k = (int)(b.hap_off[h + 1] - ho);
        const int nstrips = (k + 32 * N2 - 1) / (32 * N2);
        const int nblk = (l + 1 + 31) / 32;  // boundary blocks per buffer
        const int st_lo = strip < 0 ? 0 : strip, st_hi = strip < 0 ? nstrips : strip + 1;
        const T Cok = (T)(ldexp(1.0, p.log2C) / (double)k);
        Rec<T>* bufbase = reinterpret_cast<Rec<T>*>(p.boundary);

        for (int st = st_lo; st < st_hi; st++) {
            const Rec<T>* inb = nullptr;
            Rec<T>* outb = nullptr;
            const int* inprog = nullptr;
            int* outprog = nullptr;
            if (strip < 0) {  // sequential: ping-pong in this warp's scratch
                Rec<T>* mine = bufbase + (int64_t)gwarp * 2 * p.scratch_blocks;
                inb = mine + (int64_t)(st & 1) * p.scratch_blocks;
                outb = mine + (int64_t)((st + 1) & 1) * p.scratch_blocks;
            } else {
                inb = bufbase + buf0 + (int64_t)(st - 1) * nblk;
                outb = bufbase + buf0 + (int64_t)st * nblk;
                inprog = p.progress + prog0 + st - 1;
                outprog = p.progress + prog0 + st;
            }
            const bool has_in = st > 0, has_out = st + 1 < nstrips;

            L ln;
            ln.init();
            ln.load_hap(b.hap_bases + ho, k, (st * 32 + lane) * N2);
            const int steps = l + 64;
            for (int s = 0; s < steps; s++) {
                if ((s & 31) == 0) {
                    __syncwarp();
                    // ---- a1: constants of entries s..s+31 (entry 0 = reset row), one per lane
                    const int e = s + lane;
                    if (e <= l) {
                        T c0 = 0, c1 = 0, c2 = 0, c3 = 0, c4 = 0, c5 = 0, c6 = 1;
                        uint32_t meta = META_RESET;
                        if (e > 0) {
                            const double eps = p.lut[b.qual_base[ro + e - 1]], io = p.lut[b.qual_ins[ro + e - 1]];
                            const double de = p.lut[b.qual_del[ro + e - 1]], ga = p.lut[b.qual_gcp[ro + e - 1]];
                            const double g = 1.0 - ga;
                            const double gn = (e < l) ? 1.0 - p.lut[b.qual_gcp[ro + e]] : 1.0;
                            const double dp = (e > 1) ? p.lut[b.qual_del[ro + e - 2]] : 1.0;
                            meta = (uint32_t)base_code(b.read_bases[ro + e - 1]) | (e == l ? META_LAST : 0u);
                            c0 = (T)(1.0 - io - de); c1 = (T)(1.0 - eps); c2 = (T)(eps / 3.0); c3 = (T)(g * dp);
                            c4 = (T)(gn * io); c5 = (T)(ga * gn / g); c6 = (T)ga;
                        }
                        const int sl = e & (RING - 1);
                        rg[0][sl] = c0; rg[1][sl] = c1; rg[2][sl] = c2; rg[3][sl] = c3;
                        rg[4][sl] = c4; rg[5][sl] = c5; rg[6][sl] = c6; rg[7][sl] = (T)meta;
                    }
                    // ---- incoming boundary block for entries s..s+31 (lane 0 consumes entry s at step s)
                    if (has_in && s <= l) {
                        const int need = min(s + 32, l + 1);
                        if (inprog) {
                            while (ld_acquire(inprog) < need) __nanosleep(64);
                        }
                        const Rec<T>* src = inb + (s >> 5);
                        RI.M[lane] = src->M[lane]; RI.I[lane] = src->I[lane]; RI.S[lane] = src->S[lane];
                        RI.Sig[lane] = src->Sig[lane]; RI.ex[lane] = src->ex[lane];
                    }
                    __syncwarp();
                }
                // ---- this lane's row constants
                const int pos = s - 2 * lane;
                RowConstV0<T> E;
                E.a = E.pm = E.px = E.c = E.gi = E.gI = E.gm = (T)0;
                E.meta = 0;
                if (pos >= 0 && pos <= l) {
                    const int sl = pos & (RING - 1);
                    E.a = rg[0][sl]; E.pm = rg[1][sl]; E.px = rg[2][sl]; E.c = rg[3][sl];
                    E.gi = rg[4][sl]; E.gI = rg[5][sl]; E.gm = rg[6][sl]; E.meta = (uint32_t)rg[7][sl];
                }
                // ---- left boundary: neighbour lane (shuffle), first strip (Eq.1 injection) or buffer
                T lM = shfl_up1<T>(ln.outM()), lI = shfl_up1<T>(ln.outI()), lS = shfl_up1<T>(ln.outS());
                T lSig = shfl_up1<T>(ln.outSig());
                int exL = __shfl_up_sync(PHMM_FULL, ln.ex, 1);
                if (lane == 0) {
                    if (has_in && s <= l) {
                        const int q = s & 31;
                        lM = RI.M[q]; lI = RI.I[q]; lS = RI.S[q]; lSig = RI.Sig[q]; exL = RI.ex[q];
                    } else {
                        lM = (T)0; lI = (T)0; lSig = (T)0; exL = 0;
                        lS = (!has_in && s == 0) ? Cok : (T)0;
                    }
                }
                ln.absorb(lM, lI, lS, lSig, exL);
                ln.step(E, lM, lI, lS, lSig);
                if ((s & 15) == 15) ln.periodic();
                // ---- right boundary of the strip: lane 31's .y half finished entry s-63
                const int eo = s - 63;
                if (eo >= 0) {
                    if (has_out) {
                        if (lane == 31) {
                            const int q = eo & 31;
                            RO.M[q] = ln.outM(); RO.I[q] = ln.outI(); RO.S[q] = ln.outS(); RO.Sig[q] = ln.outSig();
                            RO.ex[q] = ln.ex;
                        }
                        if ((eo & 31) == 31 || eo == l) {
                            __syncwarp();
                            Rec<T>* dst = outb + (eo >> 5);
                            dst->M[lane] = RO.M[lane]; dst->I[lane] = RO.I[lane]; dst->S[lane] = RO.S[lane];
                            dst->Sig[lane] = RO.Sig[lane]; dst->ex[lane] = RO.ex[lane];
                            __syncwarp();
                            if (outprog && lane == 0) {
                                __threadfence();
                                st_release(outprog, eo + 1);
                            }
                            __syncwarp();
                        }
                    } else if (eo == l && lane == 31) {
                        const T sg = ln.outSig();
                        p.out[pair] = log10((double)sg) + ((double)ln.ex - (double)p.log2C) * LOG10_2;
                        if (p.flags) p.flags[pair] = p.flag_bits;
                    }
                }
            }
            __syncwarp();
        }
    }
}

static int g_chain_grid = 0;

cudaError_t launch_chain(const DevBatch& b, const ChainLaunch& p, bool fp64, bool items_are_pairs, int grid_ctas,
                         cudaStream_t st) {
    if (grid_ctas <= 0) return cudaSuccess;
    if (fp64)
        k_chain<double, CHAIN_NV_F64><<<grid_ctas, CHAIN_WARPS * 32, 0, st>>>(b, p, items_are_pairs ? 1 : 0);
    else
        k_chain<float, CHAIN_NV_F32><<<grid_ctas, CHAIN_WARPS * 32, 0, st>>>(b, p, items_are_pairs ? 1 : 0);
    (void)g_chain_grid;
    return cudaGetLastError();
}

int chain_ctas_per_sm(bool fp64) {
    int n = 0;
    if (fp64)
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_chain<double, CHAIN_NV_F64>, CHAIN_WARPS * 32, 0);
    else
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_chain<float, CHAIN_NV_F32>, CHAIN_WARPS * 32, 0);
    return n > 0 ? n : 1;
}
int chain_warps_per_cta() { return CHAIN_WARPS; }
size_t chain_block_bytes(bool fp64) { return fp64 ? sizeof(Rec<double>) : sizeof(Rec<float>); }
int chain_strip_cols(bool fp64) { return 32 * 2 * (fp64 ? CHAIN_NV_F64 : CHAIN_NV_F32); }

}  // namespace phmm
