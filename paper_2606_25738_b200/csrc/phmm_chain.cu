// Rescaled fp64 path ("chain" kernel; the fp32 long path is phmm_long.cu, the PHMM_FP64 long path phmm_long64.cu, which took over
// this kernel's concurrent mode late in round 2: the library now launches it only in its sequential mode, as the last resort
// for pairs no other kernel could represent): one warp = one strip of 32 lanes x 2NV haplotype columns of
// one pair; the strips of a pair are chained left to right through boundary-column buffers in
// global memory (per stream entry: the running sum s and the T that drop out of the strip's last
// column, and the producing thread's block exponent), either concurrently (one strip per
// warp, progress counters; warps take strips in ticket order so a producer always holds an earlier
// ticket than its consumer => forward progress) or sequentially inside one warp (fp64 rescue of
// short pairs, PHMM_FP64 mode).
//
// a1 (row constants, computed on the fly into a shared-memory ring), a4,
// a5, a6/a7 (cross-warp / cross-CTA carry -- the paper's Eq.10/11 lock-step carries, PAPER.md:263-267,
// :319-324, become a skewed wavefront with 32-row handoff blocks), a8 (rescaling), a9, a10 (fp64 rescue).
//
// Rescaling (reading G15; absent from the paper).  Block floating point per THREAD: true value = stored
// value * 2^ex with one integer ex for everything a thread holds (the T/J state of its two halves, the
// values it hands to the right).  Eq.4 needs no sum of its own: on the sum entry behind the last row the running
// sum s collects M_l + I_l of every column (phmm_engine.cuh).  The lanes of a warp are 2 read rows apart, so
// a warp spans 64 rows and, along a row, 32 columns per lane: with unrelated sequence (3.3 bits lost
// per row or per deleted column) that is more than fp32's exponent range, hence no coarser unit.
// Every 16 steps a thread takes the maximum of what it holds and, if that left the window around
// 2^TGT, multiplies everything by the power of two that brings it back (exact, except that values
// more than the format's range below the thread maximum flush to zero: G15's documented limit).
// The two values crossing a lane (or strip) boundary per step come with the producer's ex and are
// converted by one exact multiply; if they would not fit, the consumer first moves its own exponent
// up.  The recurrence step itself is exactly the short kernel's (phmm_engine.cuh).
#include "phmm_engine.cuh"
#include "phmm_kernels.h"
#include "phmm_rowconst.cuh"

namespace phmm {

#ifndef CHAIN_HSETP2
#define CHAIN_HSETP2 1  // fp32: +1-2 %
#endif
#ifndef CHAIN_MIN_CTAS_F32
#define CHAIN_MIN_CTAS_F32 3  // 164 registers with HSETP2 predicates; since Eq.4 runs through the s chain this beats 4 CTAs x 128 registers
                              // (bit-test predicates: 2.17; HSETP2 with 15 spilled registers: 2.20; 3 CTAs: 2.26 TCUPS on configs[3] x0.5)
#endif
constexpr int RING = 128;  // row-constant ring per warp (entries); covers 63 entries of skew + two 32-entry blocks

template <typename T> struct Rec {  // boundary block of 32 stream entries, SoA
    T S[32], Tn[32];
    int ex[32];
};

// ---- ring entry format: NCH chunks of 16 bytes per entry, paired (.x = entry e, .y = entry e-1) like the
// short path's table; chunk planes of RING slots, the two parities of the slot index in separate halves of
// a plane so that lanes (which read entries two apart) hit consecutive 16-byte words: conflict-free LDS.128.
template <typename T> struct RingFmt;
template <> struct RingFmt<float> {
    static constexpr int NCH = 4;  // {gam.x gam.y A.x A.y} {C.x C.y G.x G.y} {pm.x px.x pm.y px.y} {meta.x meta.y - -}
    static constexpr int SPW = 4;  // scalars per 16-byte word
    static __device__ __forceinline__ int pair_at(int f, int half) { return (f >> 1) * 4 + (f & 1) * 2 + half; }  // f: 0 gam 1 A 2 C 3 G
    static __device__ __forceinline__ int prior_at(int which, int half) { return 2 * 4 + half * 2 + which; }     // which: 0 pm 1 px
    static __device__ __forceinline__ int meta_at(int half) { return 3 * 4 + half; }
    static __device__ __forceinline__ float meta_val(uint32_t m) { return __uint_as_float(m); }
    static __device__ __forceinline__ uint32_t meta_get(float v) { return __float_as_uint(v); }
};
template <> struct RingFmt<double> {
    static constexpr int NCH = 8;  // {gam} {A} {C} {G} {pm.x px.x} {pm.y px.y} {meta.x meta.y} {-}
    static constexpr int SPW = 2;
    static __device__ __forceinline__ int pair_at(int f, int half) { return f * 2 + half; }
    static __device__ __forceinline__ int prior_at(int which, int half) { return (4 + half) * 2 + which; }
    static __device__ __forceinline__ int meta_at(int half) { return 6 * 2 + half; }
    static __device__ __forceinline__ double meta_val(uint32_t m) { return __hiloint2double(0, (int)m); }
    static __device__ __forceinline__ uint32_t meta_get(double v) { return (uint32_t)__double2loint(v); }
};

template <typename T> struct Smem {
    T ring[RingFmt<T>::NCH * RING * RingFmt<T>::SPW];  // [chunk][parity][slot/2][scalars of the 16-byte word]
    Rec<T> rin, rout;
};

__device__ __forceinline__ int ring_word(int e) {  // index (in 16-byte words, within a chunk plane) of entry e
    const int sl = e & (RING - 1);
    return (sl & 1) * (RING / 2) + (sl >> 1);
}

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// v * 2^d, exact unless it leaves the format (d may exceed one factor's exponent range)
template <typename T> __device__ __forceinline__ T scale_pow2(T v, int d) {
    d = max(-Fx<T>::CLAMP, min(Fx<T>::CLAMP, d));
    const int h = d / 2;
    return v * Fx<T>::exp2i(h) * Fx<T>::exp2i(d - h);
}

template <typename T> struct Win;  // keep the thread maximum within 2^(TGT +- WIN); incoming values above 2^(TGT+UP) move ex first
template <> struct Win<float> { static constexpr int TGT = 60, WIN = 30, UP = 50; };
template <> struct Win<double> { static constexpr int TGT = 0, WIN = 400, UP = 600; };

template <typename T> __device__ __forceinline__ T warp_max(T m) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = Fx<T>::fmax_(m, __shfl_xor_sync(PHMM_FULL, m, o));
    return m;
}
__device__ __forceinline__ int warp_max_i(int m) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(PHMM_FULL, m, o));
    return m;
}

template <typename T, int NV, typename LN> __device__ __forceinline__ T lane_max(const LN& ln) {
    T m = Fx<T>::fmax_(Fx<T>::fmax_(ln.outS.x, ln.outS.y), Fx<T>::fmax_(ln.outT.x, ln.outT.y));
#pragma unroll
    for (int x = 0; x < NV; x++) {
        m = Fx<T>::fmax_(m, Fx<T>::fmax_(ln.Tt[x].x, ln.Tt[x].y));
        m = Fx<T>::fmax_(m, Fx<T>::fmax_(ln.J[x].x, ln.J[x].y));
    }
    return m;
}
template <typename T, int NV, typename LN> __device__ __forceinline__ void lane_scale(LN& ln, int d) {  // *= 2^d
    d = max(-Fx<T>::CLAMP, min(Fx<T>::CLAMP, d));
    const int h = d / 2;
    const T f1 = Fx<T>::exp2i(h), f2 = Fx<T>::exp2i(d - h);
    typedef W2<T> P;
    const typename P::V F1 = P::mk(f1, f1), F2 = P::mk(f2, f2);
#pragma unroll
    for (int x = 0; x < NV; x++) {
        ln.Tt[x] = P::mul(P::mul(ln.Tt[x], F1), F2);
        ln.J[x] = P::mul(P::mul(ln.J[x], F1), F2);
    }
    ln.outS = P::mul(P::mul(ln.outS, F1), F2);
    ln.outT = P::mul(P::mul(ln.outT, F1), F2);
}

template <typename T, int NV, int WPC, int MINB>
__global__ void __launch_bounds__(WPC * 32, MINB)
k_chain(DevBatch b, ChainLaunch p, int items_are_pairs) {
    typedef Lane2<T, NV, (CHAIN_HSETP2 != 0) && sizeof(T) == 4 && MINB == 3> L;  // HSETP2 only where the 12 extra registers do not spill
    typedef RingFmt<T> RF;
    typedef typename W2<T>::V V;
    constexpr int N2 = 2 * NV;
    __shared__ __align__(16) Smem<T> sm_all[WPC];
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gwarp = blockIdx.x * WPC + w;
    Smem<T>& sm = sm_all[w];
    T* rg = sm.ring;
    const V* rgv = reinterpret_cast<const V*>(sm.ring);  // fp32: 8-byte pairs; fp64: 16-byte pairs
    Rec<T>& RI = sm.rin;
    Rec<T>& RO = sm.rout;
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
        const int n_ent = l + CHAIN_EXTRA_ROWS;  // run-in entry, rows 1..l, sum entry, flush entry
        const int nstrips = (k + 32 * N2 - 1) / (32 * N2);
        // The lane that holds the haplotype's last column, in the last strip: Eq.4 is taken there; the lanes behind it hold only
        // padding columns and feed nothing.  (Until round 2 the sum travelled on to lane 31 through lanes that hold only padding columns; what
        // circulates there -- mismatch diagonals that never run out of columns -- can decay more slowly than the real cells,
        // where every further read base has to be an insertion, and the sum, converted from lane to lane to ever larger
        // exponents, vanished: -inf for a 535-base read against a 2-base haplotype at GCP 40.  Found by fuzzing.)
        const int k_last = k - (nstrips - 1) * 32 * N2;   // real columns of the last strip
        const int out_lane = (k_last - 1) / N2;
        const bool full_last = (k_last % N2) == 0;        // its last real column is the last column of that lane (see the output below)
        const int nblk = (n_ent + 31) / 32;  // boundary blocks per buffer
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
            // the step at which the .y half of the haplotype's last lane processes the sum entry (entry l + 1): e = s - 2 lane - 1
            const int out_step = (!has_out && lane == out_lane) ? l + 2 + 2 * lane : -1;

            L ln;
            ln.init();
            ln.load_hap(b.hap_bases + ho, k, (st * 32 + lane) * N2, b.n_wild != 0);
            int ex = 0;        // true value = stored value * 2^ex, one exponent per thread
            bool zero = true;  // this thread holds nothing but zeros
            __syncwarp();
            for (int i = lane; i < RF::NCH * RING * RF::SPW; i += 32) rg[i] = (T)0;
            __syncwarp();
            const int steps = n_ent + 63;
            for (int s = 0; s < steps; s++) {
                if ((s & 15) == 0) {
                    const bool blk = (s & 31) == 0;
                    if (blk) {
                        __syncwarp();
                        // ---- a1: constants of entries s..s+31, one per lane; .x fields to the entry's own slot,
                        //      .y fields to the next entry's slot (whose .y half runs one entry behind)
                        const int e = s + lane;
                        const RowC c = row_constants(b, p.lut, ro, l, e < n_ent ? e : -1, true);
                        T* lo = rg + ring_word(e) * RF::SPW;
                        T* hi = rg + ring_word(e + 1) * RF::SPW;
                        constexpr int PL = RING * RF::SPW;  // scalars per chunk plane
                        const double pr[4] = {c.gam, c.A, c.C, c.G};
#pragma unroll
                        for (int f = 0; f < 4; f++) {
                            const int a0 = RF::pair_at(f, 0), a1 = RF::pair_at(f, 1);
                            lo[(a0 / RF::SPW) * PL + a0 % RF::SPW] = (T)pr[f];
                            hi[(a1 / RF::SPW) * PL + a1 % RF::SPW] = (T)pr[f];
                        }
                        const double pq[2] = {c.pm, c.px};
#pragma unroll
                        for (int q = 0; q < 2; q++) {
                            const int a0 = RF::prior_at(q, 0), a1 = RF::prior_at(q, 1);
                            lo[(a0 / RF::SPW) * PL + a0 % RF::SPW] = (T)pq[q];
                            hi[(a1 / RF::SPW) * PL + a1 % RF::SPW] = (T)pq[q];
                        }
                        {
                            const int a0 = RF::meta_at(0), a1 = RF::meta_at(1);
                            lo[(a0 / RF::SPW) * PL + a0 % RF::SPW] = RF::meta_val(entry_word16(c));
                            hi[(a1 / RF::SPW) * PL + a1 % RF::SPW] = RF::meta_val(entry_word16(c));
                        }
                    }
                    // ---- incoming boundary block for entries s..s+31 (lane 0 consumes entry s at step s)
                    if (blk && has_in && s < n_ent) {
                        const int need = min(s + 32, n_ent);
                        if (inprog) {  // one lane polls; the others park at the barrier
                            // every lane polls: measured faster (2.02 vs 1.89 TCUPS) than one polling lane + __syncwarp
                            while (ld_acquire(inprog) < need) __nanosleep(64);
                        }
                        const Rec<T>* src = inb + (s >> 5);
                        RI.S[lane] = src->S[lane]; RI.Tn[lane] = src->Tn[lane];
                        RI.ex[lane] = src->ex[lane];
                    }
                    // ---- a8: block-floating event of this thread
                    const T m = lane_max<T, NV>(ln);
                    if (m > (T)0) {
                        const int e = Fx<T>::ilogb(m);
                        if (e > Win<T>::TGT + Win<T>::WIN || e < Win<T>::TGT - Win<T>::WIN) {
                            lane_scale<T, NV>(ln, Win<T>::TGT - e);
                            ex += e - Win<T>::TGT;
                        }
                        zero = false;
                    } else {
                        zero = true;  // nothing held: the exponent is free, adopt the next incoming one
                    }
                    __syncwarp();
                }
                // ---- this lane's entry: .x half at stream position s - 2 lane, .y half one behind (same ring slot)
                Entry2<T> E;
                {
                    const int wd = ring_word(s - 2 * lane);
                    constexpr int VPW = 16 / sizeof(V);  // pairs per 16-byte word: 2 (fp32) or 1 (fp64)
                    constexpr int PLV = RING * VPW;       // pairs per chunk plane
                    const V* q = rgv + wd * VPW;
                    if (sizeof(T) == 4) {
                        E.gam = q[0]; E.A = q[1]; E.C = q[PLV]; E.G = q[PLV + 1];
                        const V pa = q[2 * PLV], pb = q[2 * PLV + 1], mm = q[3 * PLV];
                        E.pmx = pa.x; E.pxx = pa.y; E.pmy = pb.x; E.pxy = pb.y;
                        E.metaX = RF::meta_get(mm.x); E.metaY = RF::meta_get(mm.y);
                    } else {
                        E.gam = q[0]; E.A = q[PLV]; E.C = q[2 * PLV]; E.G = q[3 * PLV];
                        const V pa = q[4 * PLV], pb = q[5 * PLV], mm = q[6 * PLV];
                        E.pmx = pa.x; E.pxx = pa.y; E.pmy = pb.x; E.pxy = pb.y;
                        E.metaX = RF::meta_get(mm.x); E.metaY = RF::meta_get(mm.y);
                    }
                    E.r2 = (E.metaX & 0xff00u) | ((E.metaY & 0xff00u) << 16);
                }
                // ---- left boundary: neighbour lane (shuffle), first strip (Eq.1 injection) or boundary block
                T inS = shfl_up1<T>(ln.outS.y), inT = shfl_up1<T>(ln.outT.y);
                int exL = __shfl_up_sync(PHMM_FULL, ex, 1);
                if (lane == 0) {
                    if (has_in) {
                        const int q = s & 31;
                        const bool ok = s < n_ent;
                        inS = ok ? RI.S[q] : (T)0; inT = ok ? RI.Tn[q] : (T)0;
                        exL = ok ? RI.ex[q] : ex;
                    } else {
                        const bool f = (E.metaX & META_FIRST) != 0;  // Eq.1: only the run-in entry injects, at exponent 0
                        inS = f ? Cok : (T)0;
                        inT = f ? E.C.x * Cok : (T)0;
                        exL = 0;
                    }
                }
                // ---- bring the incoming values to this thread's exponent (exact power-of-two multiply)
                {
                    const T mi = Fx<T>::fmax_(inS, inT);
                    if (zero) {
                        if (mi > (T)0) { ex = exL; zero = false; }
                    } else if (mi > (T)0 && Fx<T>::ilogb(mi) + exL - ex > Win<T>::TGT + Win<T>::UP) {
                        const int up = Fx<T>::ilogb(mi) + exL - ex - Win<T>::TGT;  // they would not fit: move this thread up first
                        lane_scale<T, NV>(ln, -up);
                        ex += up;
                    }
                    const int d = exL - ex;
                    if (d >= -Fx<T>::CLAMP1 && d <= Fx<T>::CLAMP1) {  // the usual case: one exact factor
                        const T f = Fx<T>::exp2i(d);
                        inS *= f; inT *= f;
                    } else {  // |d| beyond one factor's exponent range
                        inS = scale_pow2<T>(inS, d); inT = scale_pow2<T>(inT, d);
                    }
                }
                const T prevT = ln.outT.y;  // at this thread's current exponent (every rescaling of this step is done)
                ln.step(E, inS, inT);
                // ---- right boundary of the strip: lane 31's .y half has just finished entry s - 63
                const int eo = s - 63;
                if (eo >= 0 && eo < n_ent) {
                    if (has_out) {
                        if (lane == 31) {
                            const int q = eo & 31;
                            RO.S[q] = ln.outS.y; RO.Tn[q] = ln.outT.y; RO.ex[q] = ex;
                        }
                        if ((eo & 31) == 31 || eo == n_ent - 1) {
                            __syncwarp();
                            Rec<T>* dst = outb + (eo >> 5);
                            dst->S[lane] = RO.S[lane]; dst->Tn[lane] = RO.Tn[lane];
                            dst->ex[lane] = RO.ex[lane];
                            __syncwarp();
                            if (outprog && lane == 0) {
                                __threadfence();
                                st_release(outprog, eo + 1);
                            }
                            __syncwarp();
                        }
                    }
                }
                if (s == out_step) {  // this lane's .y half has just done the sum entry: s has collected Eq.4; log10 in double
                    // M+I of column j reaches the chain through the T of column j+1; a haplotype that fills its last
                    // lane has the last one in what this lane handed out one step ago instead
                    const T sum = full_last ? ln.outS.y + prevT : ln.outS.y;
                    p.out[pair] = log10((double)sum) + ((double)ex - (double)p.log2C) * LOG10_2;
                    if (p.flags) p.flags[pair] = p.flag_bits | ((items_are_pairs && long_class(k, l, p.long_k, p.tall_k)) ? 2u /* PHMM_FLAG_LONG */ : 0u);
                }
            }
            __syncwarp();
        }
    }
}

// One-warp CTAs, twelve per SM (164 registers, no spills): the kernel waits on fp64 dependencies, and 12 warps per SM against
// the 8 of two-warp CTAs at 192 registers are +22 % (0.85 -> 1.04 TCUPS, configs[3] x 0.25 in PHMM_FP64).  24 or 32 columns
// per lane at 8 warps per SM measure the same; 20 columns at 12 warps spill and lose 3 %.
#ifndef CHAIN_WPC_F64
#define CHAIN_WPC_F64 1
#endif
#ifndef CHAIN_MINB_F64
#define CHAIN_MINB_F64 12
#endif
constexpr int WPC_F64 = CHAIN_WPC_F64, MINB_F64 = CHAIN_MINB_F64;

cudaError_t launch_chain(const DevBatch& b, const ChainLaunch& p, bool fp64, bool items_are_pairs, int grid_ctas, cudaStream_t st) {
    if (grid_ctas <= 0) return cudaSuccess;
    if (!fp64) return cudaErrorInvalidValue;  // the fp32 long path is phmm_long.cu
    k_chain<double, CHAIN_NV_F64, WPC_F64, MINB_F64><<<grid_ctas, WPC_F64 * 32, 0, st>>>(b, p, items_are_pairs ? 1 : 0);
    return cudaGetLastError();
}

int chain_ctas_per_sm(bool) {
    int n = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_chain<double, CHAIN_NV_F64, WPC_F64, MINB_F64>, WPC_F64 * 32, 0);
    return n > 0 ? n : 1;
}
int chain_warps_per_cta(bool) { return WPC_F64; }
size_t chain_block_bytes(bool) { return sizeof(Rec<double>); }
int chain_strip_cols(bool fp64) { return fp64 ? 32 * 2 * CHAIN_NV_F64 : SHORT_MAX_K; }

}  // namespace phmm
