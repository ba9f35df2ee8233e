// The per-lane engine of the skewed systolic wavefront ("T/J form").
//
// One CUDA thread = two "virtual lanes" held in the two halves of float2 values (FFMA2/FMUL2 on
// sm_100a; two scalars per operation in fp64): half .x owns NV consecutive haplotype columns, half .y
// the next NV columns and runs ONE stream entry (read row) behind .x; the next CUDA lane's .x runs
// one further entry behind, and so on.  With that skew everything a virtual lane needs from its left
// neighbour is already final when it is needed, so no scan is required (the paper's lock-step kernels
// need the weighted warp scan of Alg.1, plus a second running sum V, Listing 2
// :309 = 7 FP instructions per cell; this engine needs 5).
//
// Recurrence (phmm_common.cuh: M, I' = g_{i+1} I, S = weighted inclusive prefix of M, Eq.6-7 with
// every constant folded per read row).  State a virtual lane keeps for its columns x between two
// steps, when the next entry it will process is read row i:
//     T[x] = a_i M_{i-1,x-1} + I'_{i-1,x-1} + c_i S_{i-1,x-2}     everything of M_{i,x} but the prior
//     J[x] = I'_{i,x}                                              (already advanced to row i)
// One step = one row for all NV columns; per column, with U := gi_{i+1} M_{i,x} kept instead of M:
//     U      = P_{i,x} * T[x]                    P = (pm_i | px_i) * gi_{i+1}, one select (Eq.3)   MUL
//     W      = A * U + J[x]                      A = a_{i+1} / gi_{i+1}                            FMA
//     T[x+1] = C * s + W                         C = c_{i+1} / gi_{i+1};  s = gi_{i+1} S_{i,x-1}   FMA
//     J[x]   = G * J[x] + U                      G = gamma_{i+1} g_{i+2} / g_{i+1}                 FMA
//     s      = gamma_i * s + U                   the row's running sum, the only serial chain       FMA
// = 5 FP instructions per cell (4 FMA + 1 MUL, 9 flops); U, W are temporaries, T and J are updated in
// place.  What crosses a virtual-lane boundary: the T[NV] that drops out on the right (consumed by
// the neighbour two steps later = when it processes the next row) and the final s (consumed by the
// neighbour's next step = the same row).  See the row-constant table kernel for the stream of
// entries (run-in entry, rows 1..l, sum entry, flush entry) and how Eq.1 and Eq.4 are realised.
#pragma once
#include "phmm_common.cuh"

namespace phmm {

// ---- two-wide arithmetic: float2 -> FFMA2/FMUL2/FADD2 (sm_100a), double2 -> two scalar ops
template <typename T> struct W2;
template <> struct W2<float> {
    typedef float2 V;
    static __device__ __forceinline__ V mk(float x, float y) { return make_float2(x, y); }
    static __device__ __forceinline__ V fma(V a, V b, V c) { return __ffma2_rn(a, b, c); }
    static __device__ __forceinline__ V mul(V a, V b) { return __fmul2_rn(a, b); }
    static __device__ __forceinline__ V add(V a, V b) { return __fadd2_rn(a, b); }
};
template <> struct W2<double> {
    typedef double2 V;
    static __device__ __forceinline__ V mk(double x, double y) { return make_double2(x, y); }
    static __device__ __forceinline__ V fma(V a, V b, V c) { return make_double2(::fma(a.x, b.x, c.x), ::fma(a.y, b.y, c.y)); }
    static __device__ __forceinline__ V mul(V a, V b) { return make_double2(a.x * b.x, a.y * b.y); }
    static __device__ __forceinline__ V add(V a, V b) { return make_double2(a.x + b.x, a.y + b.y); }
};

// One table entry as the kernel sees it: constants of the entry the .x half processes (lo) and of the
// stream's previous entry, which the .y half processes in the same step (hi).
template <typename T> struct Entry2 {
    typename W2<T>::V gam, A, C, G;
    T pmx, pxx, pmy, pxy;
    uint32_t metaX, metaY;
    uint32_t r2;  // HS: the fp16 base codes of (.x's row, .y's row), as the table / ring stores them (entry_word16)
};

// HS (fp32 only): take the Eq.3 predicates of both halves from one HSETP2 on per-column fp16 base codes instead
// of two bit tests of the match word: 16 fewer ALU instructions per step, 12 more registers.
// Eq.4 comes out of the running sum s instead of a per-lane summation of J.  The stream then carries a
// "sum entry" behind the last row (phmm_rowconst.cuh): the last row leaves T[x+1] = M_{l,x} + I_{l,x} (A := 1, C := 0),
// and the sum entry has gamma := 1, pm := 0, px := 1 and base code 0, so that U = T on every column that does not
// "match" it and the chain s = s + U adds them up across the whole lane group.  What matches the sum entry: the columns
// behind the haplotype EXCEPT the first one, which holds T = (M+I) of the last real column.  With HS those carry code
// 0, the first one code 5 and a haplotype 'N' code 6 (= a read N's code; 5 matches no read base); without HS a sixth match
// word, hm[5], marks them (hm[4] is the word of N).  No divergent per-lane summation, no third value handed from lane to lane.
template <typename T, int NV, bool HS = false> struct Lane2 {
    typedef W2<T> P;
    typedef typename P::V V;
    static_assert(NV <= 16, "one 32-bit match word per base: 16 columns per half");

    V Tt[NV], J[NV];
    V outT, outS;              // what dropped out on the right in the last step: (.x's, .y's)
    uint32_t hm[HS ? 1 : 6];   // without HS: match words, one per base b: bit x <=> .x column x is b, bit 16+x <=> .y column x is b
    uint32_t h2[HS ? NV : 1];  // HS: per column the base codes of (.x, .y) as two fp16 numbers (1..4; 5, 6, 0: see above)

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int x = 0; x < NV; x++) { Tt[x] = P::mk((T)0, (T)0); J[x] = P::mk((T)0, (T)0); }
        outT = outS = P::mk((T)0, (T)0);
    }

    // hap: pointer to the haplotype bytes, k its length, j0 = 0-based first column of this thread
    // wild (match words only; the fp16 codes of HS cannot express it): a haplotype N matches every read base
    __device__ __forceinline__ void load_hap(const uint8_t* __restrict__ hap, int k, int j0, bool wild = false) {
        if constexpr (HS) {
#pragma unroll
            for (int x = 0; x < NV; x++) {
                const int jx = j0 + x, jy = j0 + NV + x;
                const uint32_t cx = jx < k ? col_code(hap[jx]) : (jx == k ? 0x4500u : 0u);
                const uint32_t cy = jy < k ? col_code(hap[jy]) : (jy == k ? 0x4500u : 0u);
                h2[x] = cx | (cy << 16);
            }
        } else {
#pragma unroll
            for (int c = 0; c < 5; c++) hm[c] = 0;
            const int nvx = min(max(k - j0, 0), NV), nvy = min(max(k - j0 - NV, 0), NV);  // real columns of each half
#pragma unroll
            for (int x = 0; x < NV; x++) {
                if (x < nvx) {
                    const int c = base_code(hap[j0 + x]);
#pragma unroll
                    for (int q = 0; q < 5; q++) hm[q] |= ((c == q || (wild && c == 4)) ? 1u : 0u) << x;
                }
                if (x < nvy) {
                    const int c = base_code(hap[j0 + NV + x]);
#pragma unroll
                    for (int q = 0; q < 5; q++) hm[q] |= ((c == q || (wild && c == 4)) ? 1u : 0u) << (16 + x);
                }
            }
            uint32_t v = 0;  // what "matches" the sum entry: columns more than one behind the haplotype's last
#pragma unroll
            for (int x = 0; x < NV; x++) {
                if (j0 + x > k) v |= 1u << x;
                if (j0 + NV + x > k) v |= 1u << (16 + x);
            }
            hm[5] = v;
        }
    }
    static __device__ __forceinline__ uint32_t half_code(int c) {  // fp16 bit pattern of the number c + 1
        return (uint32_t)((0x4400420040003C00ull >> (16 * c)) & 0xffffull);
    }
    static __device__ __forceinline__ uint32_t col_code(uint8_t b) {  // fp16 1..4 for A,C,G,T; 6 for anything else
        const int c = base_code(b);
        return c < 4 ? half_code(c) : 0x4600u;
    }

    // One systolic step.  (inS, inT): the left neighbour thread's (.y) outS, outT as they stand
    // after ITS last step, or the column-0 boundary for the first lane of a group (Eq.1 under reading G1:
    // the run-in entry injects s = C/k and T = g_1 C/k, every other entry 0).
    __device__ __forceinline__ void step(const Entry2<T>& E, T inS, T inT) {
        V s = P::mk(inS, outS.x);                  // .y continues the row .x finished one step ago
        const V tgrab = P::mk(inT, outT.x);        // T[0] of the NEXT step
        // match word of this step: the read base of .x's row picks the low half, that of .y's row the high half;
        // consecutive single-bit tests of one register let ptxas turn 7 of them into one R2P
        uint32_t mw = 0;
        if constexpr (!HS) {
            const uint32_t wx01 = (E.metaX & 1u) ? hm[1] : hm[0], wx23 = (E.metaX & 1u) ? hm[3] : hm[2];
            const uint32_t wy01 = (E.metaY & 1u) ? hm[1] : hm[0], wy23 = (E.metaY & 1u) ? hm[3] : hm[2];
            uint32_t wx = (E.metaX & 2u) ? wx23 : wx01, wy = (E.metaY & 2u) ? wy23 : wy01;
            wx = (E.metaX & 4u) ? hm[4] : wx;  // an N row
            wy = (E.metaY & 4u) ? hm[4] : wy;
            wx = (E.metaX & META_SUM) ? hm[5] : wx;  // (the other entries that are no read rows have pm = px = 0)
            wy = (E.metaY & META_SUM) ? hm[5] : wy;
            mw = (wx & 0xffffu) | (wy & 0xffff0000u);
        }
        const uint32_t r2 = E.r2;
        auto prior = [&](int x) {                  // Eq.3: one select per half
            if constexpr (HS && sizeof(T) == 4) {  // one HSETP2 yields both halves' predicates
                float a, b;
                asm("{.reg .pred p, q;\n setp.eq.f16x2 p|q, %2, %3;\n selp.f32 %0, %4, %5, p;\n selp.f32 %1, %6, %7, q;}"
                    : "=f"(a), "=f"(b) : "r"(h2[x]), "r"(r2), "f"((float)E.pmx), "f"((float)E.pxx), "f"((float)E.pmy), "f"((float)E.pxy));
                return P::mk((T)a, (T)b);
            }
            return P::mk((mw & (1u << x)) ? E.pmx : E.pxx, (mw & (1u << (16 + x))) ? E.pmy : E.pxy);
        };
        V U = P::mul(prior(0), Tt[0]);
        Tt[0] = tgrab;
#pragma unroll
        for (int x = 0; x < NV; x++) {
            V Un = U;
            if (x + 1 < NV) Un = P::mul(prior(x + 1), Tt[x + 1]);
            const V Wv = P::fma(E.A, U, J[x]);
            const V Tn = P::fma(E.C, s, Wv);
            J[x] = P::fma(E.G, J[x], U);
            s = P::fma(E.gam, s, U);
            if (x + 1 < NV) Tt[x + 1] = Tn; else outT = Tn;
            U = Un;
        }
        outS = s;
        // Eq.4 is the s that leaves the group's last lane on the sum entry: nothing to do here
    }
};

}  // namespace phmm
