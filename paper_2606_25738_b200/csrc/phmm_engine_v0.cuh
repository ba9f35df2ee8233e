// The per-lane engine of the skewed systolic wavefront.
//
// One CUDA thread = two "virtual lanes" packed in the two halves of 64-bit register pairs (FFMA2 on
// sm_100a): half .x owns NV consecutive haplotype columns, half .y the next NV columns and runs ONE
// read row behind .x; the next CUDA lane's .x runs one further row behind, and so on.  With that
// skew the left neighbour's last-column values (M, I', S) of a row are exact when they are needed,
// so no scan is required (the paper's lock-step kernels need the weighted warp scan of Alg.1,
// PAPER.md:221-231, plus a second running sum V, Listing 2 :309).  See phmm_common.cuh for the
// recurrence; DESIGN.md "Kernel design" for the derivation.
#pragma once
#include "phmm_common.cuh"

namespace phmm {

template <typename T> struct RowConstV0 {  // one table entry, as loaded for the .x half
    T a, pm, px, c, gi, gI, gm;
    uint32_t meta;
};

template <typename T, int NV, bool RESCALE> struct LaneV0 {
    typedef Pk<T> P;
    typedef typename P::V V;

    V M[NV], I[NV], S[NV];               // state of the rows last completed by (.x, .y); S[x] = prefix EXCLUSIVE of column x
    V cA, cPm, cPx, cC, cGi, cGI, cGm;   // row constants (.x: its current row, .y: .x's previous row)
    V inM, inI, inS;                     // left-boundary values of the rows processed in the last step
    V sig;                               // running final sums handed to the right
    uint32_t metaX, metaY;
    uint32_t mx[5], my[5];               // match bitmasks per base code for the NV columns of .x / .y
    int nvx, nvy;                        // number of real (j <= k) columns in each half
    int ex;                              // RESCALE: stored value * 2^ex = true value (one exponent per thread)

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int x = 0; x < NV; x++) { M[x] = P::zero(); I[x] = P::zero(); S[x] = P::zero(); }
        cA = cPm = cPx = cC = cGi = cGI = cGm = P::zero();
        inM = inI = inS = P::zero();
        sig = P::zero();
        metaX = metaY = 0;
        ex = EX_ZERO;
    }

    // hap: pointer to the haplotype bytes, k its length, j0 = 0-based first column of this thread
    __device__ __forceinline__ void load_hap(const uint8_t* __restrict__ hap, int k, int j0) {
#pragma unroll
        for (int b = 0; b < 5; b++) { mx[b] = 0; my[b] = 0; }
        nvx = min(max(k - j0, 0), NV);
        nvy = min(max(k - j0 - NV, 0), NV);
#pragma unroll
        for (int x = 0; x < NV; x++) {
            if (x < nvx) {
                int c = base_code(hap[j0 + x]);
#pragma unroll
                for (int b = 0; b < 5; b++) mx[b] |= (c == b ? 1u : 0u) << x;
            }
            if (x < nvy) {
                int c = base_code(hap[j0 + NV + x]);
#pragma unroll
                for (int b = 0; b < 5; b++) my[b] |= (c == b ? 1u : 0u) << x;
            }
        }
    }

    static __device__ __forceinline__ uint32_t selmask(const uint32_t* m, uint32_t code) {
        uint32_t r = (code & 1u) ? m[1] : m[0];
        uint32_t q = (code & 1u) ? m[3] : m[2];
        r = (code & 2u) ? q : r;
        return (code & 4u) ? m[4] : r;
    }

    // multiply everything this thread holds by 2^-shift, adjust the exponent (exact unless it flushes)
    __device__ __forceinline__ void rescale(int shift) {
        int s = max(-Fx<T>::CLAMP, min(Fx<T>::CLAMP, shift));
        int h = (-s) / 2;
        T f1 = Fx<T>::exp2i(h), f2 = Fx<T>::exp2i(-s - h);
        V F1 = P::pack(f1, f1), F2 = P::pack(f2, f2);
#pragma unroll
        for (int x = 0; x < NV; x++) {
            M[x] = P::mul(P::mul(M[x], F1), F2);
            I[x] = P::mul(P::mul(I[x], F1), F2);
            S[x] = P::mul(P::mul(S[x], F1), F2);
        }
        inM = P::mul(P::mul(inM, F1), F2);
        inI = P::mul(P::mul(inI, F1), F2);
        inS = P::mul(P::mul(inS, F1), F2);
        sig = P::mul(P::mul(sig, F1), F2);
        ex += shift;
    }

    // RESCALE: bring the values (lM, lI, lS, lSig), given at exponent exL, to this thread's exponent;
    // if they would be too large for it, first move this thread's exponent up (its own state can only
    // be negligible then, or still representable).
    __device__ __forceinline__ void absorb(T& lM, T& lI, T& lS, T& lSig, int exL) {
        T m = Fx<T>::fmax_(Fx<T>::fmax_(lM, lI), Fx<T>::fmax_(lS, lSig));
        if (m > (T)0) {
            if (ex == EX_ZERO) ex = exL + Fx<T>::ilogb(m) - Fx<T>::TGT;
            int d = exL - ex;
            int e_in = Fx<T>::ilogb(m) + d;
            if (e_in > Fx<T>::HI) { rescale(e_in - Fx<T>::TGT); d = exL - ex; }
            d = max(-Fx<T>::CLAMP, min(Fx<T>::CLAMP, d));
            int h = d / 2;
            T f1 = Fx<T>::exp2i(h), f2 = Fx<T>::exp2i(d - h);
            lM = lM * f1 * f2; lI = lI * f1 * f2; lS = lS * f1 * f2; lSig = lSig * f1 * f2;
        }
    }

    // RESCALE: every few rows renormalise this thread's state so that its maximum sits near 2^TGT
    __device__ __forceinline__ void periodic() {
        V mv = P::zero();
        T m = (T)0;
#pragma unroll
        for (int x = 0; x < NV; x++) {
            m = Fx<T>::fmax_(m, Fx<T>::fmax_(Fx<T>::fmax_(P::lo(M[x]), P::hi(M[x])), Fx<T>::fmax_(P::lo(I[x]), P::hi(I[x]))));
            m = Fx<T>::fmax_(m, Fx<T>::fmax_(P::lo(S[x]), P::hi(S[x])));
        }
        m = Fx<T>::fmax_(m, Fx<T>::fmax_(Fx<T>::fmax_(P::lo(inM), P::hi(inM)), Fx<T>::fmax_(P::lo(inS), P::hi(inS))));
        m = Fx<T>::fmax_(m, Fx<T>::fmax_(Fx<T>::fmax_(P::lo(inI), P::hi(inI)), Fx<T>::fmax_(P::lo(sig), P::hi(sig))));
        (void)mv;
        if (m > (T)0) {
            int e = Fx<T>::ilogb(m);
            if (e > Fx<T>::TGT + Fx<T>::PER_HI || e < Fx<T>::TGT - Fx<T>::PER_LO) rescale(e - Fx<T>::TGT);
        } else {
            ex = EX_ZERO;
        }
    }

    // One systolic step.  E: constants of the row the .x half processes now; (lM, lI, lS, lSig): the
    // left neighbour's last-column values of that same row (already at this thread's exponent).
    __device__ __forceinline__ void step(const RowConstV0<T>& E, T lM, T lI, T lS, T lSig) {
        // .y inherits what .x had one step ago
        cA = P::pack(E.a, P::lo(cA));
        cPm = P::pack(E.pm, P::lo(cPm));
        cPx = P::pack(E.px, P::lo(cPx));
        cC = P::pack(E.c, P::lo(cC));
        cGi = P::pack(E.gi, P::lo(cGi));
        cGI = P::pack(E.gI, P::lo(cGI));
        cGm = P::pack(E.gm, P::lo(cGm));
        metaY = metaX;
        metaX = E.meta;
        // diagonal inputs of column 0 = boundary of the previous row; same-row boundary = new
        V dM = inM, dI = inI, dS = inS;
        inM = P::pack(lM, P::lo(M[NV - 1]));
        inI = P::pack(lI, P::lo(I[NV - 1]));
        inS = P::pack(lS, P::lo(S[NV - 1]));
        V sigIn = P::pack(lSig, P::lo(sig));
        const uint32_t rx = selmask(mx, metaX & 7u), ry = selmask(my, metaY & 7u);
        const T pmx = P::lo(cPm), pmy = P::hi(cPm), pxx = P::lo(cPx), pxy = P::hi(cPx);
        // pass 1, columns in DESCENDING order so that every update is in place (column x reads the
        // old values of column x-1, which are overwritten only afterwards); groups of CG columns are
        // software-pipelined by hand (stage by stage) because the packed ops are order-pinned asm.
        constexpr int CG = 4;
        static_assert(NV % CG == 0, "NV must be a multiple of 4");
#pragma unroll
        for (int xb = NV - CG; xb >= 0; xb -= CG) {
            V t[CG], u[CG], p[CG];
#pragma unroll
            for (int q = CG - 1; q >= 0; q--) {
                const int x = xb + q;
                t[q] = P::fma(cA, (x > 0) ? M[x - 1] : dM, (x > 0) ? I[x - 1] : dI);
            }
#pragma unroll
            for (int q = CG - 1; q >= 0; q--) {
                const int x = xb + q;
                t[q] = P::fma(cC, (x > 0) ? S[x - 1] : dS, t[q]);
                p[q] = P::pack(((rx >> x) & 1u) ? pmx : pxx, ((ry >> x) & 1u) ? pmy : pxy);  // Eq.3
            }
#pragma unroll
            for (int q = CG - 1; q >= 0; q--) u[q] = P::mul(cGi, M[xb + q]);
#pragma unroll
            for (int q = CG - 1; q >= 0; q--) I[xb + q] = P::fma(cGI, I[xb + q], u[q]);
#pragma unroll
            for (int q = CG - 1; q >= 0; q--) M[xb + q] = P::mul(p[q], t[q]);
        }
        // pass 2, ascending: the weighted prefix sums of the new row (Eq.6), S[x] exclusive of column x
        S[0] = P::fma(cGm, inS, inM);
#pragma unroll
        for (int x = 1; x < NV; x++) S[x] = P::fma(cGm, S[x - 1], M[x - 1]);
        // Eq.4 on the last row of a read: this thread's share, added to what came from the left
        T sx = P::lo(sigIn), sy = P::hi(sigIn);
        if ((metaX | metaY) & META_LAST) {
            T ax = (T)0, ay = (T)0;
#pragma unroll
            for (int x = 0; x < NV; x++) {
                V t = P::add(M[x], I[x]);
                ax += (x < nvx) ? P::lo(t) : (T)0;
                ay += (x < nvy) ? P::hi(t) : (T)0;
            }
            sx = (metaX & META_LAST) ? sx + ax : (T)0;
            sy = (metaY & META_LAST) ? sy + ay : (T)0;
        } else {
            sx = (T)0; sy = (T)0;
        }
        sig = P::pack(sx, sy);
    }

    __device__ __forceinline__ T outM() const { return P::hi(M[NV - 1]); }
    __device__ __forceinline__ T outI() const { return P::hi(I[NV - 1]); }
    __device__ __forceinline__ T outS() const { return P::hi(S[NV - 1]); }
    __device__ __forceinline__ T outSig() const { return P::hi(sig); }
};

}  // namespace phmm
