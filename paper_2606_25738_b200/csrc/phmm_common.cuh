// Shared device-side definitions of the PairHMM forward kernels (sm_100a only).
//
// Recurrence implemented (row-wise reformulation of reference/PAPER.md Eq.6-7, :99-121, re-derived
// with every per-row constant folded; 1-based read row i, haplotype column j):
//     S_{i,j}  = gamma_i * S_{i,j-1} + M_{i,j}                 weighted prefix sum of row i (Eq.6: D_{i,j} = d_i S_{i,j-1})
//     I'_{i,j} = gi_i * M_{i-1,j} + gI_i * I'_{i-1,j}          I' = g_{i+1} I   (T_IM of the next row folded in)
//     M_{i,j}  = p_{i,j} * ( a_i M_{i-1,j-1} + I'_{i-1,j-1} + c_i S_{i-1,j-2} )
// with  a_i = 1-iota_i-d_i,  c_i = g_i d_{i-1} (d_0 := 1),  gi_i = g_{i+1} iota_i,  gI_i = gamma_i g_{i+1}/g_i,
//       g_i = 1-gamma_i,  g_{l+1} := 1  (so that I' = I on the last row, where Eq.4 sums M+I).
// The kernels keep U_i := gi_{i+1} M_i instead of M_i (gi_{l+1} := 1), which turns gi_i M_{i-1} into a plain
// operand: 5 FP instructions per cell (4 FMA + 1 MUL = 9 flops) and one select for p_{i,j} (Eq.3); see
// phmm_engine.cuh.  Row 0 (Eq.1 under reading G1: D_{0,j} = C/k for j = 0..k, M = I = 0) is realised as
// S_0 == C/k with gamma_0 := 1 and d_0 := 1: the first lane injects s = C/k on row 1 and the running sum
// carries it unchanged through every column.  When several reads stream through one lane group, a
// "reset row" (all constants 0) in front of each read zeroes the U and I' left by the previous read.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace phmm {

// ---- row-constant table entry: 8 scalars of type T per (read row), entry 0 of a read = reset row
// slot: 0 a_i/gi_i (row 1: 0) | 1 pm_i gi_{i+1} | 2 px_i gi_{i+1} | 3 c_i/gi_i (row 1: c_1) | 4 gI_i | 5 gamma_{i-1} | 6 - | 7 meta (bits)
// meta: bits 0-1 read base code (A,C,G,T; other bytes: pm := px, "matches nothing"), RESET, LAST, FIRST.
enum : uint32_t { META_CODE_MASK = 3u, META_RESET = 8u, META_LAST = 16u, META_FIRST = 32u };

#define PHMM_FULL 0xffffffffu

__host__ __device__ inline int base_code(uint8_t b) {
    // A,C,G,T,N -> 0..4; anything else -> 4 (documented: treated as N)
    switch (b) { case 'A': return 0; case 'C': return 1; case 'G': return 2; case 'T': return 3; default: return 4; }
}

// ---- packed pair of scalars: lane-local "virtual lanes" x (leading) and y (one row behind)
template <typename T> struct Pk;

template <> struct Pk<float> {
    typedef unsigned long long V;  // one 64-bit register pair, .x low, .y high
    static __device__ __forceinline__ V pack(float x, float y) {
        V v; asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(x), "f"(y)); return v;
    }
    static __device__ __forceinline__ float lo(V v) { return __uint_as_float((unsigned)(v & 0xffffffffull)); }
    static __device__ __forceinline__ float hi(V v) { return __uint_as_float((unsigned)(v >> 32)); }
    static __device__ __forceinline__ V fma(V a, V b, V c) { V d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
    static __device__ __forceinline__ V mul(V a, V b) { V d; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
    static __device__ __forceinline__ V add(V a, V b) { V d; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
    static __device__ __forceinline__ V zero() { return 0ull; }
};

template <> struct Pk<double> {
    struct V { double x, y; };
    static __device__ __forceinline__ V pack(double x, double y) { V v; v.x = x; v.y = y; return v; }
    static __device__ __forceinline__ double lo(V v) { return v.x; }
    static __device__ __forceinline__ double hi(V v) { return v.y; }
    static __device__ __forceinline__ V fma(V a, V b, V c) { V d; d.x = ::fma(a.x, b.x, c.x); d.y = ::fma(a.y, b.y, c.y); return d; }
    static __device__ __forceinline__ V mul(V a, V b) { V d; d.x = a.x * b.x; d.y = a.y * b.y; return d; }
    static __device__ __forceinline__ V add(V a, V b) { V d; d.x = a.x + b.x; d.y = a.y + b.y; return d; }
    static __device__ __forceinline__ V zero() { V v; v.x = 0.0; v.y = 0.0; return v; }
};

// ---- exponent helpers for the block-floating (rescaled) variants
template <typename T> struct Fx;
template <> struct Fx<float> {
    static constexpr int TGT = 16, HI = 56, PER_LO = 24, PER_HI = 24, CLAMP = 280, CLAMP1 = 126;
    static __device__ __forceinline__ int ilogb(float v) { return (int)((__float_as_uint(v) >> 23) & 0xffu) - 127; }
    // 2^e for e in [-126,127]; below -> 0, above -> 2^127
    static __device__ __forceinline__ float exp2i(int e) { return e < -126 ? 0.f : __uint_as_float((unsigned)(min(e, 127) + 127) << 23); }
    static __device__ __forceinline__ float fmax_(float a, float b) { return fmaxf(a, b); }
};
template <> struct Fx<double> {
    static constexpr int TGT = 0, HI = 600, PER_LO = 300, PER_HI = 300, CLAMP = 2200, CLAMP1 = 1022;
    static __device__ __forceinline__ int ilogb(double v) { return (int)((__double2hiint(v) >> 20) & 0x7ff) - 1023; }
    static __device__ __forceinline__ double exp2i(int e) { return e < -1022 ? 0.0 : __hiloint2double((min(e, 1023) + 1023) << 20, 0); }
    static __device__ __forceinline__ double fmax_(double a, double b) { return fmax(a, b); }
};
constexpr int EX_ZERO = -(1 << 28);  // exponent of a lane whose state is identically zero

template <typename T> __device__ __forceinline__ T shfl_up1(T v);
template <> __device__ __forceinline__ float shfl_up1<float>(float v) { return __shfl_up_sync(PHMM_FULL, v, 1); }
template <> __device__ __forceinline__ double shfl_up1<double>(double v) { return __shfl_up_sync(PHMM_FULL, v, 1); }

}  // namespace phmm
