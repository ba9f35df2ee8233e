// Shared device-side definitions of the PairHMM forward kernels (sm_100a only).
//
// Recurrence implemented (row-wise reformulation of reference/PAPER.md Eq.6-7, :99-121, re-derived
// with every per-row constant folded; 1-based read row i, haplotype column j):
//     S_{i,j}  = gamma_i * S_{i,j-1} + M_{i,j}                 weighted prefix sum of row i (Eq.6: D_{i,j} = d_i S_{i,j-1})
//     I'_{i,j} = gi_i * M_{i-1,j} + gI_i * I'_{i-1,j}          I' = g_{i+1} I   (T_IM of the next row folded in)
//     M_{i,j}  = p_{i,j} * ( a_i M_{i-1,j-1} + I'_{i-1,j-1} + c_i S_{i-1,j-2} )
// with  a_i = 1-iota_i-d_i,  c_i = g_i d_{i-1} (d_0 := 1),  gi_i = g_{i+1} iota_i,  gI_i = gamma_i g_{i+1}/g_i,
//       g_i = 1-gamma_i,  g_{l+1} := 1  (so that I' = I on the last row, where Eq.4 sums M+I).
// The fp32 kernels keep U_i := gi_{i+1} M_i instead of M_i (gi_{l+1} := 1) and, per column, the pre-emission sum T of
// the NEXT row instead of M: 5 FP instructions per cell (4 FMA + 1 MUL = 9 flops) and one select for p_{i,j} (Eq.3);
// see phmm_engine.cuh for the step and phmm_rowconst.cuh for the per-row constants and for how Eq.1 (run-in
// entry: S_0 == C/k under reading G1) and Eq.4 (last row leaves M+I) are realised.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace phmm {

// ---- meta word of a stream entry: bits 0-2 read base code (A,C,G,T = 0..3, N and every other byte = 4: Eq.3 compares
// literally, so N matches N and nothing else, reading G17),
// ROW = a read row (entries 1..l), LAST = the read's last row, FIRST = run-in entry (the group's first lane injects C/k),
// SUM = the sum entry behind the last row (phmm_rowconst.cuh), on which the running sum s collects Eq.4.
enum : uint32_t { META_CODE_MASK = 7u, META_ROW = 8u, META_LAST = 16u, META_FIRST = 32u, META_SUM = 64u };

#define PHMM_FULL 0xffffffffu

__host__ __device__ inline int base_code(uint8_t b) {
    // A,C,G,T,N -> 0..4; anything else -> 4 (documented: treated as N)
    switch (b) { case 'A': return 0; case 'C': return 1; case 'G': return 2; case 'T': return 3; default: return 4; }
}

// ---- exponent helpers for the block-floating (rescaled) variants
template <typename T> struct Fx;
template <> struct Fx<float> {
    static constexpr int CLAMP = 280, CLAMP1 = 126;  // largest shift applied with two factors / with one
    static __device__ __forceinline__ int ilogb(float v) { return (int)((__float_as_uint(v) >> 23) & 0xffu) - 127; }
    // 2^e for e in [-126,127]; below -> 0, above -> 2^127
    static __device__ __forceinline__ float exp2i(int e) { return e < -126 ? 0.f : __uint_as_float((unsigned)(min(e, 127) + 127) << 23); }
    static __device__ __forceinline__ float fmax_(float a, float b) { return fmaxf(a, b); }
};
template <> struct Fx<double> {
    static constexpr int CLAMP = 2200, CLAMP1 = 1022;
    static __device__ __forceinline__ int ilogb(double v) { return (int)((__double2hiint(v) >> 20) & 0x7ff) - 1023; }
    static __device__ __forceinline__ double exp2i(int e) { return e < -1022 ? 0.0 : __hiloint2double((min(e, 1023) + 1023) << 20, 0); }
    static __device__ __forceinline__ double fmax_(double a, double b) { return fmax(a, b); }
};

template <typename T> __device__ __forceinline__ T shfl_up1(T v);
template <> __device__ __forceinline__ float shfl_up1<float>(float v) { return __shfl_up_sync(PHMM_FULL, v, 1); }
template <> __device__ __forceinline__ double shfl_up1<double>(double v) { return __shfl_up_sync(PHMM_FULL, v, 1); }

}  // namespace phmm
