// Row constants of the T/J-form engine (phmm_engine.cuh), shared by the table kernel of the short path and
// the on-the-fly constant ring of the chain kernel.
//
// Stream of entries of one read of length l ("run", l + TABLE_EXTRA_ROWS entries), see phmm_engine.cuh:
//   e = 0      run-in entry: P = 0 (U = 0), gamma := 1, C := g_1, G := 0, meta FIRST.  The group's first lane
//              injects s = C/k, which the chain carries unchanged through every column, so the step leaves
//              T = g_1 C/k (= T_DM_1 D_{0,j-1}, Eq.1-2 under reading G1) and J = 0: the state in front of row 1.
//   e = 1..l   read row i = e:  P = (pm_i | px_i) gi_{i+1}, gamma_i, A = a_{i+1}/gi_{i+1}, C = g_{i+1} d_i/gi_{i+1},
//              G = gamma_{i+1} g_{i+2}/g_{i+1};  on the last row gi_{l+1} := 1, A := C := 0, G := 1, meta LAST, so
//              that the step leaves J = M_l + I_l, the summand of Eq.4.
//   e = l+1    flush entry, all zero: gives the .y half (one entry behind) its step for row l and zeroes J.
// With sum_entry (Lane2<.., SC>; l + 3 entries): the last row has A := 1, C := 0, G := 0 instead, which
// leaves T[x+1] = M_{l,x} + I_{l,x};  e = l+1 is the SUM entry (gamma := 1, pm := 0, px := 1, base code 0, all else 0):
// U = T on every column with a non-zero code, so the chain s = s + U leaves Eq.4's sum in the group's last lane;
// e = l+2 is the all-zero flush entry, which clears the J = U the sum entry left behind.
// Constants are formed in double from the 10^(-q/10) tables (lut[0..255]: insertion, deletion and continuation
// qualities; lut[256..511]: base qualities, with phmm_options.min_base_qual applied; both after qual_offset) and rounded once to the working type
// ("q32"/"q64" tables; Listing 2 :293-295 for which qualities enter which transition).
#pragma once
#include "phmm_common.cuh"
#include "phmm_kernels.h"

namespace phmm {

struct RowC { double gam, A, C, G, pm, px; uint32_t meta; };

__device__ __forceinline__ RowC row_constants(const DevBatch& b, const double* __restrict__ lut, int64_t off, int l, int e,
                                             bool sum_entry = false) {
    RowC c = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0u};
    if (sum_entry && e == l + 1) {
        c.gam = 1.0; c.px = 1.0; c.meta = META_SUM;
        return c;
    }
    if (e == 0) {
        c.gam = 1.0; c.C = 1.0 - lut[b.qual_gcp[off]]; c.meta = META_FIRST;
    } else if (e >= 1 && e <= l) {
        const int i = e;  // read row, 1-based
        const double eps = lut[256 + b.qual_base[off + i - 1]];  // (the base-quality table carries the quality floor)
        const int code = base_code(b.read_bases[off + i - 1]);
        c.meta = (uint32_t)code | META_ROW | (i == l ? META_LAST : 0u);
        c.gam = lut[b.qual_gcp[off + i - 1]];
        double gin = 1.0;  // gi_{i+1} = g_{i+2} iota_{i+1};  := 1 behind the last row
        if (i < l) {
            const double g1 = 1.0 - lut[b.qual_gcp[off + i]];                              // g_{i+1}
            const double g2 = (i + 1 < l) ? 1.0 - lut[b.qual_gcp[off + i + 1]] : 1.0;      // g_{i+2}, := 1 behind the last row
            const double io1 = lut[b.qual_ins[off + i]], de1 = lut[b.qual_del[off + i]];   // iota_{i+1}, d_{i+1}
            gin = g2 * io1;
            c.A = (1.0 - io1 - de1) / gin;
            c.C = g1 * lut[b.qual_del[off + i - 1]] / gin;
            c.G = lut[b.qual_gcp[off + i]] * g2 / g1;
        } else if (sum_entry) {
            c.A = 1.0;
        } else {
            c.G = 1.0;
        }
        c.pm = (1.0 - eps) * gin;  // (an N row matches N columns only: literal Eq.3, reading G17)
        c.px = eps / 3.0 * gin;
        if (b.n_wild && code == 4) c.px = c.pm;  // phmm_options.n_is_wildcard: a read N matches every column
    }
    return c;
}

// The 16-bit word an entry contributes to the table / ring: low byte = meta, high byte = upper byte of the fp16 number
// HSETP2 compares with the per-column base codes (A,C,G,T = 1..4, N = 6 on read rows, 0 on every other entry).
__device__ __forceinline__ uint32_t entry_word16(const RowC& c) {
    const uint32_t cd = c.meta & META_CODE_MASK;
    const uint32_t code = !(c.meta & META_ROW) ? 0u : cd < 4 ? (uint32_t)((0x4400420040003C00ull >> (16 * cd)) & 0xff00ull) : 0x4600u;
    return code | (c.meta & 0xffu);
}

}  // namespace phmm
