// Layout of the fp32 row-constant table (written by k_table_f32, phmm_short.cu) and the loads that fetch its entries:
// shared by the short kernel (phmm_short.cu) and the long kernel (phmm_long.cu).
#pragma once
#include "phmm_common.cuh"
#include "phmm_kernels.h"

#ifndef SHORT_L2_PREFETCH
#define SHORT_L2_PREFETCH 1  // table loads carry the L2 256-byte prefetch hint: +0.6 %
#endif

namespace phmm {

constexpr int TABLE_CHUNK_STRIDE = 32;  // float4 units between the chunk planes of a block
__host__ __device__ __forceinline__ int64_t table_slot(int64_t pos) {  // float4 index of chunk 0 of entry pos
    return (pos >> 5) * 128 + (pos & 1) * 16 + ((pos >> 1) & 15);
}

// read-only load that asks L2 to fetch the 256-byte pair of lines on a miss: the second line holds the slots this
// lane group reads 16 steps later
__device__ __forceinline__ float4 ldg_pf(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.L2::256B.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

__device__ __forceinline__ uint32_t ldg_pf_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.global.nc.L2::256B.b32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

struct RawEntry { float4 a, b, c; uint32_t w; };


}  // namespace phmm
