// common.cuh — shared device/host helpers of the CUDA library (sm_100a only).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include "../../include/grinqh.h"

#define GQ_G 128             // group size along K
#define GQ_GCNT 16           // bytes per group in gcnt_ge
#define GQ_MAX_K 32768       // assignment keeps keys + a 32768-bin histogram in one CTA's shared memory

namespace gq {

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }

__device__ __forceinline__ uint32_t ld_nc_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint2 ld_nc_u32x2(const uint32_t* p) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
    return v;
}

// acc += half(a_lo16) * half(x): mixed-precision FMA (PTX fma.rn.f32.f16 -> SASS FHFMA).
// The product of two fp16 values is exact in fp32; one rounding on the add.
__device__ __forceinline__ void fhfma_lo(float& acc, uint32_t a, uint16_t x) {
    asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %1;\n\tfma.rn.f32.f16 %0, lo, %2, %0;\n\t}"
        : "+f"(acc) : "r"(a), "h"(x));
}
__device__ __forceinline__ void fhfma_hi(float& acc, uint32_t a, uint16_t x) {
    asm("{\n\t.reg .b16 lo, hi;\n\tmov.b32 {lo, hi}, %1;\n\tfma.rn.f32.f16 %0, hi, %2, %0;\n\t}"
        : "+f"(acc) : "r"(a), "h"(x));
}

// Stable partition of a 128-row group by (width desc, index asc), one warp, lane l owns rows 4l..4l+3 with widths
// bu[0..3] (0..8).  Per-lane counts of the 9 widths are packed in byte fields (widths 0..7 in a u64, width 8 apart; a
// prefix never exceeds 128) and scanned once.  pos[i] = position of row 4l+i in the group's list; ge[c] = rows of
// width >= c (ge[9] = 0), the same on every lane.
__device__ __forceinline__ void partition128(const int (&bu)[4], int lane, int (&pos)[4], int (&ge)[10]) {
    unsigned long long cntA = 0;
    uint32_t cnt8 = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (bu[i] == 8) ++cnt8;
        else cntA += 1ull << (8 * bu[i]);
    }
    unsigned long long inA = cntA;
    uint32_t in8 = cnt8;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned long long oA = __shfl_up_sync(0xffffffffu, inA, d);
        const uint32_t o8 = __shfl_up_sync(0xffffffffu, in8, d);
        if (lane >= d) {
            inA += oA;
            in8 += o8;
        }
    }
    const unsigned long long totA = __shfl_sync(0xffffffffu, inA, 31);
    const uint32_t tot8 = __shfl_sync(0xffffffffu, in8, 31);
    unsigned long long exA = inA - cntA;  // rows of each width in lower lanes
    uint32_t ex8 = in8 - cnt8;
    ge[9] = 0;
    ge[8] = (int)tot8;
#pragma unroll
    for (int c = 7; c >= 0; --c) ge[c] = ge[c + 1] + (int)((totA >> (8 * c)) & 0xFF);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int c = bu[i];
        int above = 0, lower;  // above = rows of larger width
#pragma unroll
        for (int w = 0; w <= 8; ++w)
            if (w == c) above = ge[w + 1];
        if (c == 8) {
            lower = (int)ex8++;
        } else {
            lower = (int)((exA >> (8 * c)) & 0xFF);
            exA += 1ull << (8 * c);
        }
        pos[i] = above + lower;
    }
}

// Programmatic dependent launch (PDL): every per-step kernel is launched with programmatic stream serialization,
// calls pdl_launch_dependents() at its top (the next kernel of the stream may be scheduled as SMs free up) and
// pdl_wait() before its first global-memory access (blocks until the previous kernel has completed and flushed).
// Launch latency, CTA scheduling and the prologue arithmetic of kernel n+1 overlap the tail of kernel n.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    static const bool no_pdl = getenv("GRINQH_NO_PDL") != nullptr;  // measurement switch
    cfg.numAttrs = no_pdl ? 0 : 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace gq
