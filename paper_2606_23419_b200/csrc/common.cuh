// common.cuh — shared device/host helpers of the CUDA library (sm_100a only).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

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
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

}  // namespace gq
