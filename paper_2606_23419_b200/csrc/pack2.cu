// pack2.cu — grinqh_pack_seg2: the paper's own storage granularity: b_max-bit asymmetric group codes,
// b_max in {4, 6, 8}, split into b_max / 2 two-bit significance segments.
// Layout (defined by the oracle's formula, oracle/grinqh_oracle.cpp orc_pack2): segs[sigma][k][n >> 4], sigma = 0 the most
// significant pair, column n's pair at bits 2 (n & 15) + {1, 0}: sixteen 2-bit chunks per uint32.
// Offline, once per weight: two plain kernels (group min / max -> scale and zero; codes -> segment words).  The
// quantiser is that of grinqh_pack with 2^b_max - 1 steps, every fp32 step an IEEE operation (no contraction).
#include "common.cuh"

namespace gq {

// one thread per (group, column): lo / hi of the 128 fp16 values in row order (first minimum wins, zero is +0)
__global__ void __launch_bounds__(256)
pack2_scale_kernel(const __half* __restrict__ W, int K, int N, float qmax, __half* __restrict__ scales,
                   __half* __restrict__ zeros) {
    const int n = blockIdx.x * 256 + threadIdx.x, g = blockIdx.y;
    if (n >= N) return;
    const __half* p = W + (size_t)g * GQ_G * N + n;
    __half lo_h = p[0];
    float lo = __half2float(lo_h), hi = lo;
#pragma unroll 8
    for (int i = 1; i < GQ_G; ++i) {
        const __half h = p[(size_t)i * N];
        const float v = __half2float(h);
        if (v < lo) {
            lo = v;
            lo_h = h;
        }
        if (v > hi) hi = v;
    }
    if (lo == 0.0f) lo_h = __ushort_as_half((unsigned short)0);
    const float s32 = __fdiv_rn(__fsub_rn(hi, lo), qmax);
    scales[(size_t)g * N + n] = __float2half_rn(s32);
    zeros[(size_t)g * N + n] = lo_h;
}

// one thread per (row, word of 16 columns): codes against the STORED fp16 scale, b_max / 2 segment words
__global__ void __launch_bounds__(256)
pack2_codes_kernel(const __half* __restrict__ W, int K, int N, int bmax, float qmax, const __half* __restrict__ scales,
                   const __half* __restrict__ zeros, uint32_t* __restrict__ segs) {
    const int words = N >> 4;
    const int wi = blockIdx.x * 256 + threadIdx.x, k = blockIdx.y;
    if (wi >= words) return;
    const int g = k / GQ_G;
    uint32_t out[4] = {0u, 0u, 0u, 0u};
#pragma unroll
    for (int half = 0; half < 2; ++half) {
        const uint4 wv = *reinterpret_cast<const uint4*>(W + (size_t)k * N + wi * 16 + 8 * half);
        const uint4 sv = *reinterpret_cast<const uint4*>(scales + (size_t)g * N + wi * 16 + 8 * half);
        const uint4 zv = *reinterpret_cast<const uint4*>(zeros + (size_t)g * N + wi * 16 + 8 * half);
        const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w}, ss[4] = {sv.x, sv.y, sv.z, sv.w}, zz[4] = {zv.x, zv.y, zv.z, zv.w};
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float w = __half2float(__ushort_as_half((unsigned short)(ww[j >> 1] >> (16 * (j & 1)))));
            const float s = __half2float(__ushort_as_half((unsigned short)(ss[j >> 1] >> (16 * (j & 1)))));
            const float z = __half2float(__ushort_as_half((unsigned short)(zz[j >> 1] >> (16 * (j & 1)))));
            int q = 0;
            if (s != 0.0f) {
                float r = rintf(__fdiv_rn(__fsub_rn(w, z), s));  // round-half-even
                r = fminf(fmaxf(r, 0.0f), qmax);
                q = (int)r;
            }
            const int c = 8 * half + j;
#pragma unroll
            for (int sg = 0; sg < 4; ++sg)
                if (2 * sg < bmax) out[sg] |= (uint32_t)((q >> (bmax - 2 - 2 * sg)) & 3) << (2 * c);
        }
    }
    const size_t stride = (size_t)K * words;
#pragma unroll
    for (int sg = 0; sg < 4; ++sg)
        if (2 * sg < bmax) segs[(size_t)sg * stride + (size_t)k * words + wi] = out[sg];
}

}  // namespace gq

extern "C" int grinqh_pack_seg2(const void* W_f16, int K, int N, int group, int bmax, uint32_t* segs, void* scales_f16,
                                void* zeros_f16, void* stream) {
    if (!W_f16 || !segs || !scales_f16 || !zeros_f16) return GRINQH_ERR_NULL;
    if (group != GQ_G || K <= 0 || N <= 0 || K % GQ_G || N % 32 || (bmax != 4 && bmax != 6 && bmax != 8))
        return GRINQH_ERR_SHAPE;
    if (((uintptr_t)W_f16 | (uintptr_t)segs | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16) & 15) return GRINQH_ERR_ALIGN;
    const float qmax = (float)((1 << bmax) - 1);
    cudaStream_t st = (cudaStream_t)stream;
    gq::pack2_scale_kernel<<<dim3((N + 255) / 256, K / GQ_G), 256, 0, st>>>((const __half*)W_f16, K, N, qmax,
                                                                              (__half*)scales_f16, (__half*)zeros_f16);
    gq::pack2_codes_kernel<<<dim3((N / 16 + 255) / 256, K), 256, 0, st>>>((const __half*)W_f16, K, N, bmax, qmax,
                                                                           (const __half*)scales_f16,
                                                                           (const __half*)zeros_f16, segs);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
