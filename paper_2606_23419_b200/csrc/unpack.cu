// unpack.cu — grinqh_unpack: bit planes -> full-precision (b_max = 8) dequantised fp16 weights, the first half of the
// paper's prefill path (PAPER.md:101 "unpack at b_max, dense GEMM", :182).  The GEMM itself is a plain
// library call on the result (cuBLAS / torch.matmul: that is where the tensor cores belong), not part of this library.
//
// One thread = one row x 32 columns: 8 coalesced plane-word loads, the same SIMD 8x8 bit transpose as the VMM
// (gather.cuh), w = s * q + z evaluated exactly in fp64 and rounded ONCE to fp16 (so the result is the correctly
// rounded value of the oracle's fp64 dequantisation), 64 contiguous bytes written per thread.  HBM-bound in principle
// (1 B read + 2 B written per weight); the fp64 conversions keep it at about half of that, which is irrelevant next
// to the GEMM it feeds.
#include "common.cuh"
#include "gather.cuh"

namespace gq {

__global__ void __launch_bounds__(256)
unpack_kernel(const uint32_t* __restrict__ planes, const __half* __restrict__ scales, const __half* __restrict__ zeros,
              int K, int N, __half* __restrict__ W) {
    const int words = N >> 5;
    const int word = blockIdx.x * 32 + (threadIdx.x & 31);
    const int k = blockIdx.y * 8 + (threadIdx.x >> 5);
    if (word >= words || k >= K) return;
    const size_t pstride = (size_t)K * words;
    const uint32_t* src = planes + (size_t)k * words + word;
    uint32_t Wd[8], V[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) Wd[j] = ld_nc_u32(src + j * pstride);
    gather<8>(Wd, V);
    const size_t gn = (size_t)(k / GQ_G) * N + (size_t)word * 32;
    __half* dst = W + (size_t)k * N + (size_t)word * 32;
#pragma unroll
    for (int L = 0; L < 4; ++L) {  // columns 8L .. 8L+7 = byte L of V[0..7]
        const uint4 sv = *reinterpret_cast<const uint4*>(scales + gn + 8 * L);
        const uint4 zv = *reinterpret_cast<const uint4*>(zeros + gn + 8 * L);
        const __half* sh = reinterpret_cast<const __half*>(&sv);
        const __half* zh = reinterpret_cast<const __half*>(&zv);
        __align__(16) __half out[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int q = (V[r] >> (8 * L)) & 0xFF;
            const double w = fma((double)__half2float(sh[r]), (double)q, (double)__half2float(zh[r]));
            out[r] = __double2half(w);
        }
        *reinterpret_cast<uint4*>(dst + 8 * L) = *reinterpret_cast<const uint4*>(out);
    }
}

}  // namespace gq

extern "C" int grinqh_unpack(const uint32_t* planes, const void* scales_f16, const void* zeros_f16, int K, int N,
                             int group, void* W_f16, void* stream) {
    if (!planes || !scales_f16 || !zeros_f16 || !W_f16) return GRINQH_ERR_NULL;
    if (group != GQ_G || K <= 0 || N <= 0 || K % GQ_G || N % 32) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)planes | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16 | (uintptr_t)W_f16) & 15)
        return GRINQH_ERR_ALIGN;
    dim3 grid((N / 32 + 31) / 32, (K + 7) / 8);
    gq::unpack_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(planes, (const __half*)scales_f16,
                                                             (const __half*)zeros_f16, K, N, (__half*)W_f16);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
