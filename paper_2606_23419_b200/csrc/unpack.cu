// unpack.cu — grinqh_unpack: bit planes -> full-precision (b_max = 8) dequantised fp16 weights, the first half of the
// paper's prefill path (PAPER.md:101 "unpack at b_max, dense GEMM", :182).  The GEMM itself is a plain
// library call on the result (cuBLAS / torch.matmul: that is where the tensor cores belong), not part of this library.
//
// One thread = one row x 32 columns: 8 coalesced plane-word loads, the same SIMD 8x8 bit transpose as the VMM
// (gather.cuh), w = s * q + z rounded ONCE to fp16 (fp32 FMA rounded to odd, then to nearest even: the correctly
// rounded value of the oracle's fp64 dequantisation), regrouped through shared memory so that a warp store covers 512
// contiguous bytes.  HBM-bound
// (1 B read + 2 B written per weight).
#include "common.cuh"
#include "gather.cuh"

namespace gq {

__global__ void __launch_bounds__(256)
unpack_kernel(const uint32_t* __restrict__ planes, const __half* __restrict__ scales, const __half* __restrict__ zeros,
              int K, int N, __half* __restrict__ W) {
    __shared__ uint4 stage[8][128];  // per warp: its row's 32 x 64 B, regrouped so that a store covers 512 contiguous bytes
    const int words = N >> 5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int word = blockIdx.x * 32 + lane;
    const int k = blockIdx.y * 8 + warp;
    if (k >= K) return;  // warp-uniform
    const bool ok = word < words;
    if (ok) {
        const size_t pstride = (size_t)K * words;
        const uint32_t* src = planes + (size_t)k * words + word;
        uint32_t Wd[8], V[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) Wd[j] = ld_nc_u32(src + j * pstride);
        gather<8>(Wd, V);
        const size_t gn = (size_t)(k / GQ_G) * N + (size_t)word * 32;
#pragma unroll
        for (int L = 0; L < 4; ++L) {  // columns 8L .. 8L+7 = byte L of V[0..7]
            const uint4 sv = *reinterpret_cast<const uint4*>(scales + gn + 8 * L);
            const uint4 zv = *reinterpret_cast<const uint4*>(zeros + gn + 8 * L);
            const __half* sh = reinterpret_cast<const __half*>(&sv);
            const __half* zh = reinterpret_cast<const __half*>(&zv);
            __align__(16) __half out[8];
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                // q as a float without a conversion instruction: 2^23 + q has q in its low mantissa bits
                const float qf = __uint_as_float(0x4B000000u | ((V[r] >> (8 * L)) & 0xFFu)) - 8388608.0f;
                const float sf = __half2float(sh[r]), zf = __half2float(zh[r]);
                // s * q is exact in fp32 (11 + 8 bits); the sum is rounded to odd at 24 bits (the two directed
                // roundings differ iff it is inexact, and exactly one of the two neighbours has an odd last bit), so
                // that the final round-to-nearest-even to fp16's 11 bits is the single rounding of the exact value.
                const float dn = __fmaf_rd(sf, qf, zf), up = __fmaf_ru(sf, qf, zf);
                // (an exact sum takes `up`: an exact zero is +0 there, as under round-to-nearest, and -0 in `dn`)
                const float ro = (dn != up && (__float_as_uint(dn) & 1u)) ? dn : up;
                out[r] = __float2half_rn(ro);
            }
            const int c = 4 * lane + L;  // 16-byte chunk of the warp's 2 KB; swizzled slot: conflict-free both ways
            stage[warp][(c & ~7) | ((c + (c >> 3)) & 7)] = *reinterpret_cast<const uint4*>(out);
        }
    }
    __syncwarp();
    __half* dst = W + (size_t)k * N + (size_t)blockIdx.x * 1024;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int c = 32 * j + lane;
        if (blockIdx.x * 32 + (c >> 2) < words)
            *reinterpret_cast<uint4*>(dst + 8 * c) = stage[warp][(c & ~7) | ((c + (c >> 3)) & 7)];
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
