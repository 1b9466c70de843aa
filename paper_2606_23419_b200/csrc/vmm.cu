// vmm.cu — grinqh_vmm: split-K vector-matrix multiply over the bit-planar store (v1).
// PAPER.md:85 (reconstruction), :51 (only the needed planes are fetched), :440-444 (prior-art kernel).
//
// Work item = (column tile of 1024 columns, group g of 128 rows, sub-chunk q of Q): the positions
// q, q+Q, q+2Q, ... of the group's (width desc, index asc) list `grows`, so every item of a group
// sees the same width mix.  A WARP owns `ipw` consecutive items of one column tile and is fully
// independent of the other warps until the CTA epilogue (no __syncthreads in the row loop):
//
//   meta     lane l turns list positions 4l..4l+3 into s_meta[p] = row | width << 8 | x_fp16 << 16 and the
//            warp reduces the item's scalars  X = sum_{b_k>0} x_k,  Phi = sum x_k phi_{b_k}  (phi_b = 2^(7-b)).
//   stream   a warp-private ring of RING 1-KB slots in shared memory, filled by cp.async (LDGSTS.128):
//            one instruction fetches 4 planes x 128 B of a row (lanes 8j..8j+7 copy plane j), so a 4-bit
//            row costs one and an 8-bit row two; RING-1 rows are in flight while a row is consumed.
//   expand   lane l reads its plane words (columns 32l..32l+31 of the tile) from the slot, rebuilds the 32
//            truncated codes in byte lanes (gather.cuh, SIMD 8x8 bit transpose) and does 32 mixed-precision
//            FMAs  acc[c] += half(code_c) * half(x_k)   (exact product, fp32 accumulate).
//   item end y_n += s_gn * (A_n + Phi) + z_gn * X  — s and z are applied once per (item, column) and
//            summed into the warp's shared-memory accumulator.
// CTA epilogue: the 8 warps' accumulators are added in fixed order and written as one split-K partial
// part[sx][t][n]; vmm_reduce sums the Sx partials in fixed order.  Everything is deterministic.
#include "common.cuh"
#include "gather.cuh"

namespace gq {

constexpr int VW = 8;  // warps per CTA
constexpr int VTHREADS = VW * 32;
constexpr int TILE_COLS = 1024;
constexpr int SLOT_BYTES = 1024;   // 8 planes x 128 B
constexpr int YSLOT = 32 * 33;     // one warp's 1024 sums, padded: column 32*l + c lives at c*33 + l
constexpr int NUM_SMS = 148;
constexpr int CTAS_PER_SM = 2;

template <int T>
struct Cfg {
    static constexpr int RING = (T == 1) ? 8 : 4;
    // per-warp shared memory: ring | yacc[T] | meta[128] u32 | x[T][128] u16 | tb[T][128] u8
    static constexpr int RING_OFF = 0;
    static constexpr int YACC_OFF = RING * SLOT_BYTES;
    static constexpr int META_OFF = YACC_OFF + T * YSLOT * 4;
    static constexpr int X_OFF = META_OFF + 512;
    static constexpr int TB_OFF = X_OFF + T * 256;
    static constexpr int WARP_BYTES = TB_OFF + T * 128;
    static constexpr int SMEM = VW * WARP_BYTES;
    static_assert(WARP_BYTES % 16 == 0, "warp regions stay 16-byte aligned");
};

struct VmmPlan {
    int col_tiles;  // ceil(N / 1024)
    int Q;          // sub-chunks per group
    int Sx;         // CTAs (= split-K partials) per column tile
    int ipw;        // items per warp; warp slot ws owns items [ws*ipw, min(I, (ws+1)*ipw)), I = (K/128)*Q
};

// Static plan from the shape only (the workspace size depends on it).  Cost model in "rows": a warp does
// ipw * (rows per item + item overhead); pick the Q in 1..8 that minimises it under the residency limit.
static inline VmmPlan vmm_plan(int T, int K, int N) {
    VmmPlan best{};
    const int CT = (N + TILE_COLS - 1) / TILE_COLS;
    const int groups = K / GQ_G;
    const int resident = NUM_SMS * ((T <= 2) ? CTAS_PER_SM : 1);
    const int sx_max = resident / CT > 0 ? resident / CT : 1;
    double best_cost = 1e30;
    for (int Q = 1; Q <= 8; ++Q) {
        const int I = groups * Q;
        int Sx = (I + VW - 1) / VW;
        if (Sx > sx_max) Sx = sx_max;
        const int ipw = (I + VW * Sx - 1) / (VW * Sx);
        Sx = (I + VW * ipw - 1) / (VW * ipw);
        const double cost = ipw * (112.0 / Q + 3.0);
        if (cost < best_cost - 1e-9) {
            best_cost = cost;
            best = VmmPlan{CT, Q, Sx, ipw};
        }
    }
    return best;
}

// codes are fed to the FMA as fp16 bit patterns 0x00cc = cc * 2^-24 (subnormal halfs, exact)
constexpr float CODE_SCALE = 16777216.0f;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

__device__ __forceinline__ void accumulate_row(const uint32_t (&V)[8], uint16_t xh, float* acc) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const uint32_t h01 = __byte_perm(V[r], 0u, 0x4140);  // [b0, 0, b1, 0]
        const uint32_t h23 = __byte_perm(V[r], 0u, 0x4342);  // [b2, 0, b3, 0]
        fhfma_lo(acc[4 * r + 0], h01, xh);
        fhfma_hi(acc[4 * r + 1], h01, xh);
        fhfma_lo(acc[4 * r + 2], h23, xh);
        fhfma_hi(acc[4 * r + 3], h23, xh);
    }
}

// plane words of one row (ring slot) -> truncated codes V; b is warp-uniform
__device__ __forceinline__ void expand_row(const uint32_t* slot, int lane, int b, uint32_t (&V)[8]) {
    uint32_t Wd[8];
    if (b == 8) {
#pragma unroll
        for (int j = 0; j < 8; ++j) Wd[j] = slot[j * 32 + lane];
        gather<8>(Wd, V);
    } else if (b == 4) {
#pragma unroll
        for (int j = 0; j < 4; ++j) Wd[j] = slot[j * 32 + lane];
        gather<4>(Wd, V);
    } else if (b == 2) {
#pragma unroll
        for (int j = 0; j < 2; ++j) Wd[j] = slot[j * 32 + lane];
        gather<2>(Wd, V);
    } else {  // any other width: stale slot words beyond the row's planes are masked off
#pragma unroll
        for (int j = 0; j < 8; ++j) Wd[j] = (j < b) ? slot[j * 32 + lane] : 0u;
        gather<8>(Wd, V);
    }
}

// A16: every plane row is 16-byte aligned (N % 128 == 0) -> LDGSTS.128, 4 planes per instruction;
// otherwise each lane copies its own word of every plane with 4-byte cp.async.
template <int T, bool A16>
__global__ void __launch_bounds__(VTHREADS, (T <= 2) ? CTAS_PER_SM : 1)
vmm_main_kernel(const uint16_t* __restrict__ x, int K, int N, int Q, int ipw,
                const uint32_t* __restrict__ planes, const __half* __restrict__ scales,
                const __half* __restrict__ zeros, const uint8_t* __restrict__ bits,
                const uint8_t* __restrict__ grows, const uint8_t* __restrict__ gcnt_ge,
                float* __restrict__ part) {
    using C = Cfg<T>;
    constexpr int RING = C::RING;
    extern __shared__ __align__(16) uint8_t smem[];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, sx = blockIdx.y;
    const int words = N >> 5;
    const int word = tile * 32 + lane;
    const bool active = word < words;
    const size_t pstride = (size_t)K * words;
    const int groups = K / GQ_G;
    const int I = groups * Q;

    uint8_t* wbase = smem + warp * C::WARP_BYTES;
    const uint32_t* ring = reinterpret_cast<const uint32_t*>(wbase + C::RING_OFF);
    float* yacc = reinterpret_cast<float*>(wbase + C::YACC_OFF);
    uint32_t* s_meta = reinterpret_cast<uint32_t*>(wbase + C::META_OFF);
    uint16_t* s_x = reinterpret_cast<uint16_t*>(wbase + C::X_OFF);
    uint8_t* s_tb = wbase + C::TB_OFF;
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(wbase + C::RING_OFF);

    // per-lane copy geometry
    const int pj = lane >> 3, seg = lane & 7;
    const bool chunk_ok = A16 ? (tile * 32 + seg * 4 < words) : active;
    const uint32_t* lane_src = A16 ? planes + (size_t)pj * pstride + tile * 32 + seg * 4 : planes + word;
    const uint32_t lane_dst = A16 ? ring_s + pj * 128 + seg * 16 : ring_s + lane * 4;

    const int ws = sx * VW + warp;
    const int it0 = ws * ipw;
    const int it1 = min(I, it0 + ipw);
    bool first = true;

    for (int it = it0; it < it1; ++it) {
        const int g = it / Q, q = it - g * Q;
        __syncwarp();
        // ---- meta: positions 4l..4l+3 of the group's list
        const uint32_t lst = *reinterpret_cast<const uint32_t*>(grows + g * GQ_G + 4 * lane);
        const uint4 cv = *reinterpret_cast<const uint4*>(gcnt_ge + g * GQ_GCNT);
#pragma unroll
        for (int t = 0; t < T; ++t) {
            *reinterpret_cast<uint2*>(s_x + t * GQ_G + 4 * lane) =
                *reinterpret_cast<const uint2*>(x + (size_t)t * K + g * GQ_G + 4 * lane);
            if (T > 1)
                *reinterpret_cast<uint32_t*>(s_tb + t * GQ_G + 4 * lane) =
                    *reinterpret_cast<const uint32_t*>(bits + (size_t)t * K + g * GQ_G + 4 * lane);
        }
        __syncwarp();
        const int nnz = (cv.x >> 8) & 0xFF;  // cnt[1]
        float X[T], Phi[T];
#pragma unroll
        for (int t = 0; t < T; ++t) X[t] = Phi[t] = 0.f;
        uint32_t mt[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int p = 4 * lane + i;
            const int r = (lst >> (8 * i)) & 0xFF;
            int b = 0;  // b = #{w in 1..8 : p < cnt[w]}
            b += (p < (int)((cv.x >> 8) & 0xFF)) + (p < (int)((cv.x >> 16) & 0xFF)) + (p < (int)(cv.x >> 24));
            b += (p < (int)(cv.y & 0xFF)) + (p < (int)((cv.y >> 8) & 0xFF)) + (p < (int)((cv.y >> 16) & 0xFF)) +
                 (p < (int)(cv.y >> 24));
            b += (p < (int)(cv.z & 0xFF));
            mt[i] = (uint32_t)r | ((uint32_t)b << 8) | ((uint32_t)s_x[r] << 16);
            const bool mine = (p < nnz) && (p >= q) && ((p - q) % Q == 0);
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const int bt = (T == 1) ? b : (int)s_tb[t * GQ_G + r];
                if (mine && bt > 0) {
                    const float xf = __half2float(__ushort_as_half(s_x[t * GQ_G + r]));
                    X[t] += xf;
                    Phi[t] = fmaf(xf, (float)(0x80 >> bt), Phi[t]);  // phi_b = 2^(7-b), phi_8 = 0
                }
            }
        }
        *reinterpret_cast<uint4*>(s_meta + 4 * lane) = make_uint4(mt[0], mt[1], mt[2], mt[3]);
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                X[t] += __shfl_xor_sync(0xffffffffu, X[t], d);
                Phi[t] += __shfl_xor_sync(0xffffffffu, Phi[t], d);
            }
        __syncwarp();

        const int n_rows = (nnz > q) ? (nnz - q + Q - 1) / Q : 0;
        const uint32_t* item_src = lane_src + (size_t)g * GQ_G * words;

        auto issue = [&](int i) {
            const uint32_t m = s_meta[q + i * Q];
            const int r = m & 0xFF, b = (m >> 8) & 0xFF;
            const uint32_t* src = item_src + (uint32_t)(r * words);
            const uint32_t dst = lane_dst + (i % RING) * SLOT_BYTES;
            if (A16) {
                if (chunk_ok && pj < b) cp_async16(dst, src);
                if (b > 4 && chunk_ok && pj + 4 < b) cp_async16(dst + 512, src + 4 * pstride);
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (chunk_ok && j < b) cp_async4(dst + j * 128, src + j * pstride);
            }
        };

        float acc[T][32];
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int c = 0; c < 32; ++c) acc[t][c] = 0.f;

#pragma unroll
        for (int i = 0; i < RING - 1; ++i) {
            if (i < n_rows) issue(i);
            cp_async_commit();
        }
        for (int i = 0; i < n_rows; ++i) {
            cp_async_wait<RING - 2>();
            __syncwarp();
            if (i + RING - 1 < n_rows) issue(i + RING - 1);
            cp_async_commit();
            const uint32_t m = s_meta[q + i * Q];
            const int b = (m >> 8) & 0xFF;
            uint32_t V[8];
            expand_row(ring + (i % RING) * (SLOT_BYTES / 4), lane, b, V);
            if (T == 1) {
                accumulate_row(V, (uint16_t)(m >> 16), acc[0]);
            } else {
                const int r = m & 0xFF;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const int bt = s_tb[t * GQ_G + r];  // this token's own width (<= b, the union)
                    if (bt == 0) continue;              // warp-uniform
                    const uint32_t mask = 0x01010101u * ((0xFF00u >> bt) & 0xFFu);
                    uint32_t Vm[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) Vm[j] = V[j] & mask;
                    accumulate_row(Vm, s_x[t * GQ_G + r], acc[t]);
                }
            }
        }
        cp_async_wait<0>();

        // ---- item end: s and z once per (item, column), into the warp's accumulator
        if (active) {
            const size_t gn = (size_t)g * N + (size_t)word * 32;
#pragma unroll
            for (int L = 0; L < 4; ++L) {
                float sf[8], zf[8];
                if (n_rows > 0) {
                    const uint4 sv = *reinterpret_cast<const uint4*>(scales + gn + 8 * L);
                    const uint4 zv = *reinterpret_cast<const uint4*>(zeros + gn + 8 * L);
                    const uint32_t su[4] = {sv.x, sv.y, sv.z, sv.w}, zu[4] = {zv.x, zv.y, zv.z, zv.w};
#pragma unroll
                    for (int h = 0; h < 4; ++h) {
                        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&su[h]));
                        const float2 c = __half22float2(*reinterpret_cast<const __half2*>(&zu[h]));
                        sf[2 * h] = a.x; sf[2 * h + 1] = a.y;
                        zf[2 * h] = c.x; zf[2 * h + 1] = c.y;
                    }
                }
#pragma unroll
                for (int t = 0; t < T; ++t)
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        float* dst = yacc + t * YSLOT + (8 * L + r) * 33 + lane;
                        float v = first ? 0.f : *dst;
                        if (n_rows > 0) v += fmaf(sf[r], fmaf(acc[t][4 * r + L], CODE_SCALE, Phi[t]), zf[r] * X[t]);
                        *dst = v;
                    }
            }
        }
        first = false;
    }
    if (first && active) {  // a warp without items still owns a slot in the CTA sum
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int c = 0; c < 32; ++c) yacc[t * YSLOT + c * 33 + lane] = 0.f;
    }
    __syncthreads();

    // ---- CTA epilogue: fixed-order sum over the 8 warps -> one split-K partial
#pragma unroll
    for (int t = 0; t < T; ++t)
#pragma unroll
        for (int i = 0; i < TILE_COLS / VTHREADS; ++i) {
            const int c = tid + VTHREADS * i;  // column inside the tile
            const int n = tile * TILE_COLS + c;
            if (n < N) {
                const int idx = (c & 31) * 33 + (c >> 5);
                float A = 0.f;
#pragma unroll
                for (int w = 0; w < VW; ++w)
                    A += *reinterpret_cast<const float*>(smem + w * C::WARP_BYTES + C::YACC_OFF + (t * YSLOT + idx) * 4);
                part[((size_t)sx * T + t) * N + n] = A;
            }
        }
}

// y[t][n] = sum_{s=0}^{S-1} part[s][t][n], always in the same order: warp w adds s = w, w+8, ...
// sequentially, then the 8 warp sums are added in order w = 0..7.
__global__ void __launch_bounds__(VTHREADS)
vmm_reduce_kernel(const float* __restrict__ part, int S, int T, int N, float* __restrict__ y) {
    __shared__ float4 red[VW][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int t = blockIdx.y;
    const int n = blockIdx.x * 128 + lane * 4;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    if (n < N) {
        for (int s = warp; s < S; s += VW) {
            const float4 v = *reinterpret_cast<const float4*>(part + ((size_t)s * T + t) * N + n);
            a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
        }
    }
    red[warp][lane] = a;
    __syncthreads();
    if (warp == 0 && n < N) {
        float4 r = red[0][lane];
#pragma unroll
        for (int w = 1; w < VW; ++w) {
            const float4 v = red[w][lane];
            r.x += v.x; r.y += v.y; r.z += v.z; r.w += v.w;
        }
        *reinterpret_cast<float4*>(y + (size_t)t * N + n) = r;
    }
}

template <int T, bool A16>
static int launch_main_impl(const void* x, int K, int N, const VmmPlan& pl, const uint32_t* planes, const void* scales,
                            const void* zeros, const uint8_t* bits, const uint8_t* grows, const uint8_t* gcnt_ge,
                            float* part, cudaStream_t st) {
    constexpr int smem = Cfg<T>::SMEM;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(vmm_main_kernel<T, A16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) !=
            cudaSuccess)
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    dim3 grid(pl.col_tiles, pl.Sx);
    vmm_main_kernel<T, A16><<<grid, VTHREADS, smem, st>>>((const uint16_t*)x, K, N, pl.Q, pl.ipw, planes,
                                                          (const __half*)scales, (const __half*)zeros, bits, grows,
                                                          gcnt_ge, part);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

template <int T>
static int launch_main(const void* x, int K, int N, const VmmPlan& pl, const uint32_t* planes, const void* scales,
                       const void* zeros, const uint8_t* bits, const uint8_t* grows, const uint8_t* gcnt_ge,
                       float* part, cudaStream_t st) {
    if (N % 128 == 0)
        return launch_main_impl<T, true>(x, K, N, pl, planes, scales, zeros, bits, grows, gcnt_ge, part, st);
    return launch_main_impl<T, false>(x, K, N, pl, planes, scales, zeros, bits, grows, gcnt_ge, part, st);
}

static int check_vmm_args(int T, int K, int N, int group) {
    if (group != GQ_G || T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32) return GRINQH_ERR_SHAPE;
    return GRINQH_OK;
}

}  // namespace gq

extern "C" size_t grinqh_vmm_workspace_bytes(int T, int K, int N) {
    if (gq::check_vmm_args(T, K, N, GQ_G) != GRINQH_OK) return 0;
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    return (size_t)pl.Sx * T * N * sizeof(float);
}

extern "C" int grinqh_vmm_main(const void* x_f16, int T, int K, int N, int group, const uint32_t* planes,
                               const void* scales_f16, const void* zeros_f16, const uint8_t* bits,
                               const uint8_t* bits_union, const uint8_t* grows, const uint8_t* gcnt_ge,
                               void* workspace, size_t workspace_bytes, void* stream) {
    if (!x_f16 || !planes || !scales_f16 || !zeros_f16 || !bits || !bits_union || !grows || !gcnt_ge || !workspace)
        return GRINQH_ERR_NULL;
    int rc = gq::check_vmm_args(T, K, N, group);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)x_f16 | (uintptr_t)planes | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16 | (uintptr_t)bits |
         (uintptr_t)grows | (uintptr_t)gcnt_ge | (uintptr_t)workspace) & 15)
        return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    cudaStream_t st = (cudaStream_t)stream;
    float* part = (float*)workspace;
    switch (T) {
        case 1: return gq::launch_main<1>(x_f16, K, N, pl, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        case 2: return gq::launch_main<2>(x_f16, K, N, pl, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        case 3: return gq::launch_main<3>(x_f16, K, N, pl, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        default: return gq::launch_main<4>(x_f16, K, N, pl, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
    }
}

extern "C" int grinqh_vmm_reduce(int T, int K, int N, float* y, const void* workspace, size_t workspace_bytes,
                                 void* stream) {
    if (!y || !workspace) return GRINQH_ERR_NULL;
    int rc = gq::check_vmm_args(T, K, N, GQ_G);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)y | (uintptr_t)workspace) & 15) return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    dim3 grid((N + 127) / 128, T);
    gq::vmm_reduce_kernel<<<grid, gq::VTHREADS, 0, (cudaStream_t)stream>>>((const float*)workspace, pl.Sx, T, N, y);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

extern "C" int grinqh_vmm(const void* x_f16, int T, int K, int N, int group, const uint32_t* planes,
                          const void* scales_f16, const void* zeros_f16, const uint8_t* bits,
                          const uint8_t* bits_union, const uint8_t* grows, const uint8_t* gcnt_ge, float* y,
                          void* workspace, size_t workspace_bytes, void* stream) {
    if (!y) return GRINQH_ERR_NULL;
    if ((uintptr_t)y & 15) return GRINQH_ERR_ALIGN;
    int rc = grinqh_vmm_main(x_f16, T, K, N, group, planes, scales_f16, zeros_f16, bits, bits_union, grows, gcnt_ge,
                             workspace, workspace_bytes, stream);
    if (rc != GRINQH_OK) return rc;
    return grinqh_vmm_reduce(T, K, N, y, workspace, workspace_bytes, stream);
}
