// vmm.cu — grinqh_vmm: split-K vector-matrix multiply over the bit-planar store, CTAs walking the
// compacted per-group row lists; deterministic second-pass reduce.
// PAPER.md:85 (reconstruction), :51 (only the needed planes are fetched), :440-444 (prior-art kernel).
//
// Work unit = (group g of 128 rows, column tile of 1024 columns, strided sub-chunk q of Q):
// sub-chunk q takes positions q, q+Q, ... of the group's (width desc) list, so every sub-chunk sees the
// same width mix.  One CTA of 8 warps per unit; warp w takes every 8th of those positions; lane l owns
// the 32 columns of plane word (32*tile + l).  Per row a lane loads one word per fetched plane,
// rebuilds the 32 truncated codes in byte lanes (gather.cuh), and does 32 mixed-precision FMAs
//     acc[c] += half(code_c) * half(x_k)          (fp16 x fp16 product is exact in fp32)
// The midpoint bias phi and the zero-point need only per-group scalars:
//     y_n += s_gn * (A_n + Phi_g) + z_gn * X_g,   Phi_g = sum x_k phi_{b_k},  X_g = sum_{b_k>0} x_k.
// The CTA reduces its warps in fixed order in shared memory, applies s and z once per (group, column)
// and writes one split-K partial; vmm_reduce sums the partials in fixed order s = 0..S-1.
#include "common.cuh"
#include "gather.cuh"

namespace gq {

constexpr int VW = 8;          // warps per CTA
constexpr int VTHREADS = VW * 32;
constexpr int TILE_COLS = 1024;
constexpr int SLOT = 32 * 33;  // one warp's 1024 partial sums, padded: column 32*l + p lives at p*33 + l
constexpr int NUM_SMS = 148;

struct VmmGeom {
    int Q, S, col_tiles;
};

static inline VmmGeom vmm_geometry(int K, int N) {
    VmmGeom g;
    g.col_tiles = (N + TILE_COLS - 1) / TILE_COLS;
    const int groups = K / GQ_G;
    const int target = NUM_SMS * 4;
    int Q = (target + groups * g.col_tiles - 1) / (groups * g.col_tiles);
    g.Q = Q < 1 ? 1 : (Q > 8 ? 8 : Q);
    g.S = groups * g.Q;
    return g;
}

// codes are fed to the FMA as fp16 bit patterns 0x00cc = cc * 2^-24 (subnormal halfs, exact)
constexpr float CODE_SCALE = 16777216.0f;

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

template <int T>
__global__ void __launch_bounds__(VTHREADS)
vmm_main_kernel(const uint16_t* __restrict__ x, int K, int N, int Q, const uint32_t* __restrict__ planes,
                const __half* __restrict__ scales, const __half* __restrict__ zeros,
                const uint8_t* __restrict__ bits, const uint8_t* __restrict__ grows,
                const uint8_t* __restrict__ gcnt_ge, float* __restrict__ part) {
    extern __shared__ __align__(16) float slots[];  // [VW][T][SLOT]
    __shared__ uint16_t s_x[T][GQ_G];
    __shared__ uint8_t s_tb[T][GQ_G];
    __shared__ uint8_t s_list[GQ_G];
    __shared__ uint8_t s_cnt[GQ_GCNT];
    __shared__ float s_X[VW][T], s_Phi[VW][T];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x;
    const int g = blockIdx.y / Q, q = blockIdx.y - g * Q;
    const int words = N >> 5;
    const int word = tile * 32 + lane;
    const bool active = word < words;
    const size_t pstride = (size_t)K * words;

    if (tid < GQ_G) {
        s_list[tid] = grows[g * GQ_G + tid];
#pragma unroll
        for (int t = 0; t < T; ++t) {
            s_x[t][tid] = x[(size_t)t * K + g * GQ_G + tid];
            if (T > 1) s_tb[t][tid] = bits[(size_t)t * K + g * GQ_G + tid];
        }
    }
    if (tid < GQ_GCNT) s_cnt[tid] = gcnt_ge[g * GQ_GCNT + tid];
    __syncthreads();

    int cnt[9];
#pragma unroll
    for (int w = 1; w <= 8; ++w) cnt[w] = s_cnt[w];
    const int nnz = cnt[1];

    float acc[T][32];
    float X[T], Phi[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        X[t] = 0.f;
        Phi[t] = 0.f;
#pragma unroll
        for (int i = 0; i < 32; ++i) acc[t][i] = 0.f;
    }

    for (int p = q + Q * warp; p < nnz; p += Q * VW) {
        int b = 0;
#pragma unroll
        for (int w = 1; w <= 8; ++w) b += (p < cnt[w]);
        const int r = s_list[p];
        const uint32_t* src = planes + (size_t)(g * GQ_G + r) * words + word;
        uint32_t Wd[8], V[8];
        if (b > 4) {
#pragma unroll
            for (int j = 0; j < 8; ++j) Wd[j] = (active && j < b) ? ld_nc_u32(src + j * pstride) : 0u;
            gather<8>(Wd, V);
        } else if (b > 2) {
#pragma unroll
            for (int j = 0; j < 4; ++j) Wd[j] = (active && j < b) ? ld_nc_u32(src + j * pstride) : 0u;
            gather<4>(Wd, V);
        } else {
#pragma unroll
            for (int j = 0; j < 2; ++j) Wd[j] = (active && j < b) ? ld_nc_u32(src + j * pstride) : 0u;
            gather<2>(Wd, V);
        }
        if (T == 1) {
            const uint16_t xh = s_x[0][r];
            const float xf = __half2float(__ushort_as_half(xh));
            X[0] += xf;
            Phi[0] = fmaf(xf, (float)(0x80 >> b), Phi[0]);  // phi_b = 2^(7-b), phi_8 = 0
            accumulate_row(V, xh, acc[0]);
        } else {
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const int bt = s_tb[t][r];  // this token's own width (<= b, the union)
                if (bt == 0) continue;      // warp-uniform
                const uint16_t xh = s_x[t][r];
                const float xf = __half2float(__ushort_as_half(xh));
                X[t] += xf;
                Phi[t] = fmaf(xf, (float)(0x80 >> bt), Phi[t]);
                const uint32_t mask = 0x01010101u * ((0xFF00u >> bt) & 0xFFu);
                uint32_t Vm[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) Vm[i] = V[i] & mask;
                accumulate_row(Vm, xh, acc[t]);
            }
        }
    }

    // warp partials -> shared slots (conflict-free: consecutive lanes, stride-33 rows)
#pragma unroll
    for (int t = 0; t < T; ++t) {
        float* slot = slots + ((size_t)warp * T + t) * SLOT;
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int L = 0; L < 4; ++L) slot[(8 * L + r) * 33 + lane] = acc[t][4 * r + L];
        if (lane == 0) {
            s_X[warp][t] = X[t];
            s_Phi[warp][t] = Phi[t];
        }
    }
    __syncthreads();

    // fixed-order reduce over the 8 warps, then scale / zero-point once per (group, column)
    const int sidx = g * Q + q;
#pragma unroll
    for (int t = 0; t < T; ++t) {
        float Xs = 0.f, Ps = 0.f;
#pragma unroll
        for (int w = 0; w < VW; ++w) {
            Xs += s_X[w][t];
            Ps += s_Phi[w][t];
        }
#pragma unroll
        for (int i = 0; i < TILE_COLS / VTHREADS; ++i) {
            const int c = tid + VTHREADS * i;  // column inside the tile
            const int n = tile * TILE_COLS + c;
            if (n < N) {
                const int idx = (c & 31) * 33 + (c >> 5);
                float A = 0.f;
#pragma unroll
                for (int w = 0; w < VW; ++w) A += slots[((size_t)w * T + t) * SLOT + idx];
                const float s = __half2float(scales[(size_t)g * N + n]);
                const float z = __half2float(zeros[(size_t)g * N + n]);
                part[((size_t)sidx * T + t) * N + n] = fmaf(s, fmaf(A, CODE_SCALE, Ps), z * Xs);
            }
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

template <int T>
static int launch_main(const void* x, int K, int N, const VmmGeom& geo, const uint32_t* planes, const void* scales,
                       const void* zeros, const uint8_t* bits, const uint8_t* grows, const uint8_t* gcnt_ge,
                       float* part, cudaStream_t st) {
    const size_t smem = (size_t)VW * T * SLOT * sizeof(float);
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(vmm_main_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
            cudaSuccess)
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    dim3 grid(geo.col_tiles, (K / GQ_G) * geo.Q);
    vmm_main_kernel<T><<<grid, VTHREADS, smem, st>>>((const uint16_t*)x, K, N, geo.Q, planes, (const __half*)scales,
                                                    (const __half*)zeros, bits, grows, gcnt_ge, part);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

static int check_vmm_args(int T, int K, int N, int group) {
    if (group != GQ_G || T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32) return GRINQH_ERR_SHAPE;
    return GRINQH_OK;
}

}  // namespace gq

extern "C" size_t grinqh_vmm_workspace_bytes(int T, int K, int N) {
    if (gq::check_vmm_args(T, K, N, GQ_G) != GRINQH_OK) return 0;
    const gq::VmmGeom geo = gq::vmm_geometry(K, N);
    return (size_t)geo.S * T * N * sizeof(float);
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
    const gq::VmmGeom geo = gq::vmm_geometry(K, N);
    cudaStream_t st = (cudaStream_t)stream;
    float* part = (float*)workspace;
    switch (T) {
        case 1: return gq::launch_main<1>(x_f16, K, N, geo, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        case 2: return gq::launch_main<2>(x_f16, K, N, geo, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        case 3: return gq::launch_main<3>(x_f16, K, N, geo, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
        default: return gq::launch_main<4>(x_f16, K, N, geo, planes, scales_f16, zeros_f16, bits, grows, gcnt_ge, part, st);
    }
}

extern "C" int grinqh_vmm_reduce(int T, int K, int N, float* y, const void* workspace, size_t workspace_bytes,
                                 void* stream) {
    if (!y || !workspace) return GRINQH_ERR_NULL;
    int rc = gq::check_vmm_args(T, K, N, GQ_G);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)y | (uintptr_t)workspace) & 15) return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    const gq::VmmGeom geo = gq::vmm_geometry(K, N);
    dim3 grid((N + 127) / 128, T);
    gq::vmm_reduce_kernel<<<grid, gq::VTHREADS, 0, (cudaStream_t)stream>>>((const float*)workspace, geo.S, T, N, y);
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
