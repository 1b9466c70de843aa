// assign.cu — grinqh_assign: |x| ranking -> per-channel bit widths -> compacted row lists.
// PAPER.md:61-65 (assignment), :271 (top-p partition of the live vector); readings #2-#4.
//
// One CTA of 1024 threads.  Per token: a 32768-bin shared-memory histogram (u16 bins, padded so that
// each thread's 32 bins load conflict-free) of the 15-bit fp16 magnitudes, a block scan to find the (at most 8) histogram bins that contain a cut C_w, and an
// ordered (index-ascending) count inside those bins so that ties go to the lower index.  No sort.
// Then the union over tokens, the global (width desc, index asc) list by a 9-way stable partition,
// and the per-128-row-group lists by warp ballots.
#include "common.cuh"

namespace gq {

constexpr int AT = 1024;       // threads
constexpr int HIST_TSTRIDE = 80;                 // bytes per thread: 32 u16 bins + 16 B pad (bank spread)
constexpr int HIST_BYTES = AT * HIST_TSTRIDE;    // 80 KB
constexpr int SROW = AT + AT / 32;               // padded scratch row: entry tid lives at tid + tid/32
constexpr int SCRATCH_BYTES = 9 * SROW * 4;      // 38016
static_assert(SCRATCH_BYTES % 16 == 0 && SCRATCH_BYTES + GQ_MAX_K <= HIST_BYTES, "alias layout");
__device__ __forceinline__ int sidx(int tid) { return tid + (tid >> 5); }

struct AssignParams {
    int T, K;
    int C[10];  // C[w] = rows with width >= w (C[0] = K, C[9] = 0)
};

// inclusive block scan of one int per thread (1024 threads); red = 32-int shared scratch
__device__ __forceinline__ int block_scan_incl(int v, int* red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    if (lane == 31) red[warp] = v;
    __syncthreads();
    if (warp == 0) {
        int w = red[lane];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int o = __shfl_up_sync(0xffffffffu, w, d);
            if (lane >= d) w += o;
        }
        red[lane] = w;
    }
    __syncthreads();
    if (warp > 0) v += red[warp - 1];
    __syncthreads();
    return v;
}

// rows of `scratch` ([nrows][SROW] ints, entry tid at sidx(tid)) -> exclusive prefix over the AT
// entries, in place; totals[row] = sum.  Warp `row` scans row `row`; lane l owns entries 32l..32l+31,
// which sit at 33l + i: conflict-free.
__device__ __forceinline__ void scan_rows_excl(int* scratch, int nrows, int* totals) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp < nrows) {
        int* row = scratch + warp * SROW + lane * 33;
        int s = 0;
#pragma unroll 8
        for (int i = 0; i < 32; ++i) s += row[i];
        int incl = s;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int o = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= d) incl += o;
        }
        int run = incl - s;
#pragma unroll 8
        for (int i = 0; i < 32; ++i) {
            int v = row[i];
            row[i] = run;
            run += v;
        }
        if (lane == 31) totals[warp] = incl;
    }
}

__global__ void __launch_bounds__(AT, 1)
assign_kernel(const uint16_t* __restrict__ x, AssignParams p, uint8_t* __restrict__ bits,
              uint8_t* __restrict__ bits_union, int32_t* __restrict__ rows, int32_t* __restrict__ cnt_ge,
              uint8_t* __restrict__ grows, uint8_t* __restrict__ gcnt_ge) {
    extern __shared__ __align__(16) uint8_t smem[];
    uint8_t* hist = smem;                                                // 80 KB, u16 bins, padded per thread
    int* scratch = reinterpret_cast<int*>(smem);                         // aliases hist: [9][SROW] ints
    uint8_t* tokbits = smem + SCRATCH_BYTES;                             // aliases hist beyond scratch: K bytes
    uint16_t* keys = reinterpret_cast<uint16_t*>(smem + HIST_BYTES);     // K u16
    uint8_t* ubits = smem + HIST_BYTES + GQ_MAX_K * 2;                   // K u8
    __shared__ int red[32];
    __shared__ int s_cutbin[9], s_take[9], s_tot[9];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = p.K;
    const int chunk = (K + AT - 1) / AT;
    const int k0 = min(K, tid * chunk), k1 = min(K, k0 + chunk);

    for (int t = 0; t < p.T; ++t) {
        // A. clear histogram
        {
            uint4* h4 = reinterpret_cast<uint4*>(hist);
            for (int i = tid; i < HIST_BYTES / 16; i += AT) h4[i] = make_uint4(0, 0, 0, 0);
            if (tid < 9) {
                s_cutbin[tid] = 0x8000;  // above every key: no channel reaches this width
                s_take[tid] = 0;
            }
        }
        __syncthreads();
        // B. keys + histogram
        for (int k = tid; k < K; k += AT) {
            uint16_t m = x[(size_t)t * K + k] & 0x7FFFu;
            keys[k] = m;
            // u16 bin inside a 32-bit word; a bin never exceeds K <= 32768, so no carry into its neighbour
            atomicAdd(reinterpret_cast<uint32_t*>(hist + (m >> 5) * HIST_TSTRIDE + ((m & 31) >> 1) * 4),
                      1u << ((m & 1) * 16));
        }
        __syncthreads();
        // C. per-thread sum of its 32 bins, block scan -> number of keys in higher bins
        uint32_t loc[32];
        {
            const uint4* h4 = reinterpret_cast<const uint4*>(hist + tid * HIST_TSTRIDE);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 v = h4[i];
                loc[8 * i + 0] = v.x & 0xFFFFu; loc[8 * i + 1] = v.x >> 16;
                loc[8 * i + 2] = v.y & 0xFFFFu; loc[8 * i + 3] = v.y >> 16;
                loc[8 * i + 4] = v.z & 0xFFFFu; loc[8 * i + 5] = v.z >> 16;
                loc[8 * i + 6] = v.w & 0xFFFFu; loc[8 * i + 7] = v.w >> 16;
            }
        }
        int tsum = 0;
#pragma unroll
        for (int i = 0; i < 32; ++i) tsum += (int)loc[i];
        const int incl = block_scan_incl(tsum, red);
        const int above = K - incl;  // keys strictly above this thread's bins
        // D. locate cut bins
        bool mine = false;
#pragma unroll
        for (int w = 1; w <= 8; ++w) mine |= (above < p.C[w]) && (p.C[w] <= above + tsum);
        if (mine) {
            int G = above;
#pragma unroll
            for (int i = 31; i >= 0; --i) {
                const int h = (int)loc[i];
                if (h > 0) {
#pragma unroll
                    for (int w = 1; w <= 8; ++w)
                        if (G < p.C[w] && p.C[w] <= G + h) {
                            s_cutbin[w] = tid * 32 + i;
                            s_take[w] = p.C[w] - G;
                        }
                }
                G += h;
            }
        }
        __syncthreads();  // hist no longer needed: scratch / tokbits alias it from here on
        int cutbin[9], take[9];
#pragma unroll
        for (int w = 1; w <= 8; ++w) {
            cutbin[w] = s_cutbin[w];
            take[w] = s_take[w];
        }
        // E. ordered tie counts inside the cut bins
        {
            int cnt[9];
#pragma unroll
            for (int w = 1; w <= 8; ++w) cnt[w] = 0;
            for (int k = k0; k < k1; ++k) {
                const int m = keys[k];
#pragma unroll
                for (int w = 1; w <= 8; ++w) cnt[w] += (m == cutbin[w]);
            }
#pragma unroll
            for (int w = 1; w <= 8; ++w) scratch[(w - 1) * SROW + sidx(tid)] = cnt[w];
        }
        __syncthreads();
        scan_rows_excl(scratch, 8, s_tot);
        __syncthreads();
        // G. widths
        {
            int run[9];
#pragma unroll
            for (int w = 1; w <= 8; ++w) run[w] = scratch[(w - 1) * SROW + sidx(tid)];
            for (int k = k0; k < k1; ++k) {
                const int m = keys[k];
                int b = 0;
#pragma unroll
                for (int w = 1; w <= 8; ++w) {
                    const bool eq = (m == cutbin[w]);
                    b += (m > cutbin[w]) || (eq && run[w] < take[w]);
                    run[w] += eq;
                }
                tokbits[k] = (uint8_t)b;
                ubits[k] = (t == 0) ? (uint8_t)b : max(ubits[k], (uint8_t)b);
            }
        }
        __syncthreads();
        {
            const uint4* src = reinterpret_cast<const uint4*>(tokbits);
            uint4* dst = reinterpret_cast<uint4*>(bits + (size_t)t * K);
            for (int i = tid; i < K / 16; i += AT) dst[i] = src[i];
        }
        __syncthreads();
    }

    // H. union out
    {
        const uint4* src = reinterpret_cast<const uint4*>(ubits);
        uint4* dst = reinterpret_cast<uint4*>(bits_union);
        for (int i = tid; i < K / 16; i += AT) dst[i] = src[i];
    }
    // I. global list: stable 9-way partition, width descending, index ascending
    {
        int cnt[9];
#pragma unroll
        for (int w = 0; w < 9; ++w) cnt[w] = 0;
        for (int k = k0; k < k1; ++k) {
            const int b = ubits[k];
#pragma unroll
            for (int w = 0; w < 9; ++w) cnt[w] += (b == w);
        }
#pragma unroll
        for (int w = 0; w < 9; ++w) scratch[w * SROW + sidx(tid)] = cnt[w];
    }
    __syncthreads();
    scan_rows_excl(scratch, 9, s_tot);
    __syncthreads();
    {
        int base[9], acc = 0;
#pragma unroll
        for (int w = 8; w >= 0; --w) {
            base[w] = acc + scratch[w * SROW + sidx(tid)];
            acc += s_tot[w];
        }
        for (int k = k0; k < k1; ++k) {
            const int b = ubits[k];
            int pos = 0;
#pragma unroll
            for (int w = 0; w < 9; ++w)
                if (b == w) {
                    pos = base[w];
                    base[w]++;
                }
            rows[pos] = k;
        }
        if (tid < 10) {
            int c = 0;
            for (int w = 8; w >= tid; --w) c += s_tot[w];
            cnt_ge[tid] = (tid == 9) ? 0 : c;
        }
    }
    // J. per-group lists: one warp per 128-row group
    for (int g = warp; g < K / GQ_G; g += AT / 32) {
        int b[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) b[r] = ubits[g * GQ_G + lane + 32 * r];
        int base = 0, myge = 0;
#pragma unroll
        for (int w = 8; w >= 0; --w) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const uint32_t m = __ballot_sync(0xffffffffu, b[r] == w);
                if (b[r] == w) grows[g * GQ_G + base + __popc(m & ((1u << lane) - 1u))] = (uint8_t)(lane + 32 * r);
                base += __popc(m);
            }
            if (lane == w) myge = base;
        }
        if (lane < GQ_GCNT) gcnt_ge[g * GQ_GCNT + lane] = (uint8_t)(lane <= 8 ? myge : 0);
    }
}

}  // namespace gq

extern "C" size_t grinqh_assign_workspace_bytes(int T, int K) {
    (void)T;
    (void)K;
    return 0;  // everything lives in shared memory; the argument is kept for ABI stability
}

extern "C" int grinqh_assign(const void* x_f16, int T, int K, const uint32_t counts[9], uint8_t* bits,
                             uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge,
                             void* workspace, size_t workspace_bytes, void* stream) {
    (void)workspace;
    (void)workspace_bytes;
    if (!x_f16 || !counts || !bits || !bits_union || !rows || !cnt_ge || !grows || !gcnt_ge) return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || K % GQ_G || K > GQ_MAX_K) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_f16 | (uintptr_t)bits | (uintptr_t)bits_union | (uintptr_t)rows | (uintptr_t)cnt_ge |
         (uintptr_t)grows | (uintptr_t)gcnt_ge) & 15)
        return GRINQH_ERR_ALIGN;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    gq::AssignParams p;
    p.T = T;
    p.K = K;
    p.C[9] = 0;
    for (int w = 8; w >= 0; --w) p.C[w] = p.C[w + 1] + (int)counts[w];
    const size_t smem = (size_t)gq::HIST_BYTES + (size_t)GQ_MAX_K * 2 + (size_t)GQ_MAX_K;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(gq::assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
            cudaSuccess)
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    gq::assign_kernel<<<1, gq::AT, smem, (cudaStream_t)stream>>>((const uint16_t*)x_f16, p, bits, bits_union, rows,
                                                                cnt_ge, grows, gcnt_ge);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
