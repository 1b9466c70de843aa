// assign.cu — grinqh_assign: |x| ranking -> per-channel bit widths -> compacted row lists (v2).
// PAPER.md:61-65 (assignment), :271 (top-p partition of the live vector); readings #2-#4.
//
// One CTA of 1024 threads, no sort.  Per token a two-level radix select on the 15-bit fp16 magnitude:
//   level 1  256-bin histogram of key >> 7 (8 sub-histograms against atomic contention); one warp scans it
//            from the top and finds, for each of the (at most 8) cuts C_w, the bin that contains it;
//   level 2  128-bin histograms of key & 127 restricted to those bins; warp w finds the exact cut key thr_w,
//            how many of the keys equal to thr_w are still inside (take_w), and whether the cut splits a run
//            of equal keys.
// Widths are then b = #{w : key >= thr_w}.  Only if some cut splits a tie run (ties go to the lower index) an
// ordered count of the equal keys (per 128-row group, then a scan over groups) decides them.
// Lists: one warp per 128-row group partitions its rows by (width desc, index asc) with ballots -> grows,
// gcnt_ge, gsched; a scan over the groups' per-width counts places every group's runs in the global `rows`.
#include "common.cuh"

namespace gq {

constexpr int AT = 1024;  // threads
constexpr int AWARPS = AT / 32;
constexpr int NSUB = 8;
constexpr int MAXG = GQ_MAX_K / GQ_G;  // 256 groups

struct AssignParams {
    int T, K;
    int C[10];  // C[w] = rows with width >= w (C[0] = K, C[9] = 0)
};

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// tab[g][col], g < groups: exclusive prefix over g, in place; returns the total to lane 31's caller via *tot.
// One warp per column; lane l owns groups 8l..8l+7.
__device__ __forceinline__ void scan_groups(uint16_t (*tab)[10], int col, int groups, int lane, int* tot) {
    int v[8], s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int g = 8 * lane + i;
        v[i] = (g < groups) ? tab[g][col] : 0;
        s += v[i];
    }
    const int incl = warp_incl_scan(s, lane);
    int run = incl - s;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int g = 8 * lane + i;
        if (g < groups) tab[g][col] = (uint16_t)run;
        run += v[i];
    }
    if (lane == 31) *tot = incl;
}

__global__ void __launch_bounds__(AT, 1)
assign_kernel(const uint16_t* __restrict__ x, AssignParams p, uint8_t* __restrict__ bits,
              uint8_t* __restrict__ bits_union, int32_t* __restrict__ rows, int32_t* __restrict__ cnt_ge,
              uint8_t* __restrict__ grows, uint8_t* __restrict__ gcnt_ge, uint32_t* __restrict__ gsched) {
    extern __shared__ __align__(16) uint8_t smem[];
    uint16_t* keys = reinterpret_cast<uint16_t*>(smem);  // K u16 (current token); later aliased by glist (K u8)
    uint8_t* glist = smem;
    uint8_t* ubits = smem + (size_t)p.K * 2;             // K u8, union of the token widths
    __shared__ uint32_t hist1[NSUB][256];
    __shared__ uint32_t hist2[8][128];
    __shared__ uint16_t tab[MAXG][10];
    __shared__ int s_B[9], s_above[9], s_thr[9], s_take[9], s_split[9], s_tot[10];
    __shared__ int s_anysplit;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = p.K, groups = K / GQ_G;
    const uint32_t lt_mask = (1u << lane) - 1u;

    for (int t = 0; t < p.T; ++t) {
        // ---- P0: clear, keys, level-1 histogram
        for (int i = tid; i < NSUB * 256; i += AT) (&hist1[0][0])[i] = 0;
        (&hist2[0][0])[tid] = 0;
        if (tid < 9) {
            s_B[tid] = -1;
            s_above[tid] = 0;
            s_thr[tid] = 0x8000;  // above every key: no channel reaches this width
            s_take[tid] = 0;
            s_split[tid] = 0;
        }
        if (tid == 0) s_anysplit = 0;
        __syncthreads();
        {
            const uint32_t* x2 = reinterpret_cast<const uint32_t*>(x + (size_t)t * K);
            uint32_t* h = hist1[warp & (NSUB - 1)];
            for (int i = tid; i < K / 2; i += AT) {
                const uint32_t v = x2[i] & 0x7FFF7FFFu;
                reinterpret_cast<uint32_t*>(keys)[i] = v;
                atomicAdd(&h[(v & 0xFFFFu) >> 7], 1u);
                atomicAdd(&h[v >> 23], 1u);
            }
        }
        __syncthreads();
        // ---- P1: warp 0 scans the 256 bins from the top and locates the bin of every cut
        if (warp == 0) {
            int h[8], s = 0;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const int bin = 255 - 8 * lane - i;
                int c = 0;
#pragma unroll
                for (int u = 0; u < NSUB; ++u) c += (int)hist1[u][bin];
                h[i] = c;
                s += c;
            }
            const int above = warp_incl_scan(s, lane) - s;
#pragma unroll
            for (int w = 1; w <= 8; ++w) {
                const int Cw = p.C[w];
                if (Cw > 0 && above < Cw && Cw <= above + s) {
                    int run = above;
                    bool done = false;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        if (!done && Cw <= run + h[i]) {
                            s_B[w] = 255 - 8 * lane - i;
                            s_above[w] = run;
                            done = true;
                        }
                        run += h[i];
                    }
                }
            }
        }
        __syncthreads();
        // ---- P2: level-2 histograms inside the cut bins (cuts that share a bin share histogram `slot`)
        int B[9], slot[9];
#pragma unroll
        for (int w = 1; w <= 8; ++w) B[w] = s_B[w];
#pragma unroll
        for (int w = 1; w <= 8; ++w) {
            slot[w] = w;
#pragma unroll
            for (int v = w - 1; v >= 1; --v)
                if (B[v] == B[w]) slot[w] = v;
        }
        for (int i = tid; i < K; i += AT) {
            const int m = keys[i];
            const int top = m >> 7;
#pragma unroll
            for (int w = 1; w <= 8; ++w)
                if (top == B[w] && slot[w] == w) atomicAdd(&hist2[w - 1][m & 127], 1u);
        }
        __syncthreads();
        // ---- P3: warp w-1 finds the exact cut key of cut w
        if (warp < 8) {
            const int w = warp + 1;
            int Bw = -1, sl = 1, ab = 0;
#pragma unroll
            for (int v = 1; v <= 8; ++v)
                if (v == w) { Bw = B[v]; sl = slot[v]; }
            ab = s_above[w];
            if (Bw >= 0) {
                const int need = p.C[w] - ab;  // 1 <= need <= keys in bin Bw
                int h[4], s = 0;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    h[i] = (int)hist2[sl - 1][127 - 4 * lane - i];
                    s += h[i];
                }
                const int above = warp_incl_scan(s, lane) - s;
                if (above < need && need <= above + s) {
                    int run = above;
                    bool done = false;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        if (!done && need <= run + h[i]) {
                            s_thr[w] = (Bw << 7) | (127 - 4 * lane - i);
                            s_take[w] = need - run;
                            if (need - run < h[i]) {
                                s_split[w] = 1;
                                s_anysplit = 1;
                            }
                            done = true;
                        }
                        run += h[i];
                    }
                }
            }
        }
        __syncthreads();
        int thr[9], take[9], split[9];
#pragma unroll
        for (int w = 1; w <= 8; ++w) {
            thr[w] = s_thr[w];
            take[w] = s_take[w];
            split[w] = s_split[w];
        }
        const bool anysplit = s_anysplit != 0;
        if (anysplit) {
            // ---- a cut splits a run of equal keys: ordered (index-ascending) count of the equal keys
            for (int g = warp; g < groups; g += AWARPS) {
                const uint2 kv = *reinterpret_cast<const uint2*>(keys + g * GQ_G + 4 * lane);
                const int m[4] = {(int)(kv.x & 0xFFFF), (int)(kv.x >> 16), (int)(kv.y & 0xFFFF), (int)(kv.y >> 16)};
#pragma unroll
                for (int w = 1; w <= 8; ++w)
                    if (split[w]) {
                        int c = 0;
#pragma unroll
                        for (int i = 0; i < 4; ++i) c += (m[i] == thr[w]);
                        c = __reduce_add_sync(0xffffffffu, c);
                        if (lane == 0) tab[g][w] = (uint16_t)c;
                    }
            }
            __syncthreads();
            if (warp < 8 && split[warp + 1]) {
                int dummy;
                scan_groups(tab, warp + 1, groups, lane, &dummy);
            }
            __syncthreads();
        }
        // ---- P4: widths of this token
        for (int g = warp; g < groups; g += AWARPS) {
            const uint2 kv = *reinterpret_cast<const uint2*>(keys + g * GQ_G + 4 * lane);
            const int m[4] = {(int)(kv.x & 0xFFFF), (int)(kv.x >> 16), (int)(kv.y & 0xFFFF), (int)(kv.y >> 16)};
            int b[4] = {0, 0, 0, 0};
#pragma unroll
            for (int w = 1; w <= 8; ++w) {
                if (!split[w]) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) b[i] += (m[i] >= thr[w]);
                } else {
                    bool eq[4];
                    int below = tab[g][w];  // equal keys in earlier groups
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        eq[i] = (m[i] == thr[w]);
                        below += __popc(__ballot_sync(0xffffffffu, eq[i]) & lt_mask);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        b[i] += (m[i] > thr[w]) || (eq[i] && below < take[w]);
                        below += eq[i];
                    }
                }
            }
            const uint32_t packed = (uint32_t)b[0] | ((uint32_t)b[1] << 8) | ((uint32_t)b[2] << 16) | ((uint32_t)b[3] << 24);
            *reinterpret_cast<uint32_t*>(bits + (size_t)t * K + g * GQ_G + 4 * lane) = packed;
            uint32_t* u = reinterpret_cast<uint32_t*>(ubits + g * GQ_G + 4 * lane);
            *u = (t == 0) ? packed : __vmaxu4(*u, packed);
        }
        __syncthreads();
    }

    // ---- P5: per-group lists (keys are dead: glist aliases them)
    __shared__ __align__(16) uint8_t gcs[MAXG][GQ_GCNT];
    for (int g = warp; g < groups; g += AWARPS) {
        const uint32_t bu4 = *reinterpret_cast<const uint32_t*>(ubits + g * GQ_G + 4 * lane);
        *reinterpret_cast<uint32_t*>(bits_union + g * GQ_G + 4 * lane) = bu4;
        int bu[4], pos[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) bu[i] = (bu4 >> (8 * i)) & 0xFF;
        int base = 0, myge = 0, myn = 0;
#pragma unroll
        for (int c = 8; c >= 0; --c) {
            int lower = base, n = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint32_t m = __ballot_sync(0xffffffffu, bu[i] == c);
                lower += __popc(m & lt_mask);
                n += __popc(m);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (bu[i] == c) pos[i] = lower++;
            base += n;
            if (lane == c) {
                myge = base;
                myn = n;
            }
        }
        if (lane < GQ_GCNT) {
            const uint8_t v = (uint8_t)(lane <= 8 ? myge : 0);
            gcnt_ge[g * GQ_GCNT + lane] = v;
            gcs[g][lane] = v;
        }
        if (lane < 9) tab[g][lane] = (uint16_t)myn;
#pragma unroll
        for (int i = 0; i < 4; ++i) glist[g * GQ_G + pos[i]] = (uint8_t)(4 * lane + i);
        for (int t = 0; t < p.T; ++t) {
            const uint32_t bt4 = *reinterpret_cast<const uint32_t*>(bits + (size_t)t * K + g * GQ_G + 4 * lane);
            const uint2 xv = *reinterpret_cast<const uint2*>(x + (size_t)t * K + g * GQ_G + 4 * lane);
            const uint32_t xs[4] = {xv.x & 0xFFFFu, xv.x >> 16, xv.y & 0xFFFFu, xv.y >> 16};
#pragma unroll
            for (int i = 0; i < 4; ++i)
                gsched[(size_t)t * K + g * GQ_G + pos[i]] = (uint32_t)(4 * lane + i) | (((bt4 >> (8 * i)) & 0xFFu) << 8) |
                                                            ((uint32_t)bu[i] << 12) | (xs[i] << 16);
        }
        __syncwarp();
        *reinterpret_cast<uint32_t*>(grows + g * GQ_G + 4 * lane) =
            *reinterpret_cast<const uint32_t*>(glist + g * GQ_G + 4 * lane);
    }
    __syncthreads();
    // ---- P6: where each group's run of every width starts in the global list
    if (warp < 9) scan_groups(tab, warp, groups, lane, &s_tot[warp]);
    __syncthreads();
    // ---- P7: global list (width desc, index asc) and cnt_ge
    int cbase[9];
    {
        int acc = 0;
#pragma unroll
        for (int c = 8; c >= 0; --c) {
            cbase[c] = acc;
            acc += s_tot[c];
        }
    }
    if (tid < 10) cnt_ge[tid] = (tid == 9) ? 0 : cbase[tid] + s_tot[tid];
    for (int g = warp; g < groups; g += AWARPS) {
        const uint4 cv = *reinterpret_cast<const uint4*>(gcs[g]);
        const int cge[10] = {(int)(cv.x & 0xFF), (int)((cv.x >> 8) & 0xFF), (int)((cv.x >> 16) & 0xFF), (int)(cv.x >> 24),
                             (int)(cv.y & 0xFF), (int)((cv.y >> 8) & 0xFF), (int)((cv.y >> 16) & 0xFF), (int)(cv.y >> 24),
                             (int)(cv.z & 0xFF), 0};
        const uint32_t l4 = *reinterpret_cast<const uint32_t*>(glist + g * GQ_G + 4 * lane);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int pp = 4 * lane + i;
            int dst = 0;
#pragma unroll
            for (int c = 0; c <= 8; ++c)
                if (pp < cge[c] && pp >= cge[c + 1]) dst = cbase[c] + (int)tab[g][c] + (pp - cge[c + 1]);
            rows[dst] = g * GQ_G + (int)((l4 >> (8 * i)) & 0xFF);
        }
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
                             uint32_t* gsched, void* workspace, size_t workspace_bytes, void* stream) {
    (void)workspace;
    (void)workspace_bytes;
    if (!x_f16 || !counts || !bits || !bits_union || !rows || !cnt_ge || !grows || !gcnt_ge || !gsched)
        return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || K % GQ_G || K > GQ_MAX_K) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_f16 | (uintptr_t)bits | (uintptr_t)bits_union | (uintptr_t)rows | (uintptr_t)cnt_ge |
         (uintptr_t)grows | (uintptr_t)gcnt_ge | (uintptr_t)gsched) & 15)
        return GRINQH_ERR_ALIGN;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    gq::AssignParams p;
    p.T = T;
    p.K = K;
    p.C[9] = 0;
    for (int w = 8; w >= 0; --w) p.C[w] = p.C[w + 1] + (int)counts[w];
    const size_t smem = (size_t)K * 3;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(gq::assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GQ_MAX_K * 3) !=
            cudaSuccess)
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    gq::assign_kernel<<<1, gq::AT, smem, (cudaStream_t)stream>>>((const uint16_t*)x_f16, p, bits, bits_union, rows,
                                                                cnt_ge, grows, gcnt_ge, gsched);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
