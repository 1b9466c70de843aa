// assign.cu — grinqh_assign (rank form) and grinqh_assign_thresholds (the paper's threshold form):
// |x| -> per-channel bit widths -> compacted row lists.
// PAPER.md:61-65 (assignment), :271 (top-p partition of the live vector); readings #2-#4.
//
// A small grid of independent CTAs, no cluster, no exchange between CTAs: every CTA repeats the cheap global steps on
// its own copy and writes the outputs of its own groups.
//   select   per token the cut keys of the level mix (select.cuh: one shared-memory atomic per key into a 15-bit
//            histogram, block scan, the owning warp scans the cut's bins) — or the given thresholds;
//   ties     a cut that splits a run of equal keys: equal keys per group (16 lanes = one group, shuffles), exclusive
//            prefix over the groups = ordered tie offsets (ties go to the lower index);
//   widths   one warp per 128-row group: widths4 per token, union over tokens, partition128 by (width desc, index
//            asc) -> bits, bits_union, grows, gcnt_ge, gsched of the CTA's own groups; the nine per-width counts of
//            EVERY group stay in shared memory;
//   rows     a scan over the groups' per-width counts (warp w scans width w) places each group's runs in the global
//            list `rows`; cnt_ge are the totals.
// Any output pointer may be NULL (grinqh_vmm needs gsched only): its work is skipped.
#include "common.cuh"
#include "select.cuh"

namespace gq {

constexpr int AT = 512;   // threads per CTA
constexpr int AW = AT / 32;
constexpr int AMAXG = GQ_MAX_K / GQ_G;  // 256 groups

struct AssignOut {
    uint8_t* bits;
    uint8_t* bits_union;
    int32_t* rows;
    int32_t* cnt_ge;
    uint8_t* grows;
    uint8_t* gcnt_ge;
    uint32_t* gsched;
};

__global__ void __launch_bounds__(AT, 1)
assign_kernel(const uint16_t* __restrict__ x, int T, int K, CutParams cp, int use_thr, AssignOut o) {
    extern __shared__ __align__(16) uint8_t smem[];
    uint32_t* hist = reinterpret_cast<uint32_t*>(smem);                       // 64 KB
    uint16_t* skeys = reinterpret_cast<uint16_t*>(smem + 65536);               // K x 2 bytes
    uint16_t* s_tie = reinterpret_cast<uint16_t*>(smem + 65536 + GQ_MAX_K * 2);  // [T][groups][8]
    __shared__ __align__(16) uint8_t s_gcnt[AMAXG][GQ_GCNT];  // ge[0..9] of every group's union widths
    __shared__ uint16_t s_off[AMAXG][10];                     // rows of width w in lower groups
    __shared__ int s_tot[10];
    __shared__ __align__(16) TokenCuts s_tc[GRINQH_MAX_T];
    __shared__ SelectScratch s_sel;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int groups = K / GQ_G, nd = cp.nd;
    const int gpc = (groups + gridDim.x - 1) / gridDim.x;  // groups per CTA
    const int g_lo = blockIdx.x * gpc, g_hi = min(groups, g_lo + gpc);

    pdl_launch_dependents();
    if (!use_thr) {
        uint4* z = reinterpret_cast<uint4*>(hist);
        for (int i = tid; i < 4096; i += AT) z[i] = make_uint4(0, 0, 0, 0);
        __syncthreads();
    }
    pdl_wait();  // x may come from the previous kernel, and the outputs may still be read by it

#pragma unroll 1
    for (int t = 0; t < T; ++t) {
        if (!use_thr) {
            rank_select<AT>(x + (size_t)t * K, skeys, K, nd, cp.Cd, hist, t + 1 < T, &s_sel, &s_tc[t]);
        } else {
            if (tid < 8) {
                s_tc[t].thr[tid] = cp.thr[tid];
                s_tc[t].take[tid] = 0;
                s_tc[t].hh[tid] = 0;
            }
            if (tid == 0) {
                s_tc[t].split = 0;
                s_tc[t].nd = nd;
            }
            __syncthreads();
        }
        const uint32_t split = s_tc[t].split;
        if (split) {
            uint16_t* tie = s_tie + (size_t)t * groups * 8;
#pragma unroll 1
            for (int c0 = warp * 32; c0 < (K >> 3); c0 += AT) {  // (warp-uniform bounds: every lane shuffles)
                const int c = c0 + lane;
                const bool valid = c < (K >> 3);
                const uint4 kv = valid ? reinterpret_cast<const uint4*>(skeys)[c] : make_uint4(~0u, ~0u, ~0u, ~0u);
                const uint32_t kw[4] = {kv.x, kv.y, kv.z, kv.w};
                uint32_t pk[2] = {0u, 0u};  // equal counts of cuts 0..3 and 4..7, 8 bits each
#pragma unroll
                for (int d = 0; d < 8; ++d) {
                    if (d < nd) {
                        const uint32_t th = (uint32_t)s_tc[t].thr[d];
                        uint32_t ce = 0;
#pragma unroll
                        for (int j = 0; j < 8; ++j) ce += (((kw[j >> 1] >> (16 * (j & 1))) & 0x7FFFu) == th) ? 1u : 0u;
                        pk[d >> 2] += ce << (8 * (d & 3));
                    }
                }
#pragma unroll
                for (int s = 8; s >= 1; s >>= 1) {
                    pk[0] += __shfl_xor_sync(0xffffffffu, pk[0], s);
                    if (nd > 4) pk[1] += __shfl_xor_sync(0xffffffffu, pk[1], s);
                }
                if (valid && (lane & 15) < 8) {
                    const int d = lane & 15;
                    tie[(c >> 4) * 8 + d] = (uint16_t)((pk[d >> 2] >> (8 * (d & 3))) & 0xFFu);
                }
            }
            __syncthreads();
#pragma unroll 1
            for (int d = warp; d < nd; d += AW) {
                int v[8], inc[8];
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const int g = 32 * r + lane;
                    v[r] = (g < groups) ? (int)tie[g * 8 + d] : 0;
                    inc[r] = (32 * r < groups) ? warp_incl_scan_i(v[r], lane) : 0;
                }
                int carry = 0;
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    const int g = 32 * r + lane;
                    if (g < groups) tie[g * 8 + d] = (uint16_t)(carry + inc[r] - v[r]);
                    carry += __shfl_sync(0xffffffffu, inc[r], 31);
                }
            }
            __syncthreads();
        }
    }

    // ---- widths, union and per-group lists: every group's counts, the outputs of the CTA's own groups
    const bool need_all = o.rows != nullptr || o.cnt_ge != nullptr;  // the global list needs every group's counts
#pragma unroll 1
    for (int g = need_all ? warp : g_lo + warp; g < (need_all ? groups : g_hi); g += AW) {
        const bool mine = g >= g_lo && g < g_hi;
        const int go = g * GQ_G + 4 * lane;
        uint2 xv[GRINQH_MAX_T];
        int bt[GRINQH_MAX_T][4], bu[4] = {0, 0, 0, 0};
#pragma unroll
        for (int t = 0; t < GRINQH_MAX_T; ++t)
            if (t < T) {
                xv[t] = *reinterpret_cast<const uint2*>(x + (size_t)t * K + go);
                int m[4];
                keys4(xv[t], m);
                widths4(m, &s_tc[t], cp.mult, nd, s_tie + ((size_t)t * groups + g) * 8, lane, bt[t]);
#pragma unroll
                for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], bt[t][i]);
            }
        int pos[4], ge[10];
        partition128(bu, lane, pos, ge);
        int myge = 0;
#pragma unroll
        for (int c = 0; c <= 9; ++c)
            if (lane == c) myge = ge[c];
        const uint8_t gv = (uint8_t)(lane <= 9 ? myge : 0);
        if (lane < GQ_GCNT) s_gcnt[g][lane] = gv;
        if (!mine) continue;
        if (o.gcnt_ge && lane < GQ_GCNT) o.gcnt_ge[(size_t)g * GQ_GCNT + lane] = gv;
        if (o.bits_union)
            *reinterpret_cast<uint32_t*>(o.bits_union + go) =
                (uint32_t)bu[0] | ((uint32_t)bu[1] << 8) | ((uint32_t)bu[2] << 16) | ((uint32_t)bu[3] << 24);
#pragma unroll
        for (int t = 0; t < GRINQH_MAX_T; ++t)
            if (t < T) {
                if (o.bits)
                    *reinterpret_cast<uint32_t*>(o.bits + (size_t)t * K + go) =
                        (uint32_t)bt[t][0] | ((uint32_t)bt[t][1] << 8) | ((uint32_t)bt[t][2] << 16) | ((uint32_t)bt[t][3] << 24);
                if (o.gsched) {
                    const uint32_t xq[4] = {xv[t].x & 0xFFFFu, xv[t].x >> 16, xv[t].y & 0xFFFFu, xv[t].y >> 16};
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        o.gsched[(size_t)t * K + g * GQ_G + pos[i]] =
                            (uint32_t)(4 * lane + i) | ((uint32_t)bt[t][i] << 8) | ((uint32_t)bu[i] << 12) | (xq[i] << 16);
                }
            }
        if (o.grows) {
#pragma unroll
            for (int i = 0; i < 4; ++i) o.grows[(size_t)g * GQ_G + pos[i]] = (uint8_t)(4 * lane + i);
        }
    }
    if (!need_all) return;
    __syncthreads();

    // ---- where each group's run of every width starts in the global list: warp w scans width w over the groups
#pragma unroll 1
    for (int w = warp; w <= 8; w += AW) {
        int v[8], inc[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int g = 32 * r + lane;
            v[r] = (g < groups) ? (int)s_gcnt[g][w] - (int)s_gcnt[g][w + 1] : 0;
            inc[r] = (32 * r < groups) ? warp_incl_scan_i(v[r], lane) : 0;
        }
        int carry = 0;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int g = 32 * r + lane;
            if (g < groups) s_off[g][w] = (uint16_t)(carry + inc[r] - v[r]);
            carry += __shfl_sync(0xffffffffu, inc[r], 31);
        }
        if (lane == 0) s_tot[w] = carry;
    }
    __syncthreads();
    int cbase[9];  // rows of larger width
    {
        int acc = 0;
#pragma unroll
        for (int c = 8; c >= 0; --c) {
            cbase[c] = acc;
            acc += s_tot[c];
        }
    }
    if (o.cnt_ge && blockIdx.x == 0 && tid < 10) o.cnt_ge[tid] = (tid == 9) ? 0 : cbase[tid] + s_tot[tid];
    if (!o.rows) return;
    // ---- global list (width desc, index asc): the CTA's own groups again (their widths are cheap to redo)
#pragma unroll 1
    for (int g = g_lo + warp; g < g_hi; g += AW) {
        const int go = g * GQ_G + 4 * lane;
        int bu[4] = {0, 0, 0, 0};
#pragma unroll
        for (int t = 0; t < GRINQH_MAX_T; ++t)
            if (t < T) {
                int m[4], b[4];
                keys4(*reinterpret_cast<const uint2*>(x + (size_t)t * K + go), m);
                widths4(m, &s_tc[t], cp.mult, nd, s_tie + ((size_t)t * groups + g) * 8, lane, b);
#pragma unroll
                for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], b[i]);
            }
        int pos[4], ge[10];
        partition128(bu, lane, pos, ge);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            int dst = 0;
#pragma unroll
            for (int c = 0; c <= 8; ++c)
                if (bu[i] == c) dst = cbase[c] + (int)s_off[g][c] + (pos[i] - ge[c + 1]);
            o.rows[dst] = g * GQ_G + 4 * lane + i;
        }
    }
}

static int check_assign_args(const void* x_f16, int T, int K, const void* spec, const AssignOut& o) {
    if (!x_f16 || !spec) return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || K % GQ_G || K > GQ_MAX_K) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_f16 | (uintptr_t)o.bits | (uintptr_t)o.bits_union | (uintptr_t)o.rows | (uintptr_t)o.cnt_ge |
         (uintptr_t)o.grows | (uintptr_t)o.gcnt_ge | (uintptr_t)o.gsched) & 15)
        return GRINQH_ERR_ALIGN;
    return GRINQH_OK;
}

static int launch_assign(const CutParams& cp, int use_thr, const void* x_f16, int T, int K, const AssignOut& o,
                         void* stream) {
    const int groups = K / GQ_G;
    // CTAs: each repeats the select and the counting of all groups; the outputs are split.  4 groups per CTA keeps a
    // CTA's own part at one group per warp or less.
    int nc = (groups + 3) / 4;
    if (nc > 32) nc = 32;
    if (nc < 1) nc = 1;
    const size_t smem = 65536 + (size_t)GQ_MAX_K * 2 + (size_t)T * groups * 16;
    if (cudaFuncSetAttribute(assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return GRINQH_ERR_CUDA;  // (the attribute belongs to the device: set on every launch)
    const cudaError_t e = launch_pdl(assign_kernel, dim3(nc), dim3(AT), smem, (cudaStream_t)stream,
                                     (const uint16_t*)x_f16, T, K, cp, use_thr, o);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
}  // namespace gq

extern "C" size_t grinqh_assign_workspace_bytes(int T, int K) {
    (void)T;
    (void)K;
    return 0;  // everything lives in shared memory; the call and its workspace arguments are kept for ABI stability
}

extern "C" int grinqh_assign(const void* x_f16, int T, int K, const uint32_t counts[9], uint8_t* bits,
                             uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge,
                             uint32_t* gsched, void* workspace, size_t workspace_bytes, void* stream) {
    (void)workspace;
    (void)workspace_bytes;
    const gq::AssignOut o{bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched};
    int rc = gq::check_assign_args(x_f16, T, K, counts, o);
    if (rc != GRINQH_OK) return rc;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    return gq::launch_assign(gq::cuts_from_counts(counts), 0, x_f16, T, K, o, stream);
}

extern "C" int grinqh_assign_thresholds(const void* x_f16, int T, int K, const uint16_t theta[9], uint8_t* bits,
                                        uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows,
                                        uint8_t* gcnt_ge, uint32_t* gsched, void* stream) {
    const gq::AssignOut o{bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched};
    int rc = gq::check_assign_args(x_f16, T, K, theta, o);
    if (rc != GRINQH_OK) return rc;
    for (int w = 1; w <= 8; ++w)
        if (theta[w] > 0x8000 || (w > 1 && theta[w] < theta[w - 1])) return GRINQH_ERR_MIX;
    return gq::launch_assign(gq::cuts_from_thetas(theta), 1, x_f16, T, K, o, stream);
}
