// assign.cu — grinqh_assign (rank form) and grinqh_assign_thresholds (the paper's threshold form):
// |x| -> per-channel bit widths -> compacted row lists.
// PAPER.md:61-65 (assignment), :271 (top-p partition of the live vector); readings #2-#4.
//
// One thread-block cluster of 8 CTAs x 512 threads (8 SMs: a single SM is compute-bound on this, ~400 lane-ops
// per key), no sort and no shared-memory atomics (measured here: ~2.3 ns per key per pass, the LSU serialises
// them per lane; ballot-matching inside a warp costs as much in issue slots).  Counting is THREAD-PRIVATE instead:
// thread t owns byte column t of cnt[slot][digit][512], so a histogram update is a plain LDS/ADD/STS with no
// conflicts; a row is summed afterwards with dp4a, the 8 CTAs' row sums are read through DSMEM and every CTA
// takes the same decisions on its own copy (no central CTA, one cluster barrier per level, 3 levels).
// Per token a radix select on the 15-bit fp16 magnitude, 5 + 5 + 5 bits from the top: every distinct cut
// C_d keeps (prefix, rank still needed inside the prefix); cuts with the same prefix share a histogram slot.
// After the last level thr_d is the exact cut key, take_d how many of the keys equal to thr_d are inside, and
// the cut "splits" if take_d is smaller than their number (ties go to the lower index): only then an ordered
// count of the equal keys decides them (lower-ranked CTAs: known from the last level's row sums; inside a CTA:
// per 128-row group, then a scan over its groups — no extra cluster barrier).  fp16 has few distinct
// magnitudes, so splits are the common case, not the exception.
// Widths: b = sum_d mult_d [key above cut d].  Lists: one warp per 128-row group partitions its rows by
// (width desc, index asc) with one packed warp scan (partition128) -> grows, gcnt_ge, gsched; a scan over the
// groups' per-width counts places every group's runs in the global `rows`.  The threshold form skips the select:
// the cut keys are given.
#include <cooperative_groups.h>

#include "common.cuh"

namespace cg = cooperative_groups;

namespace gq {

constexpr int AT = 512;   // threads per CTA
constexpr int AWARPS = AT / 32;
constexpr int MAXG = GQ_MAX_K / GQ_G;     // 256 groups
constexpr int CNT_BYTES = 8 * 32 * AT;    // cnt[8 slots][32 digits][512 thread columns] u8 = 128 KB

struct AssignParams {
    int T, K;
    int nd;       // distinct non-zero cuts
    int Cd[8];    // their ranks: the Cd[d] largest keys are "above" cut d
    int mult[8];  // how many widths w share the cut: b = sum_d mult[d] * [above cut d]
    int C[10];    // C[w] = rows with width >= w (for cnt_ge bookkeeping only)
    int use_thr;  // threshold form (grinqh_assign_thresholds): no selection, the cut keys are given
    int thr[8];   // use_thr: key of distinct cut d ("above" = magnitude pattern >= thr[d])
};

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// tab[g][col], g < groups: exclusive prefix over g, in place; *tot = total.  One warp per column;
// lane l owns groups 8l..8l+7.
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

constexpr int MAXNC = 8;          // CTAs in the cluster (portable maximum); CTA r owns a contiguous run of groups.
                                  // (a launch attribute; the kernel reads it back with cluster.num_blocks()).
constexpr int NLEVEL = 3;         // 5 + 5 + 5 bits of the 15-bit magnitude
constexpr int NDIG = 32;          // digits per level = lanes of the locating warp

__global__ void __launch_bounds__(AT, 1)
assign_kernel(const uint16_t* __restrict__ x, AssignParams p, uint8_t* __restrict__ bits,
              uint8_t* __restrict__ bits_union, int32_t* __restrict__ rows, int32_t* __restrict__ cnt_ge,
              uint8_t* __restrict__ grows, uint8_t* __restrict__ gcnt_ge, uint32_t* __restrict__ gsched) {
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), NC = (int)cluster.num_blocks();
    const int gpc = (p.K / GQ_G + NC - 1) / NC;                     // groups per CTA
    extern __shared__ __align__(16) uint8_t cnt[];                  // [8 slots][32 digits][AT] u8 thread-private counters
    uint16_t* xs = reinterpret_cast<uint16_t*>(cnt + CNT_BYTES);    // raw fp16 patterns, local groups, current token
    uint8_t* glist = cnt + CNT_BYTES + (size_t)gpc * GQ_G * 2;      // local groups' lists
    __shared__ __align__(16) uint8_t gcs[MAXG][GQ_GCNT];
    __shared__ __align__(16) uint8_t ubits[32 * GQ_G];              // union of the token widths, local groups (<= 32)
    __shared__ uint16_t tab[MAXG][10];                              // replicated: per-width counts of every group
    __shared__ uint16_t ltab[MAXG][8];                              // local groups: equal-key counts per cut
    __shared__ int s_rowL[NLEVEL][8 * NDIG];                        // this CTA's row sums, one array per level
    __shared__ int s_pre[2][8], s_need[8], s_h[8], s_tiebase[8], s_tot[10];  // s_pre: double-buffered by level parity

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int K = p.K, groups = K / GQ_G, nd = p.nd;
    const int gl0 = rank * gpc;                                     // first local group
    const int nloc = max(0, min(gpc, groups - gl0));
    const uint32_t lt_mask = (1u << lane) - 1u;

    // cnt is used as two regions of 4 slots (64 KB each) alternating between levels, so the region of level l+1 is
    // cleared while level l runs; with more than 4 distinct cuts a level needs the whole buffer and clears it first.
    const bool two_regions = nd <= 4;
    auto zero_region = [&](int level) {
        uint4* z = reinterpret_cast<uint4*>(cnt + (two_regions ? (level & 1) * (CNT_BYTES / 2) : 0));
        for (int i = tid; i < nd * NDIG * AT / 16; i += AT) z[i] = make_uint4(0, 0, 0, 0);
    };

    pdl_launch_dependents();

    for (int t = 0; t < p.T; ++t) {
        zero_region(0);
        if (tid < 8) {
            s_pre[0][tid] = (tid < nd) ? 0 : -1 - tid;  // level 0: one empty prefix shared by every cut
            s_need[tid] = (tid < nd) ? p.Cd[tid] : 0;
            s_h[tid] = 0;
            s_tiebase[tid] = 0;
        }
        // x may come from the previous kernel, and the outputs may still be read by it: nothing global before this
        if (t == 0) pdl_wait();
        // ---- load the token's local groups (raw patterns; the key is pattern & 0x7FFF)
        for (int i = tid; i < nloc * (GQ_G / 4); i += AT)
            reinterpret_cast<uint2*>(xs)[i] = reinterpret_cast<const uint2*>(x + (size_t)t * K + gl0 * GQ_G)[i];
        __syncthreads();

        if (p.use_thr) {  // the paper's run-time form: static thresholds, nothing to select
            if (tid < 8) {
                s_pre[NLEVEL & 1][tid] = (tid < nd) ? p.thr[tid] : 0x8000;
                s_need[tid] = 0;
                s_h[tid] = 0;  // take == h == 0: no cut splits a tie run, every key >= thr is above the cut
            }
            __syncthreads();
        }
        // ---- radix select, 5 + 5 + 5 bits: every distinct cut keeps (prefix, rank still needed inside it);
        //      cuts with the same prefix share the histogram slot of the lowest such cut
#pragma unroll 1
        for (int level = p.use_thr ? NLEVEL : 0; level < NLEVEL; ++level) {
            const int sh = 10 - 5 * level;
            const int* pre = s_pre[level & 1];
            uint8_t* reg = cnt + (two_regions ? (level & 1) * (CNT_BYTES / 2) : 0);
            // pass: count the digit of every local key whose prefix is live, in this thread's own byte columns
            for (int i = tid; i < nloc * GQ_G; i += AT) {
                const uint32_t m = xs[i] & 0x7FFFu;
                const int pe = (int)(m >> (sh + 5));
                int s = -1;
                for (int d = nd - 1; d >= 0; --d)
                    if (pre[d] == pe) s = d;
                if (s >= 0) {
                    uint8_t* c = reg + ((s * NDIG + (int)((m >> sh) & 31u)) * AT + tid);
                    *c = (uint8_t)(*c + 1);
                }
            }
            if (two_regions && level + 1 < NLEVEL) zero_region(level + 1);
            __syncthreads();
            // reduce: a warp sums rows (AT bytes each) four at a time
            for (int r0 = warp * 4; r0 < nd * NDIG; r0 += AWARPS * 4) {
                uint4 a[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) a[u] = reinterpret_cast<const uint4*>(reg + (r0 + u) * AT)[lane];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    uint32_t s = 0;
                    s = __dp4a(a[u].x, 0x01010101u, s); s = __dp4a(a[u].y, 0x01010101u, s);
                    s = __dp4a(a[u].z, 0x01010101u, s); s = __dp4a(a[u].w, 0x01010101u, s);
                    s = __reduce_add_sync(0xffffffffu, s);
                    if (lane == 0) s_rowL[level][r0 + u] = (int)s;
                }
            }
            cluster.sync();
            // locate: warp d reads the 8 CTAs' sums of its slot's 32 digits (DSMEM) and scans them from the top;
            // every CTA takes the same decision on its own copy
            if (warp < nd) {
                const int d = warp, digit = NDIG - 1 - lane;
                const int pr = pre[d];
                int sl = d;
                for (int e = d - 1; e >= 0; --e)
                    if (pre[e] == pr) sl = e;
                const int idx = level * (8 * NDIG) + sl * NDIG + digit;
                int h = 0, mine_below = 0;
                for (int r = 0; r < NC; ++r) {
                    const int v = cluster.map_shared_rank(&s_rowL[0][0], r)[idx];
                    h += v;
                    if (r < rank) mine_below += v;
                }
                const int incl = warp_incl_scan(h, lane);
                const int above = incl - h, need = s_need[d];
                __syncwarp();
                if (above < need && need <= above + h) {
                    s_pre[(level + 1) & 1][d] = (pr << 5) | digit;
                    s_need[d] = need - above;
                    s_h[d] = h;
                    s_tiebase[d] = mine_below;  // after the last level: keys equal to the cut in lower-ranked CTAs
                }
            }
            if (!two_regions && level + 1 < NLEVEL) zero_region(level + 1);
            if (tid >= 8 * 32 && tid < 8 * 32 + 8 && tid - 8 * 32 >= nd) s_pre[(level + 1) & 1][tid - 8 * 32] = -1 - (tid - 8 * 32);
            __syncthreads();
        }
        int thr[8], take[8], mult[8];
        bool split[8], anysplit = false;
#pragma unroll
        for (int d = 0; d < 8; ++d) {
            thr[d] = (d < nd) ? s_pre[NLEVEL & 1][d] : 0x8000;
            take[d] = (d < nd) ? s_need[d] : 0;
            mult[d] = (d < nd) ? p.mult[d] : 0;
            split[d] = (d < nd) && take[d] < s_h[d];
            anysplit |= split[d];
        }
        if (anysplit) {  // cluster-uniform, but everything in here is CTA-local
            // ---- a cut splits a run of equal keys: ordered (index-ascending) count of the equal keys.  Keys equal
            //      to the cut in lower-ranked CTAs are already known (s_tiebase, from the last level's row sums);
            //      inside the CTA: count per local group, then a scan over the (at most 32) local groups.
            for (int lg = warp; lg < nloc; lg += AWARPS) {
                const uint2 kv = *reinterpret_cast<const uint2*>(xs + lg * GQ_G + 4 * lane);
                const int m[4] = {(int)(kv.x & 0x7FFF), (int)((kv.x >> 16) & 0x7FFF), (int)(kv.y & 0x7FFF),
                                  (int)((kv.y >> 16) & 0x7FFF)};
                int mine = 0;
#pragma unroll
                for (int d = 0; d < 8; ++d)
                    if (split[d]) {
                        int c = 0;
#pragma unroll
                        for (int i = 0; i < 4; ++i) c += (m[i] == thr[d]);
                        c = __reduce_add_sync(0xffffffffu, c);
                        if (lane == d) mine = c;
                    }
                if (lane < 8) ltab[lg][lane] = (uint16_t)mine;
            }
            __syncthreads();
            if (warp < 8 && split[warp]) {  // warp d scans cut d over the local groups, 32 at a time
                int carry = s_tiebase[warp];
                for (int l0 = 0; l0 < nloc; l0 += 32) {
                    const int lg = l0 + lane;
                    const int v = (lg < nloc) ? ltab[lg][warp] : 0;
                    const int incl = warp_incl_scan(v, lane);
                    if (lg < nloc) ltab[lg][warp] = (uint16_t)(carry + incl - v);
                    carry += __shfl_sync(0xffffffffu, incl, 31);
                }
            }
            __syncthreads();
        }
        // ---- widths of this token
        for (int lg = warp; lg < nloc; lg += AWARPS) {
            const int g = gl0 + lg;
            const uint2 kv = *reinterpret_cast<const uint2*>(xs + lg * GQ_G + 4 * lane);
            const int m[4] = {(int)(kv.x & 0x7FFF), (int)((kv.x >> 16) & 0x7FFF), (int)(kv.y & 0x7FFF),
                              (int)((kv.y >> 16) & 0x7FFF)};
            int b[4] = {0, 0, 0, 0};
#pragma unroll
            for (int d = 0; d < 8; ++d) {
                if (!split[d]) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) b[i] += (m[i] >= thr[d]) ? mult[d] : 0;
                } else {
                    bool eq[4];
                    int below = ltab[lg][d];  // equal keys at lower indices outside this group
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        eq[i] = (m[i] == thr[d]);
                        below += __popc(__ballot_sync(0xffffffffu, eq[i]) & lt_mask);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        b[i] += ((m[i] > thr[d]) || (eq[i] && below < take[d])) ? mult[d] : 0;
                        below += eq[i];
                    }
                }
            }
            const uint32_t packed = (uint32_t)b[0] | ((uint32_t)b[1] << 8) | ((uint32_t)b[2] << 16) | ((uint32_t)b[3] << 24);
            *reinterpret_cast<uint32_t*>(bits + (size_t)t * K + g * GQ_G + 4 * lane) = packed;
            uint32_t* u = reinterpret_cast<uint32_t*>(ubits + lg * GQ_G + 4 * lane);  // union over tokens, shared memory
            if (t == 0) *u = packed;
            else *u = __vmaxu4(*u, packed);
        }
        __syncthreads();
    }

    // ---- per-group lists of the local groups
    const bool single_pass = nloc <= AWARPS;  // every warp has at most one group
    for (int lg = warp; lg < nloc; lg += AWARPS) {
        const int g = gl0 + lg;
        const int go = g * GQ_G + 4 * lane, lo = lg * GQ_G + 4 * lane;
        const uint32_t bu4 = *reinterpret_cast<const uint32_t*>(ubits + lo);
        uint32_t bt4[GRINQH_MAX_T];
        uint2 xv[GRINQH_MAX_T];
#pragma unroll
        for (int t = 0; t < GRINQH_MAX_T; ++t)
            if (t < p.T) {
                bt4[t] = (p.T == 1) ? bu4 : *reinterpret_cast<const uint32_t*>(bits + (size_t)t * K + go);
                xv[t] = (p.T == 1) ? *reinterpret_cast<const uint2*>(xs + lo)
                                   : *reinterpret_cast<const uint2*>(x + (size_t)t * K + go);
            }
        int bu[4], pos[4], ge[10];
#pragma unroll
        for (int i = 0; i < 4; ++i) bu[i] = (bu4 >> (8 * i)) & 0xFF;
        partition128(bu, lane, pos, ge);
        int myge = 0, myn = 0;
#pragma unroll
        for (int c = 0; c <= 8; ++c)
            if (lane == c) {
                myge = ge[c];
                myn = ge[c] - ge[c + 1];
            }
        const uint8_t gv = (uint8_t)(lane <= 8 ? myge : 0);
        if (lane < GQ_GCNT) gcs[lg][lane] = gv;
        {   // every CTA gets the group's 9 per-width counts: lane = 9 * r' + c stores column c to CTA r' (and r' + 3, r' + 6)
            const int c = lane % 9, r0 = lane / 9;
            const int n = __shfl_sync(0xffffffffu, myn, c);
            if (lane < 27)
                for (int r = r0; r < NC; r += 3) cluster.map_shared_rank(&tab[0][0], r)[g * 10 + c] = (uint16_t)n;
        }
        // the cluster barrier only has to cover the counts just sent: arrive now (when this warp has no further group),
        // then write the outputs to global memory in its shadow
        if (single_pass) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        *reinterpret_cast<uint32_t*>(bits_union + go) = bu4;
        if (lane < GQ_GCNT) gcnt_ge[g * GQ_GCNT + lane] = gv;
#pragma unroll
        for (int i = 0; i < 4; ++i) glist[lg * GQ_G + pos[i]] = (uint8_t)(4 * lane + i);
#pragma unroll
        for (int t = 0; t < GRINQH_MAX_T; ++t)
            if (t < p.T) {
                const uint32_t xq[4] = {xv[t].x & 0xFFFFu, xv[t].x >> 16, xv[t].y & 0xFFFFu, xv[t].y >> 16};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    gsched[(size_t)t * K + g * GQ_G + pos[i]] = (uint32_t)(4 * lane + i) |
                                                                (((bt4[t] >> (8 * i)) & 0xFFu) << 8) |
                                                                ((uint32_t)bu[i] << 12) | (xq[i] << 16);
            }
        __syncwarp();
        *reinterpret_cast<uint32_t*>(grows + go) = *reinterpret_cast<const uint32_t*>(glist + lo);
    }
    if (!single_pass || warp >= nloc) asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");  // the last remote access is before this barrier
    // ---- where each group's run of every width starts in the global list (every CTA scans its own copy)
    if (warp < 9) scan_groups(tab, warp, groups, lane, &s_tot[warp]);
    __syncthreads();
    // ---- global list (width desc, index asc) and cnt_ge
    int cbase[9];
    {
        int acc = 0;
#pragma unroll
        for (int c = 8; c >= 0; --c) {
            cbase[c] = acc;
            acc += s_tot[c];
        }
    }
    if (rank == 0 && tid < 10) cnt_ge[tid] = (tid == 9) ? 0 : cbase[tid] + s_tot[tid];
    for (int lg = warp; lg < nloc; lg += AWARPS) {
        const int g = gl0 + lg;
        const uint4 cv = *reinterpret_cast<const uint4*>(gcs[lg]);
        const int cge[10] = {(int)(cv.x & 0xFF), (int)((cv.x >> 8) & 0xFF), (int)((cv.x >> 16) & 0xFF), (int)(cv.x >> 24),
                             (int)(cv.y & 0xFF), (int)((cv.y >> 8) & 0xFF), (int)((cv.y >> 16) & 0xFF), (int)(cv.y >> 24),
                             (int)(cv.z & 0xFF), 0};
        const uint32_t l4 = *reinterpret_cast<const uint32_t*>(glist + lg * GQ_G + 4 * lane);
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

namespace gq {
static int check_assign_args(const void* x_f16, int T, int K, const void* spec, uint8_t* bits, uint8_t* bits_union,
                             int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge, uint32_t* gsched) {
    if (!x_f16 || !spec || !bits || !bits_union || !rows || !cnt_ge || !grows || !gcnt_ge || !gsched)
        return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || K % GQ_G || K > GQ_MAX_K) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_f16 | (uintptr_t)bits | (uintptr_t)bits_union | (uintptr_t)rows | (uintptr_t)cnt_ge |
         (uintptr_t)grows | (uintptr_t)gcnt_ge | (uintptr_t)gsched) & 15)
        return GRINQH_ERR_ALIGN;
    return GRINQH_OK;
}

static int launch_assign(const AssignParams& p, const void* x_f16, uint8_t* bits, uint8_t* bits_union, int32_t* rows,
                         int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge, uint32_t* gsched, void* stream) {
    // cluster size: measured on B200 (T=1, K=4096): 1 CTA 23.5 us, 2: 16.4, 4: 13.4, 8: 12.3 — the kernel is bound by
    // per-CTA instruction latency, not by the cluster barriers, so always the portable maximum (a non-portable cluster
    // of 16 for K >= 4096 was measured too: layer step 110.8 us against 109.5 us, the 16 remote row-sum reads and the
    // wider barrier cost more than the halved per-CTA work saves)
    const int nc = MAXNC;
    const int gpc = (p.K / GQ_G + nc - 1) / nc;
    const size_t smem = (size_t)CNT_BYTES + (size_t)gpc * GQ_G * 3;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 CNT_BYTES + 32 * GQ_G * 3) != cudaSuccess)  // at most 32 groups per CTA
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(nc);
    cfg.blockDim = dim3(AT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = (cudaStream_t)stream;
    cudaLaunchAttribute at[2];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = nc;
    at[1].val.clusterDim.y = 1;
    at[1].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 2;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, assign_kernel, (const uint16_t*)x_f16, p, bits, bits_union, rows,
                                             cnt_ge, grows, gcnt_ge, gsched);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
}  // namespace gq

extern "C" int grinqh_assign(const void* x_f16, int T, int K, const uint32_t counts[9], uint8_t* bits,
                             uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge,
                             uint32_t* gsched, void* workspace, size_t workspace_bytes, void* stream) {
    (void)workspace;
    (void)workspace_bytes;
    int rc = gq::check_assign_args(x_f16, T, K, counts, bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched);
    if (rc != GRINQH_OK) return rc;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    gq::AssignParams p{};
    p.T = T;
    p.K = K;
    p.C[9] = 0;
    for (int w = 8; w >= 0; --w) p.C[w] = p.C[w + 1] + (int)counts[w];
    for (int w = 1; w <= 8; ++w) {  // distinct non-zero cuts
        if (p.C[w] == 0) continue;
        int d = 0;
        while (d < p.nd && p.Cd[d] != p.C[w]) ++d;
        if (d == p.nd) {
            p.Cd[p.nd] = p.C[w];
            p.mult[p.nd++] = 0;
        }
        p.mult[d]++;
    }
    return gq::launch_assign(p, x_f16, bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched, stream);
}

extern "C" int grinqh_assign_thresholds(const void* x_f16, int T, int K, const uint16_t theta[9], uint8_t* bits,
                                        uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge, uint8_t* grows,
                                        uint8_t* gcnt_ge, uint32_t* gsched, void* stream) {
    int rc = gq::check_assign_args(x_f16, T, K, theta, bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched);
    if (rc != GRINQH_OK) return rc;
    for (int w = 1; w <= 8; ++w)
        if (theta[w] > 0x8000 || (w > 1 && theta[w] < theta[w - 1])) return GRINQH_ERR_MIX;
    gq::AssignParams p{};
    p.T = T;
    p.K = K;
    p.use_thr = 1;
    for (int w = 1; w <= 8; ++w) {  // distinct reachable thresholds
        if (theta[w] == 0x8000) continue;
        int d = 0;
        while (d < p.nd && p.thr[d] != (int)theta[w]) ++d;
        if (d == p.nd) {
            p.thr[p.nd] = (int)theta[w];
            p.mult[p.nd++] = 0;
        }
        p.mult[d]++;
    }
    return gq::launch_assign(p, x_f16, bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched, stream);
}
