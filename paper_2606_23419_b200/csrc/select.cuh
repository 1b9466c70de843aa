// select.cuh — rank selection and per-key widths, shared by grinqh_assign (assign.cu) and by the VMM launches that
// make the assignment themselves (vmm.cu: grinqh_vmm_rank, grinqh_vmm_thresholds).
// PAPER.md:61-65 (assignment), :271 (top-p partition of the live vector); readings #2-#4.
//
// One CTA does the whole selection on its own copy of the keys (every CTA of a grid repeats it: the CTAs would
// otherwise wait for one another, and a redundant select needs no grid-wide exchange).  Radix select on the 15-bit
// fp16 magnitude, 5 + 5 + 5 bits from the top; every distinct cut C_d keeps (prefix, rank still needed inside the
// prefix), cuts with the same prefix share a histogram slot.  It runs once per launch on the critical path: what
// counts is the number of instructions and the length of the dependent chains.
#pragma once
#include "common.cuh"

namespace gq {

#ifdef GQ_TIMING
__device__ long long g_sel_stamp[32];
__device__ int g_sel_n;
#define SEL_STAMP() do { if (threadIdx.x == 0 && blockIdx.x == 0 && blockIdx.y == 0) g_sel_stamp[g_sel_n++] = clock64(); } while (0)
#else
#define SEL_STAMP()
#endif

constexpr int SEL_NDIG = 32;   // digits per level
constexpr int SEL_LEVELS = 3;  // 5 + 5 + 5 bits

// What the launch knows about the level mix (host-made, passed by value).
struct CutParams {
    int nd;       // distinct non-empty cuts, ordered from the highest width down (Cd non-decreasing)
    int Cd[8];    // rank form: the Cd[d] largest keys are above cut d
    int mult[8];  // widths sharing the cut: b = sum_d mult[d] * [key above cut d]
    int thr[8];   // threshold form: key of cut d ("above" = magnitude pattern >= thr[d])
    int cw[9];    // cut that decides width w: a row has >= w bits iff its key is above cut cw[w] (-1: never)
};

static inline void cuts_fill_cw(CutParams& p) {
    int w = 8, btot = 0;
    for (int d = 0; d < p.nd; ++d) btot += p.mult[d];
    for (int i = 0; i < 9; ++i) p.cw[i] = -1;
    w = btot;
    for (int d = 0; d < p.nd; ++d)
        for (int m = 0; m < p.mult[d]; ++m) p.cw[w--] = d;
}

// Run-time result of the selection for one token, in shared memory: what the width computation reads.
struct TokenCuts {
    int thr[8];        // cut keys (0x8000 = unreachable)
    int take[8];       // how many of the keys equal to thr[d] are above the cut (ties go to the lower index)
    int hh[8];         // number of keys equal to thr[d]
    uint32_t split;    // bit d: cut d splits a run of equal keys (take[d] < hh[d])
    int nd;
    uint32_t pad[2];
};

// scratch of the select (shared memory)
struct SelectScratch {
    int wsum[32];          // block scan: keys in each warp's histogram blocks
};

__device__ __forceinline__ int warp_incl_scan_i(int v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += o;
    }
    return v;
}

// hist: 16384 words of shared memory (64 KB), ALL ZERO on entry and left all zero: two 16-bit bins per word, bin =
// the 15-bit magnitude.  x: the token's K raw fp16 patterns in GLOBAL memory (16-byte aligned, K % 8 == 0); they are
// copied to skeys (shared) on the way.  All NT threads of the CTA call this; the result is written to *tc (valid
// after the final barrier inside).
//
// One pass: every key is one shared-memory atomic into its own bin (measured here: 1.6 cycles per warp-wide atomic
// when the addresses are spread, which fp16 magnitudes of real activations are; equal keys in one warp serialise, so
// degenerate inputs are slower, not wrong).  Then every thread sums its block of 16384 / NT words (the two halves
// cannot overflow: the total is K <= 32768), a block scan gives ascending ranks, and the warp holding the block with
// rank K - C_d scans that block's bins: the cut key is the bin holding ascending rank K - C_d, `hh` its count,
// `take` how many of them lie inside the top C_d.  Three block barriers in all.
template <int NT>
__device__ __noinline__ void rank_select(const uint16_t* __restrict__ x, uint16_t* skeys, int K, int nd, const int* Cd,
                                         uint32_t* hist, bool clear, SelectScratch* sc, TokenCuts* tc) {
    constexpr int NW = NT / 32;
    constexpr int WPT = 16384 / NT;  // histogram words per thread
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    SEL_STAMP();
    // (four 16-byte loads in flight per thread before their 32 atomics: the loop is bound by the load latency otherwise)
#pragma unroll 1
    for (int c0 = tid; c0 < (K >> 3); c0 += 4 * NT) {
        uint4 kv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (c0 + u * NT < (K >> 3)) kv[u] = reinterpret_cast<const uint4*>(x)[c0 + u * NT];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (c0 + u * NT < (K >> 3)) {
                reinterpret_cast<uint4*>(skeys)[c0 + u * NT] = kv[u];
                const uint32_t kw[4] = {kv[u].x, kv[u].y, kv[u].z, kv[u].w};
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const uint32_t m = (kw[j >> 1] >> (16 * (j & 1))) & 0x7FFFu;
                    atomicAdd(&hist[m >> 1], (m & 1u) ? 0x10000u : 1u);
                }
            }
        }
    }
    SEL_STAMP();
    __syncthreads();
    SEL_STAMP();
    // ---- block sums and block scan (ascending)
    uint32_t packed = 0;
    {
        // (the threads' blocks are 128 or 256 bytes apart: each starts at its own 16-byte piece so that the lanes of
        // a warp spread over all banks)
        const uint4* hp = reinterpret_cast<const uint4*>(hist + tid * WPT);
#pragma unroll
        for (int q = 0; q < WPT / 4; ++q) {
            const uint4 v = hp[(q + tid) & (WPT / 4 - 1)];
            packed += v.x + v.y + v.z + v.w;
        }
    }
    const int mysum = (int)((packed & 0xFFFFu) + (packed >> 16));
    const int incl = warp_incl_scan_i(mysum, lane);
    if (lane == 31) sc->wsum[warp] = incl;
    if (tid >= nd && tid < 8) {
        tc->thr[tid] = 0x8000;
        tc->take[tid] = 0;
        tc->hh[tid] = 0;
    }
    SEL_STAMP();
    __syncthreads();
    SEL_STAMP();
    int wbase = 0;  // keys in lower warps' blocks (every warp scans the warp sums itself: no second barrier)
    {
        const int v = (lane < NW) ? sc->wsum[lane] : 0;
        const int i2 = warp_incl_scan_i(v, lane);
        wbase = __shfl_sync(0xffffffffu, i2 - v, warp);
    }
    const int excl = wbase + incl - mysum;  // keys in lower blocks
    // ---- the warp that holds the block with cut d's rank scans that block's bins right away
#pragma unroll 1
    for (int d = 0; d < nd; ++d) {
        const int R = K - Cd[d];  // ascending rank (0-based) of the smallest key inside the top C_d
        const uint32_t own = __ballot_sync(0xffffffffu, excl <= R && R < excl + mysum);
        if (own == 0) continue;  // (exactly one thread of the CTA owns it)
        const int src = __ffs(own) - 1;
        const int rem = R - __shfl_sync(0xffffffffu, excl, src);
        const int blk0 = (warp * 32 + src) * WPT;
        int carry = 0;
#pragma unroll 1
        for (int w0 = 0; w0 < WPT; w0 += 32) {
            const uint32_t v = hist[blk0 + w0 + lane];
            const int c0 = (int)(v & 0xFFFFu), c1 = (int)(v >> 16);
            const int inc2 = warp_incl_scan_i(c0 + c1, lane);
            const int ex2 = carry + inc2 - (c0 + c1);
            if (ex2 <= rem && rem < ex2 + c0 + c1) {  // exactly one lane of one round
                const bool hi = rem - ex2 >= c0;
                const int h = hi ? c1 : c0;
                const int below = rem - ex2 - (hi ? c0 : 0);  // equal keys below the rank: outside the top C_d
                tc->thr[d] = (blk0 + w0 + lane) * 2 + (hi ? 1 : 0);
                tc->hh[d] = h;
                tc->take[d] = h - below;
            }
            carry += __shfl_sync(0xffffffffu, inc2, 31);
        }
    }
    SEL_STAMP();
    __syncthreads();
    SEL_STAMP();
    if (clear) {  // the histogram is cleared for the next use (otherwise the caller does it, off the critical path)
        uint4* hp = reinterpret_cast<uint4*>(hist + tid * WPT);
#pragma unroll
        for (int q = 0; q < WPT / 4; ++q) hp[(q + tid) & (WPT / 4 - 1)] = make_uint4(0, 0, 0, 0);
    }
    if (tid == 0) {
        uint32_t sp = 0;
        for (int d = 0; d < nd; ++d)
            if (tc->take[d] < tc->hh[d]) sp |= 1u << d;
        tc->split = sp;
        tc->nd = nd;
    }
    SEL_STAMP();
    __syncthreads();
}

// Widths of the lane's 4 consecutive rows (4 lane .. 4 lane + 3 of a 128-row group) for one token.
// m: magnitude patterns.  tc: the token's cuts (shared memory).  tie8: for split cuts, the number of keys equal to the
// cut at lower indices OUTSIDE this group (8 x u16, ignored when tc->split == 0).
__device__ __forceinline__ void widths4(const int (&m)[4], const TokenCuts* tc, const int* mult, int nd,
                                        const uint16_t* tie8, int lane, int (&b)[4]) {
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t split = tc->split;
#pragma unroll
    for (int i = 0; i < 4; ++i) b[i] = 0;
#pragma unroll 1
    for (int d = 0; d < nd; ++d) {
        const int th = tc->thr[d], mu = mult[d];
        if (!((split >> d) & 1u)) {
#pragma unroll
            for (int i = 0; i < 4; ++i) b[i] += (m[i] >= th) ? mu : 0;
        } else {
            const int tk = tc->take[d];
            bool eq[4];
            int below = (int)tie8[d];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                eq[i] = (m[i] == th);
                below += __popc(__ballot_sync(0xffffffffu, eq[i]) & lt_mask);
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                b[i] += ((m[i] > th) || (eq[i] && below < tk)) ? mu : 0;
                below += eq[i];
            }
        }
    }
}

__device__ __forceinline__ void keys4(uint2 kv, int (&m)[4]) {
    m[0] = (int)(kv.x & 0x7FFF);
    m[1] = (int)((kv.x >> 16) & 0x7FFF);
    m[2] = (int)(kv.y & 0x7FFF);
    m[3] = (int)((kv.y >> 16) & 0x7FFF);
}

// Host side: level mix -> distinct cuts.
static inline CutParams cuts_from_counts(const uint32_t counts[9]) {
    CutParams p{};
    int C[10];
    C[9] = 0;
    for (int w = 8; w >= 0; --w) C[w] = C[w + 1] + (int)counts[w];
    for (int w = 8; w >= 1; --w) {  // from the highest width down: Cd is non-decreasing
        if (C[w] == 0) continue;
        if (p.nd > 0 && p.Cd[p.nd - 1] == C[w]) {
            p.mult[p.nd - 1]++;
        } else {
            p.Cd[p.nd] = C[w];
            p.mult[p.nd++] = 1;
        }
    }
    for (int d = 0; d < 8; ++d) p.thr[d] = 0x8000;
    cuts_fill_cw(p);
    return p;
}

// theta[w], w = 1..8, non-decreasing in w, 0x8000 = unreachable -> distinct reachable thresholds (highest first)
static inline CutParams cuts_from_thetas(const uint16_t theta[9]) {
    CutParams p{};
    for (int d = 0; d < 8; ++d) p.thr[d] = 0x8000;
    for (int w = 8; w >= 1; --w) {
        if (theta[w] == 0x8000) continue;
        if (p.nd > 0 && p.thr[p.nd - 1] == (int)theta[w]) {
            p.mult[p.nd - 1]++;
        } else {
            p.thr[p.nd] = (int)theta[w];
            p.mult[p.nd++] = 1;
        }
    }
    cuts_fill_cw(p);
    return p;
}

}  // namespace gq
