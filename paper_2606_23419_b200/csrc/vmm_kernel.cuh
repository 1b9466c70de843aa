// vmm_kernel.cuh — the VMM kernel template (instantiated in vmm.cu for one token and in vmm_multi.cu for 2..4).
// PAPER.md:85 (reconstruction), :51 (only the needed planes are fetched), :61-65 / :271 (assignment),
// :440-444 (prior-art kernel).
//
// Decomposition.  Grid = (column tiles of 1024 columns) x (Sx split-K slices), one CTA per SM.  For one column tile the
// work is the "row stream": all groups in order, inside a group the rows with b > 0 in (width desc, index asc) order.
// A row of width b costs ROW_COST + b units (measured instruction counts), a group's cost follows from its nine
// per-width counts, and warp slot ws of the tile's Sx * VW warps owns the rows whose start cost falls into
// [ws * W / S, (ws + 1) * W / S): every warp of the grid gets the same amount of work whatever the width mix and
// however the rows are spread over the groups (no per-step planning on the host, no tail of unlucky CTAs).
// VW (warps per CTA) is chosen from the shape: few fat warps for small problems (the per-warp fixed work — range,
// lists, scale/zero chunks, epilogue — is what a small launch pays for), 16 for large ones; the ring depth grows as
// VW shrinks so that an SM keeps the same bytes in flight.
//
// A warp runs without block barriers from the prologue to the CTA epilogue:
//   list     the warp's rows and, behind the rows of each group, four "scale/zero chunk" entries are appended to a
//            circular list in shared memory, one group segment at a time and ahead of the copies; the entries come from
//            gsched (grinqh_assign ran before) or are made on the spot from x and the cuts (threshold / rank form:
//            widths4 + partition128), so the assignment needs no kernel of its own.
//   stream   a warp-private ring of RING 1-KB slots filled by cp.async (LDGSTS.128): lanes 8j..8j+7 copy the 128-byte
//            segment of plane j, so a 4-bit row is one instruction and an 8-bit row two; list entry v always lives in
//            slot v mod RING and is one cp.async group; RING-2 entries are in flight while one is consumed, across
//            group boundaries.
//   expand   lane l owns columns 32l..32l+31 of the tile: b conflict-free LDS, SIMD-in-register 8x8 bit transpose
//            (gather.cuh), PRMT to fp16 subnormal patterns, 32 mixed-precision FMAs acc[c] += half(code_c) * half(x_k)
//            (exact product, fp32 accumulate).
//   chunk    y_n += s_gn * (A_n * 2^24 + Phi) + z_gn * X for 8 of the lane's columns per chunk entry: s and z are
//            applied once per (group segment, column); Phi = sum x_k phi_{b_k}, X = sum x_k ride along in registers.
// CTA epilogue: the warps' sums are added in fixed order into one split-K partial part[sx][t][n]; the last CTA of the
// tile (ticket) sums the Sx partials in fixed order.  Deterministic: the result depends on the shape and the widths only.
//
// Rank form inside the launch (grinqh_vmm_rank): every CTA selects the cut keys itself (select.cuh), counts per group
// the keys above / equal to each cut, turns the equal counts into ordered tie offsets with one scan, and (one token)
// derives every group's per-width counts arithmetically; the per-row widths are only made for the groups a warp walks.
#pragma once
#include <cstdio>
#include <type_traits>

#include "common.cuh"
#include "gather.cuh"
#include "select.cuh"

namespace gq {

constexpr int TILE_COLS = 1024;
constexpr int SLOT_BYTES = 1024;   // 8 planes x 128 B
constexpr int YSLOT = 32 * 33;     // one warp's 1024 sums, padded: column 32*l + c lives at c*33 + l
constexpr int GLC = 8;             // group lists a CTA builds once for all its warps (one token, in-kernel assignment)
constexpr int MAXG = GQ_MAX_K / GQ_G;
constexpr int ROW_COST = 12;       // cost of a row of width b = ROW_COST + b (loop bodies: ~94 / 106 / 137 instructions)
constexpr uint32_t ENTRY_SZ = 0x80u;  // list entry is a scale/zero chunk (bits 0..1 = chunk); rows use bits 0..6
constexpr size_t TICKET_BYTES = 16384;  // head of the workspace: one int per column tile, zero between launches

enum { MODE_SCHED = 0, MODE_THR = 1, MODE_RANK = 2 };

constexpr int cmax(int a, int b) { return a > b ? a : b; }

template <int T, int VW>
struct Cfg {
    static constexpr int NT = VW * 32;
    static constexpr int RING = (T == 1) ? 128 / VW : (T <= 3) ? 8 : 4;
    static constexpr int LISTN = ((T == 1 && VW == 16) || T >= 3) ? 128 : 256;  // circular list entries per warp
    // per-warp shared memory: ring | yacc[T] | list[LISTN] {word, offset} | words of tokens 1..T-1 | {X, Phi}[16][T]
    static constexpr int RING_OFF = 0;
    static constexpr int YACC_OFF = RING * SLOT_BYTES;
    static constexpr int LIST_OFF = YACC_OFF + T * YSLOT * 4;
    static constexpr int XPHI_OFF = LIST_OFF + LISTN * 8 + (T - 1) * LISTN * 4;
    static constexpr int WARP_BYTES = XPHI_OFF + 16 * T * 8;
    // the assignment prologue aliases the warp regions: one token's keys and the select's 64-KB histogram
    static constexpr int KEYS_OFF = 0;
    static constexpr int HIST_OFF = GQ_MAX_K * 2;
    static constexpr int GTEQ_OFF = HIST_OFF + 65536;  // keys above / equal to each cut per group: 2 x [MAXG][8] bytes
    static constexpr int BASE_BYTES = cmax(VW * WARP_BYTES, GTEQ_OFF + 2 * MAXG * 8);  // the tie offsets live behind
    static_assert(WARP_BYTES % 16 == 0, "warp regions stay 16-byte aligned");
    static_assert(T == 1 || VW == 8, "several tokens: 8 warps (registers: acc[T][32])");
};

struct VmmPlan {
    int col_tiles;  // ceil(N / 1024)
    int Sx;         // CTAs (= split-K partials) per column tile
    int vw;         // warps per CTA
};

struct VmmArgs {
    int T, K, N, fused, mode;
    const uint32_t* planes;
    const void *scales, *zeros;
    const uint32_t* gsched;
    const uint8_t* gcnt_ge;
    const uint16_t* xraw;
    CutParams cp;
    void* workspace;
    float* y;
    cudaStream_t st;
};

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

// cost of a group from its per-width counts ge[w] = rows of width >= w (bytes of cv):
// sum_w n_w (ROW_COST + w) = ROW_COST ge[1] + sum_{w>=1} ge[w]
__device__ __forceinline__ int group_cost(const uint4 cv) {
    const uint32_t s = __dp4a(cv.x & 0xFFFFFF00u, 0x01010101u, 0u) + __dp4a(cv.y, 0x01010101u, 0u) + (cv.z & 0xFFu);
    return (int)(ROW_COST * ((cv.x >> 8) & 0xFFu) + s);
}

// First list position of a group whose start cost is >= off (rows in width desc order), lane-parallel: lane w = 1..8
// looks at the rows of width w.  gc = the group's 16 count bytes in shared memory.  Same result on every lane.
__device__ __forceinline__ int pos_from_cost(const uint8_t* gc, int off, int lane) {
    const int w = (lane >= 1 && lane <= 8) ? lane : 0;
    const int hi = w ? (int)gc[w + 1] : 0;                 // rows of larger width = position of the class
    const int n = w ? (int)gc[w] - hi : 0;
    const int c = ROW_COST + w;
    int cum = n * c;                                       // suffix sum over larger widths: lanes above
#pragma unroll
    for (int d = 1; d < 8; d <<= 1) {
        const int o = __shfl_down_sync(0xffffffffu, cum, d);
        if (lane + d <= 8) cum += o;
    }
    const int before = cum - n * c;                        // cost of all rows of larger width
    const bool mine = w && off >= before && off < before + n * c;
    const uint32_t bal = __ballot_sync(0xffffffffu, mine);
    const int pos = hi + (off - before + c - 1) / c;
    if (bal == 0) return (int)gc[1];                       // off at or beyond the group's cost
    return __shfl_sync(0xffffffffu, pos, __ffs(bal) - 1);
}

// A16: every plane row is 16-byte aligned (N % 128 == 0) -> LDGSTS.128, 4 planes per instruction;
// otherwise each lane copies its own word of every plane with 4-byte cp.async.
//
// gsched[t][g*128 + p] (MODE_SCHED, written by grinqh_assign) is position p of group g's list for token t:
//   bits 0..7 local row r | 8..11 b_t (token's width) | 12..15 b (union width = planes fetched) | 16..31 x_t[r] fp16
// The in-kernel forms build the same entries from xraw.
template <int T, int VW, bool A16, int MODE>
__global__ void __launch_bounds__(VW * 32, 1)
vmm_kernel(int K, int N, int Sx, int fused, const uint32_t* __restrict__ planes, const __half* __restrict__ scales,
           const __half* __restrict__ zeros, const uint32_t* __restrict__ gsched, const uint8_t* __restrict__ gcnt_ge,
           const uint16_t* __restrict__ xraw, CutParams cp, float* __restrict__ part, int* __restrict__ tickets,
           float* __restrict__ y) {
    using C = Cfg<T, VW>;
    constexpr int RING = C::RING, NT = C::NT;
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ __align__(16) uint8_t s_gcnt[MAXG][GQ_GCNT];  // per-group counts ge[0..9] of the union widths
    __shared__ uint32_t s_glist[GLC][GQ_G];                 // lists of the first GLC groups of this CTA's range
    __shared__ int s_pref[MAXG + 1];                         // exclusive prefix of the groups' costs
    __shared__ __align__(16) TokenCuts s_tc[T];
    __shared__ SelectScratch s_sel;
    __shared__ int s_wsum[32], s_total, s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, sx = blockIdx.y;
    const int words = N >> 5;
    const int word = tile * 32 + lane;
    const bool active = word < words;
    const uint32_t rowbytes = (uint32_t)words * 4u;
    const size_t pbytes = (size_t)K * rowbytes;  // one plane
    const int groups = K / GQ_G;
    const int nd = cp.nd;

    uint8_t* wbase = smem + warp * C::WARP_BYTES;
    const uint8_t* ring = wbase + C::RING_OFF;
    float* yacc = reinterpret_cast<float*>(wbase + C::YACC_OFF);
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(wbase + C::RING_OFF);
    uint16_t* s_tie = reinterpret_cast<uint16_t*>(smem + C::BASE_BYTES);  // [T][groups][8] ordered tie offsets
    uint8_t (*s_gt)[8] = reinterpret_cast<uint8_t (*)[8]>(smem + C::GTEQ_OFF);  // prologue only (aliases warp regions)
    uint8_t (*s_eq)[8] = s_gt + MAXG;

#ifdef GQ_TIMING
    long long stamp[16];
    int nst = 0;
#define GQ_STAMP() stamp[nst++] = clock64()
#else
#define GQ_STAMP()
#endif
    GQ_STAMP();
    pdl_launch_dependents();

    // ================================================================== prologue: per-group counts of the union widths
    if (MODE == MODE_SCHED) {
        pdl_wait();  // nothing global is touched before the previous kernel has finished
        for (int g = tid; g < groups; g += NT)
            *reinterpret_cast<uint4*>(s_gcnt[g]) = *reinterpret_cast<const uint4*>(gcnt_ge + (size_t)g * GQ_GCNT);
    } else {
        uint16_t* skeys = reinterpret_cast<uint16_t*>(smem + C::KEYS_OFF);
        if (MODE == MODE_RANK) {  // the select's histogram: cleared while the previous kernel is still running
            uint4* z = reinterpret_cast<uint4*>(smem + C::HIST_OFF);
            for (int i = tid; i < 4096; i += NT) z[i] = make_uint4(0, 0, 0, 0);
            __syncthreads();
        }
        pdl_wait();
#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            if (MODE == MODE_RANK) {
                GQ_STAMP();
                rank_select<NT>(xraw + (size_t)t * K, skeys, K, nd, cp.Cd, reinterpret_cast<uint32_t*>(smem + C::HIST_OFF),
                                t + 1 < T, &s_sel, &s_tc[t]);
                GQ_STAMP();
            } else {
                for (int i = tid; i < (K >> 3); i += NT)
                    reinterpret_cast<uint4*>(skeys)[i] = reinterpret_cast<const uint4*>(xraw + (size_t)t * K)[i];
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
            // ---- per group and cut: keys above and keys equal (one token: every group's per-width counts follow
            //      from them; several tokens: only the ordered tie offsets are needed, and only if a cut splits)
            if (T == 1 || split) {
                uint16_t* tie = s_tie + (size_t)t * groups * 8;
#pragma unroll 1
                for (int g = warp; g < groups; g += VW) {
                    const uint2 kv = *reinterpret_cast<const uint2*>(skeys + g * GQ_G + 4 * lane);
                    int m[4];
                    keys4(kv, m);
                    uint32_t mine = 0;
#pragma unroll 1
                    for (int d = 0; d < nd; ++d) {
                        const int th = s_tc[t].thr[d];
                        uint32_t c2 = 0;  // keys above in the low half, keys equal in the high half
#pragma unroll
                        for (int i = 0; i < 4; ++i) c2 += (m[i] > th) ? 1u : ((m[i] == th) ? 0x10000u : 0u);
                        c2 = __reduce_add_sync(0xffffffffu, c2);
                        if (lane == d) mine = c2;
                    }
                    if (lane < 8) {
                        s_gt[g][lane] = (uint8_t)(mine & 0xFFFFu);
                        s_eq[g][lane] = (uint8_t)(mine >> 16);
                    }
                }
                __syncthreads();
                // ---- equal counts -> exclusive prefix over the groups (warp d scans cut d, 32 groups at a time)
#pragma unroll 1
                for (int d = warp; d < nd; d += VW) {
                    int carry = 0;
#pragma unroll 1
                    for (int g0 = 0; g0 < groups; g0 += 32) {
                        const int g = g0 + lane;
                        const int v = (g < groups) ? (int)s_eq[g][d] : 0;
                        const int incl = warp_incl_scan_i(v, lane);
                        if (g < groups) tie[g * 8 + d] = (uint16_t)(carry + incl - v);
                        carry += __shfl_sync(0xffffffffu, incl, 31);
                    }
                }
                __syncthreads();
            }
        }
        GQ_STAMP();
        if (T == 1) {
            // ---- keys above cut d in group g = gt + (split ? clamp(take - tie offset, 0, eq) : eq), and a row has
            //      >= w bits iff its key is above cut cw[w].  One thread per (group, width).
            const uint32_t split = s_tc[0].split;
#pragma unroll 1
            for (int i = tid; i < groups * 8; i += NT) {
                const int g = i >> 3, w = (i & 7) + 1, d = cp.cw[w];
                int above = 0;
                if (d >= 0) {
                    const int eq = s_eq[g][d];
                    above = s_gt[g][d];
                    if ((split >> d) & 1u) above += max(0, min(s_tc[0].take[d] - (int)s_tie[g * 8 + d], eq));
                    else above += eq;
                }
                s_gcnt[g][w] = (uint8_t)above;
                if (w == 1) {
                    s_gcnt[g][0] = GQ_G;
                    s_gcnt[g][9] = 0;
                }
            }
        } else {
            // ---- several tokens: the union width of a key is the maximum over the tokens: per-key widths, one warp
            //      per group
#pragma unroll 1
            for (int g = warp; g < groups; g += VW) {
                int bu[4] = {0, 0, 0, 0};
#pragma unroll 1
                for (int t = 0; t < T; ++t) {
                    int m[4], b[4];
                    keys4(*reinterpret_cast<const uint2*>(xraw + (size_t)t * K + g * GQ_G + 4 * lane), m);
                    widths4(m, &s_tc[t], cp.mult, nd, s_tie + ((size_t)t * groups + g) * 8, lane, b);
#pragma unroll
                    for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], b[i]);
                }
                int pos[4], ge[10];
                partition128(bu, lane, pos, ge);
                int myge = 0;
#pragma unroll
                for (int c = 0; c <= 9; ++c)
                    if (lane == c) myge = ge[c];
                if (lane < GQ_GCNT) s_gcnt[g][lane] = (uint8_t)(lane <= 9 ? myge : 0);
            }
        }
    }
    __syncthreads();
    // ---- exclusive prefix of the groups' costs (block scan, NT groups at a time)
    {
        int carry = 0;
#pragma unroll 1
        for (int g0 = 0; g0 < groups; g0 += NT) {
            const int g = g0 + tid;
            const int c = (g < groups) ? group_cost(*reinterpret_cast<const uint4*>(s_gcnt[g])) : 0;
            const int incl = warp_incl_scan_i(c, lane);
            if (lane == 31) s_wsum[warp] = incl;
            __syncthreads();
            if (warp == 0) {
                const int v = (lane < VW) ? s_wsum[lane] : 0;
                const int i2 = warp_incl_scan_i(v, lane);
                s_wsum[lane] = i2 - v;
                if (lane == 31) s_total = i2;
            }
            __syncthreads();
            if (g < groups) s_pref[g] = carry + s_wsum[warp] + incl - c;
            carry += s_total;
            if (g0 + NT < groups) __syncthreads();  // s_wsum is reused
        }
        if (tid == 0) s_pref[groups] = carry;
    }
    GQ_STAMP();
    __syncthreads();
    GQ_STAMP();

    // ================================================================== the warp's range of the tile's row stream
    int g_a, pos_a, g_b, pos_b;  // rows [(g_a, pos_a), (g_b, pos_b)) in stream order; g_b may be `groups`
    int G0 = 0;                  // first group of the CTA's range
    {
        const int total = s_pref[groups];
        const int S = Sx * VW, ws = sx * VW + warp;
        // total <= 256 * 128 * 20 < 2^20 and S <= 2^12 when it matters: 32-bit products (64-bit division is ~100 instructions)
        const bool small = total < (1 << 20) && S <= (1 << 12);
        auto bound = [&](int i) {
            return small ? (int)(((uint32_t)total * (uint32_t)i) / (uint32_t)S) : (int)(((long long)total * i) / S);
        };
        // the group holding cost c = the last g with pref[g] <= c (g = groups when c == total): 8-way blocks first
        auto locate_group = [&](int c) {
            const int gi = min(8 * lane, groups);
            const uint32_t b1 = __ballot_sync(0xffffffffu, 8 * lane <= groups && s_pref[gi] <= c);
            const int blk = 31 - __clz(b1);  // lane 0 always qualifies (pref[0] = 0 <= c)
            const int gj = min(8 * blk + (lane & 7), groups);
            const uint32_t b2 = __ballot_sync(0xffffffffu, lane < 8 && 8 * blk + lane <= groups && s_pref[gj] <= c);
            return 8 * blk + (31 - __clz(b2));
        };
        const int lo = bound(ws), hi = bound(ws + 1);
        g_a = locate_group(lo);
        pos_a = (g_a < groups) ? pos_from_cost(s_gcnt[g_a], lo - s_pref[g_a], lane) : 0;
        g_b = locate_group(hi);
        pos_b = (g_b < groups) ? pos_from_cost(s_gcnt[g_b], hi - s_pref[g_b], lane) : 0;
        if (T == 1 && MODE != MODE_SCHED) {
            // ---- the lists of the first GLC groups of the CTA's range are made once, by one warp each, from the keys
            //      still in shared memory (every warp of the CTA walks one or two of the same few groups)
            const int cta_hi = bound((sx + 1) * VW);
            G0 = locate_group(bound(sx * VW));
#pragma unroll 1
            for (int gi = warp; gi < GLC; gi += VW) {
                const int g = G0 + gi;
                if (g >= groups || s_pref[g] >= cta_hi) break;
                const uint16_t* skeys = reinterpret_cast<const uint16_t*>(smem + C::KEYS_OFF);
                const uint2 xv = *reinterpret_cast<const uint2*>(skeys + g * GQ_G + 4 * lane);
                int m[4], b[4], pos[4], ge[10];
                keys4(xv, m);
                widths4(m, &s_tc[0], cp.mult, nd, s_tie + (size_t)g * 8, lane, b);
                partition128(b, lane, pos, ge);
                const uint32_t xs[4] = {xv.x & 0xFFFFu, xv.x >> 16, xv.y & 0xFFFFu, xv.y >> 16};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    s_glist[gi][pos[i]] = (uint32_t)(4 * lane + i) | ((uint32_t)b[i] << 8) | ((uint32_t)b[i] << 12) | (xs[i] << 16);
            }
        }
    }
    GQ_STAMP();
    __syncthreads();  // from here on the warp regions belong to their warps
    GQ_STAMP();

    // the warp's accumulator tile starts at zero
    {
        float4* yz = reinterpret_cast<float4*>(yacc);
#pragma unroll 1
        for (int i = lane; i < T * YSLOT / 4; i += 32) yz[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }

    // per-lane copy geometry: lane copies chunk `seg` (16 B) of plane pj (and pj + 4); pjx = 99 disables the lane
    const int pj = lane >> 3, seg = lane & 7;
    const bool chunk_ok = A16 ? (tile * 32 + seg * 4 < words) : active;
    const int pjx = chunk_ok ? (A16 ? pj : 0) : 99;
    const uint8_t* lane_src = reinterpret_cast<const uint8_t*>(planes) +
                              (A16 ? (size_t)pj * pbytes + (size_t)(tile * 32 + seg * 4) * 4 : (size_t)word * 4);
    const uint32_t lane_dst = A16 ? ring_s + pj * 128 + seg * 16 : ring_s + lane * 4;
    const size_t hi_off = 4 * pbytes;  // planes 4..7 of the same row

    // ================================================================== list: pieces of group segments appended ahead of the copies
    // entry = {word, byte offset of the row inside a plane}; word of a row: the gsched format; word of a scale/zero
    // chunk: ENTRY_SZ | chunk L (bits 0..1) | group (bits 8..15) | X/Phi slot (bits 16..19).
    constexpr int LN = C::LISTN;
    constexpr int SUBMAX = LN / 2 - 4;  // rows appended per call: the list holds a piece + what is still in flight
    uint2* list = reinterpret_cast<uint2*>(wbase + C::LIST_OFF);              // [LN]
    uint32_t* tok = reinterpret_cast<uint32_t*>(wbase + C::LIST_OFF + LN * 8);  // [T-1][LN] words of tokens 1..T-1
    float2* xphi = reinterpret_cast<float2*>(wbase + C::XPHI_OFF);            // [16][T] {X, Phi} of the segments in flight
    int app = 0;                  // list entries appended so far
    int iv = 0, cv = 0;           // next entry to issue / to consume
    int seg_g = g_a, seg_p = pos_a, seg_p1 = 0, segj = 0;  // group being appended, next position, end position
    float Xrun[T], Prun[T];       // X = sum x, Phi = sum x phi_b over the segment's rows appended so far
#pragma unroll
    for (int t = 0; t < T; ++t) Xrun[t] = Prun[t] = 0.f;

    auto seg_end = [&](int g) { return (g == g_b) ? min(pos_b, (int)s_gcnt[g][1]) : (int)s_gcnt[g][1]; };
    // skips groups without rows for this warp; false when the range is exhausted
    auto more_rows = [&]() {
        while (seg_g < groups && seg_g <= g_b) {
            seg_p1 = seg_end(seg_g);
            if (seg_p < seg_p1) return true;
            ++seg_g;
            seg_p = 0;
        }
        return false;
    };

    // appends up to SUBMAX rows of the current group (+ the 4 chunk entries when they were its last)
    auto append_piece = [&]() {
        const int g = seg_g, p0 = seg_p;
        const int n = min(seg_p1 - p0, SUBMAX);
        if (MODE == MODE_SCHED) {
#pragma unroll 1
            for (int i = lane; i < n; i += 32) {
                list[(app + i) & (LN - 1)].x = gsched[(size_t)g * GQ_G + p0 + i];
#pragma unroll
                for (int t = 1; t < T; ++t)
                    tok[(t - 1) * LN + ((app + i) & (LN - 1))] = gsched[(size_t)t * K + g * GQ_G + p0 + i];
            }
        } else if (T == 1 && g - G0 < GLC) {
#pragma unroll 1
            for (int i = lane; i < n; i += 32) list[(app + i) & (LN - 1)].x = s_glist[g - G0][p0 + i];
        } else {
            uint2 xv[T];
            int bt[T][4], bu[4] = {0, 0, 0, 0}, pos[4], ge[10];
#pragma unroll
            for (int t = 0; t < T; ++t) {
                xv[t] = *reinterpret_cast<const uint2*>(xraw + (size_t)t * K + g * GQ_G + 4 * lane);
                int m[4];
                keys4(xv[t], m);
                widths4(m, &s_tc[t], cp.mult, nd, s_tie + ((size_t)t * groups + g) * 8, lane, bt[t]);
#pragma unroll
                for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], bt[t][i]);
            }
            partition128(bu, lane, pos, ge);
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const uint32_t xs[4] = {xv[t].x & 0xFFFFu, xv[t].x >> 16, xv[t].y & 0xFFFFu, xv[t].y >> 16};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (pos[i] >= p0 && pos[i] < p0 + n) {
                        const uint32_t w = (uint32_t)(4 * lane + i) | ((uint32_t)bt[t][i] << 8) | ((uint32_t)bu[i] << 12) |
                                           (xs[i] << 16);
                        const int idx = (app + pos[i] - p0) & (LN - 1);
                        if (t == 0) list[idx].x = w;
                        else tok[(t - 1) * LN + idx] = w;
                    }
            }
        }
        __syncwarp();
        // ---- common to all forms (same lane <-> position mapping, so every form sums X and Phi in the same order):
        //      row byte offsets, and this piece's share of the segment's X and Phi
        float Xp[T], Pp[T];
#pragma unroll
        for (int t = 0; t < T; ++t) Xp[t] = Pp[t] = 0.f;
        const uint32_t gbase = (uint32_t)g * GQ_G * rowbytes;
#pragma unroll 1
        for (int i = lane; i < n; i += 32) {
            const int idx = (app + i) & (LN - 1);
            const uint32_t w0 = list[idx].x;
            list[idx].y = gbase + (w0 & 0x7Fu) * rowbytes;
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const uint32_t w = (t == 0) ? w0 : tok[(t - 1) * LN + idx];
                const int b = (w >> 8) & 15;
                if (b > 0) {
                    const float xf = __half2float(__ushort_as_half((uint16_t)(w >> 16)));
                    Xp[t] += xf;
                    Pp[t] = fmaf(xf, (float)(0x80 >> b), Pp[t]);  // phi_b = 2^(7-b), phi_8 = 0
                }
            }
        }
#pragma unroll
        for (int t = 0; t < T; ++t) {
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                Xp[t] += __shfl_xor_sync(0xffffffffu, Xp[t], d);
                Pp[t] += __shfl_xor_sync(0xffffffffu, Pp[t], d);
            }
            Xrun[t] += Xp[t];
            Prun[t] += Pp[t];
        }
        app += n;
        seg_p = p0 + n;
        if (seg_p == seg_p1) {  // the warp's last row of this group: scale/zero chunks, X and Phi, next group
            const int slot = segj & 15;
            if (lane < 4)
                list[(app + lane) & (LN - 1)] =
                    make_uint2(ENTRY_SZ | (uint32_t)lane | ((uint32_t)slot << 16) | ((uint32_t)g << 8), 0u);
            if (lane < T) {
                float xs_ = 0.f, ps_ = 0.f;
#pragma unroll
                for (int t = 0; t < T; ++t)
                    if (lane == t) {
                        xs_ = Xrun[t];
                        ps_ = Prun[t];
                    }
                xphi[slot * T + lane] = make_float2(xs_, ps_);
            }
#pragma unroll
            for (int t = 0; t < T; ++t) Xrun[t] = Prun[t] = 0.f;
            app += 4;
            ++segj;
            ++seg_g;
            seg_p = 0;
        }
        __syncwarp();
    };

    // issues list entry iv into ring slot iv mod RING (one cp.async group, empty past the end of the list)
    auto issue_one = [&]() {
        if (iv < app) {
            const uint2 e = list[iv & (LN - 1)];
            const uint32_t so = (uint32_t)(iv & (RING - 1)) * SLOT_BYTES;
            if (!(e.x & ENTRY_SZ)) {
                const int b = (e.x >> 12) & 15;
                const uint8_t* src = lane_src + e.y;
                const uint32_t dst = lane_dst + so;
                if (A16) {
                    if (pjx < b) cp_async16(dst, src);
                    if (pjx + 4 < b) cp_async16(dst + 512, src + hi_off);
                } else {
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        if (pjx + j < b) cp_async4(dst + j * 128, src + j * pbytes);
                }
            } else if (active) {
                const size_t gn = (size_t)((e.x >> 8) & 0xFFu) * N + (size_t)word * 32 + 8 * (e.x & 3u);
                cp_async16(ring_s + so + lane * 16, scales + gn);
                cp_async16(ring_s + so + 512 + lane * 16, zeros + gn);
            }
            ++iv;
        }
        cp_async_commit();
    };

    GQ_STAMP();
    while (app - iv < RING && more_rows()) append_piece();
    GQ_STAMP();
#pragma unroll 1
    for (int i = 0; i < RING - 2; ++i) issue_one();
    GQ_STAMP();

    float acc[T][32];
    float X[T], Phi[T];
#pragma unroll
    for (int t = 0; t < T; ++t) {
        X[t] = Phi[t] = 0.f;
#pragma unroll
        for (int c = 0; c < 32; ++c) acc[t][c] = 0.f;
    }

    // one row: plane words of its ring slot -> 32 truncated codes -> 32 FMAs per token
    auto consume = [&](auto b_tag, uint32_t m, int v) {
        constexpr int B = decltype(b_tag)::value;
        const uint32_t* slot = reinterpret_cast<const uint32_t*>(ring + (uint32_t)(v & (RING - 1)) * SLOT_BYTES) + lane;
        uint32_t Wd[8], V[8];
        if (B == 8) {
#pragma unroll
            for (int j = 0; j < 8; ++j) Wd[j] = slot[j * 32];
            gather<8>(Wd, V);
        } else if (B == 4) {
#pragma unroll
            for (int j = 0; j < 4; ++j) Wd[j] = slot[j * 32];
            gather<4>(Wd, V);
        } else if (B == 2) {
#pragma unroll
            for (int j = 0; j < 2; ++j) Wd[j] = slot[j * 32];
            gather<2>(Wd, V);
        } else {  // stale slot words beyond the row's planes are masked off
            const int bb = (m >> 12) & 15;
#pragma unroll
            for (int j = 0; j < 8; ++j) Wd[j] = (j < bb) ? slot[j * 32] : 0u;
            gather<8>(Wd, V);
        }
        if (T == 1) {
            accumulate_row(V, (uint16_t)(m >> 16), acc[0]);
        } else {
            const int b = (B != 0) ? B : (int)((m >> 12) & 15);
            uint32_t H[16];
            if (T >= 3) {
                // 3 or 4 tokens: the bytes are widened to fp16 lanes once per row; a token narrower than the union
                // masks the 16-bit lanes instead of the bytes
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    H[2 * r] = __byte_perm(V[r], 0u, 0x4140);
                    H[2 * r + 1] = __byte_perm(V[r], 0u, 0x4342);
                }
            }
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const uint32_t e = (t == 0) ? m : tok[(t - 1) * LN + (v & (LN - 1))];
                const int bt = (e >> 8) & 15;  // this token's own width (<= b, the union)
                if (bt == 0) continue;         // warp-uniform
                const uint16_t xh = (uint16_t)(e >> 16);
                if (T == 2) {
                    if (bt == b) {
                        accumulate_row(V, xh, acc[t]);
                    } else {
                        const uint32_t mask = 0x01010101u * ((0xFF00u >> bt) & 0xFFu);
                        uint32_t Vm[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) Vm[j] = V[j] & mask;
                        accumulate_row(Vm, xh, acc[t]);
                    }
                } else {
                    const uint32_t mask = (bt == b) ? 0x00FF00FFu : 0x00010001u * ((0xFF00u >> bt) & 0xFFu);
#pragma unroll
                    for (int r = 0; r < 8; ++r) {
                        const uint32_t h01 = H[2 * r] & mask, h23 = H[2 * r + 1] & mask;
                        fhfma_lo(acc[t][4 * r + 0], h01, xh);
                        fhfma_hi(acc[t][4 * r + 1], h01, xh);
                        fhfma_lo(acc[t][4 * r + 2], h23, xh);
                        fhfma_hi(acc[t][4 * r + 3], h23, xh);
                    }
                }
            }
        }
    };

    // scale/zero chunk L of the segment: columns 8L..8L+7 of the lane (acc[4r + L], r = 0..7) leave the accumulators
    auto chunk = [&](auto l_tag, uint32_t e, int v) {
        constexpr int L = decltype(l_tag)::value;
        if (L == 0) {  // the segment's X and Phi (made when its list was)
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const float2 xp = xphi[((e >> 16) & 15u) * T + t];
                X[t] = xp.x;
                Phi[t] = xp.y;
            }
        }
        if (active) {
            const uint8_t* sz = ring + (uint32_t)(v & (RING - 1)) * SLOT_BYTES + lane * 16;
            const uint4 sv = *reinterpret_cast<const uint4*>(sz);
            const uint4 zv = *reinterpret_cast<const uint4*>(sz + 512);
            const uint32_t su[4] = {sv.x, sv.y, sv.z, sv.w}, zu[4] = {zv.x, zv.y, zv.z, zv.w};
            float sf[8], zf[8];
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&su[h]));
                const float2 c = __half22float2(*reinterpret_cast<const __half2*>(&zu[h]));
                sf[2 * h] = a.x; sf[2 * h + 1] = a.y;
                zf[2 * h] = c.x; zf[2 * h + 1] = c.y;
            }
#pragma unroll
            for (int t = 0; t < T; ++t)
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    float* dst = yacc + t * YSLOT + (8 * L + r) * 33 + lane;
                    *dst = fmaf(zf[r], X[t], fmaf(sf[r], fmaf(acc[t][4 * r + L], CODE_SCALE, Phi[t]), *dst));
                }
        }
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int r = 0; r < 8; ++r) acc[t][4 * r + L] = 0.f;
    };

    // ================================================================== stream
    using std::integral_constant;
#pragma unroll 1
    for (;;) {
        while (app - iv < RING && more_rows()) append_piece();
        if (cv == app) break;
        // entries that can be consumed before the list has to grow again (the copies run RING-2 entries ahead)
        const int stop = more_rows() ? max(cv + 1, app - 2 * RING + 3) : app;
        // runs of rows of one width class keep the accumulators in place (one tight loop per class; rows are sorted by
        // width inside a segment, so a run is long)
        uint32_t e = list[cv & (LN - 1)].x;
#pragma unroll 1
        while (cv < stop) {
            auto run = [&](auto b_tag) {
                constexpr int B = decltype(b_tag)::value;
#pragma unroll 1
                do {
                    cp_async_wait<RING - 3>();
                    __syncwarp();
                    issue_one();
                    consume(b_tag, e, cv);
                    ++cv;
                    e = list[cv & (LN - 1)].x;
                } while (cv < stop && !(e & ENTRY_SZ) &&
                         (B != 0 ? (int)((e >> 12) & 15) == B
                                 : ((e >> 12) & 15) != 8 && ((e >> 12) & 15) != 4 && ((e >> 12) & 15) != 2));
            };
            if (e & ENTRY_SZ) {
                cp_async_wait<RING - 3>();
                __syncwarp();
                issue_one();
                const int L = (int)(e & 3u);
                if (L == 0) chunk(integral_constant<int, 0>{}, e, cv);
                else if (L == 1) chunk(integral_constant<int, 1>{}, e, cv);
                else if (L == 2) chunk(integral_constant<int, 2>{}, e, cv);
                else chunk(integral_constant<int, 3>{}, e, cv);
                ++cv;
                e = list[cv & (LN - 1)].x;
            } else {
                const int b = (e >> 12) & 15;
                if (b == 8) run(integral_constant<int, 8>{});
                else if (b == 4) run(integral_constant<int, 4>{});
                else if (b == 2) run(integral_constant<int, 2>{});
                else run(integral_constant<int, 0>{});
            }
        }
    }
    cp_async_wait<0>();
    GQ_STAMP();
    __syncthreads();
    GQ_STAMP();

    // ================================================================== CTA epilogue: fixed-order sum over the warps
    float* out = (fused && Sx == 1) ? y : part + (size_t)sx * T * N;
#pragma unroll 1
    for (int t = 0; t < T; ++t)
#pragma unroll 1
        for (int c = tid; c < TILE_COLS; c += NT) {  // column inside the tile
            const int n = tile * TILE_COLS + c;
            if (n < N) {
                const int idx = (c & 31) * 33 + (c >> 5);
                float A = 0.f;
#pragma unroll
                for (int w = 0; w < VW; ++w)
                    A += *reinterpret_cast<const float*>(smem + w * C::WARP_BYTES + C::YACC_OFF + (t * YSLOT + idx) * 4);
                out[(size_t)t * N + n] = A;
            }
        }
    if (fused && Sx > 1) {
        __syncthreads();  // the CTA's partial is complete ...
        if (tid == 0) {
            __threadfence();  // ... and (fence cumulativity over the barrier) visible device-wide before its ticket
            const int last = (atomicAdd(&tickets[tile], 1) == Sx - 1);
            if (last) __threadfence();  // acquire side: the other CTAs' partials, read below with ld.global.cg
            s_last = last;
        }
        __syncthreads();
        if (s_last) {
            // float2 columns spread over all the CTA's threads, 16 partials per column in flight, added in the fixed
            // order s = 0..Sx-1
            constexpr int BATCH = 16;
#pragma unroll 1
            for (int t = 0; t < T; ++t)
#pragma unroll 1
                for (int c = 2 * tid; c < TILE_COLS; c += 2 * NT) {
                    const int n = tile * TILE_COLS + c;
                    if (n >= N) break;
                    float2 a = make_float2(0.f, 0.f);
#pragma unroll 1
                    for (int s0 = 0; s0 < Sx; s0 += BATCH) {
                        float2 v[BATCH];
#pragma unroll
                        for (int j = 0; j < BATCH; ++j)
                            if (s0 + j < Sx)
                                v[j] = __ldcg(reinterpret_cast<const float2*>(part + ((size_t)(s0 + j) * T + t) * N + n));
#pragma unroll
                        for (int j = 0; j < BATCH; ++j)
                            if (s0 + j < Sx) {
                                a.x += v[j].x;
                                a.y += v[j].y;
                            }
                    }
                    *reinterpret_cast<float2*>(y + (size_t)t * N + n) = a;
                }
            if (tid == 0) tickets[tile] = 0;  // ready for the next launch on this workspace
        }
    }
#ifdef GQ_TIMING
    GQ_STAMP();
    if (lane == 0 && (warp == 0 || warp == VW - 1) && blockIdx.x == 0 && (blockIdx.y == 0 || blockIdx.y == gridDim.y - 1)) {
        if (MODE == MODE_RANK && warp == 0 && blockIdx.y == 0) {
            printf("select:");
            for (int i = 1; i < g_sel_n; ++i) printf(" %lld", g_sel_stamp[i] - g_sel_stamp[0]);
            printf("\n");
        }
        printf("blk %3d warp %2d entries %3d:", blockIdx.y, warp, cv);
        for (int i = 1; i < nst; ++i) printf(" %6lld", stamp[i] - stamp[0]);
        printf("\n");
    }
#endif
}

// y[t][n] = sum_{s=0}^{S-1} part[s][t][n], sequentially in s: the same order as the fused second pass, so the
// two-launch form returns the same bits.
__global__ void __launch_bounds__(256)
vmm_reduce_kernel(const float* __restrict__ part, int S, int T, int N, float* __restrict__ y);

template <int T, int VW, bool A16, int MODE>
static int launch_impl(const VmmArgs& a, const VmmPlan& pl) {
    using C = Cfg<T, VW>;
    const size_t smem = (size_t)C::BASE_BYTES + (MODE == MODE_SCHED ? 0 : (size_t)T * (a.K / GQ_G) * 16);
    // the attribute belongs to the device: set it on every launch (cheap, legal during stream capture)
    if (cudaFuncSetAttribute(vmm_kernel<T, VW, A16, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
        cudaSuccess)
        return GRINQH_ERR_CUDA;
    dim3 grid(pl.col_tiles, pl.Sx);
    const cudaError_t e =
        launch_pdl(vmm_kernel<T, VW, A16, MODE>, grid, dim3(C::NT), smem, a.st, a.K, a.N, pl.Sx, a.fused, a.planes,
                   (const __half*)a.scales, (const __half*)a.zeros, a.gsched, a.gcnt_ge, a.xraw, a.cp,
                   (float*)((char*)a.workspace + TICKET_BYTES), (int*)a.workspace, a.y);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

int launch_vmm_multi(const VmmArgs& a, const VmmPlan& pl);  // vmm_multi.cu: T = 2..4

}  // namespace gq
