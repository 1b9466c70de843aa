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
#include "vmm_args.cuh"

namespace gq {

constexpr int TILE_COLS = 1024;
constexpr int SLOT_BYTES = 1024;   // 8 planes x 128 B
constexpr int YSLOT = 32 * 33;     // one warp's 1024 sums, padded: column 32*l + c lives at c*33 + l
constexpr int GLC = 8;             // group lists a CTA builds once for all its warps (one token, in-kernel assignment)
constexpr int MAXG = GQ_MAX_K / GQ_G;
constexpr uint32_t ENTRY_SZ = 0x80u;  // list entry is a scale/zero chunk (bits 0..1 = chunk); rows use bits 0..6


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
    static constexpr int MBAR_OFF = XPHI_OFF + 16 * T * 8;  // RING mbarriers (bulk-copy form)
    static constexpr int WARP_BYTES = MBAR_OFF + RING * 8;
    // the assignment prologue aliases the warp regions: one token's keys and the select's 64-KB histogram
    static constexpr int KEYS_OFF = 0;
    static constexpr int HIST_OFF = GQ_MAX_K * 2;
    static constexpr int BASE_BYTES = cmax(VW * WARP_BYTES, HIST_OFF + 65536);  // the tie offsets live behind
    static_assert(WARP_BYTES % 16 == 0, "warp regions stay 16-byte aligned");
    static_assert(T == 1 || VW == 8, "several tokens: 8 warps (registers: acc[T][32])");
};

struct VmmPlan {
    int col_tiles;  // ceil(N / 1024)
    int Sx;         // CTAs (= split-K partials) per column tile
    int vw;         // warps per CTA
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

// TMA bulk copies (cp.async.bulk, SASS UBLKCP) completing on an mbarrier in shared memory
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t mbar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "GQ_WAIT:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra GQ_DONE;\n\t"
        "bra GQ_WAIT;\n\t"
        "GQ_DONE:\n\t}" ::"r"(mbar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(mbar) : "memory");
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

// A16: every plane row is 16-byte aligned (N % 128 == 0) -> LDGSTS.128, 4 planes per instruction;
// otherwise each lane copies its own word of every plane with 4-byte cp.async.
//
// gsched[t][g*128 + p] (MODE_SCHED, written by grinqh_assign) is position p of group g's list for token t:
//   bits 0..7 local row r | 8..11 b_t (token's width) | 12..15 b (union width = planes fetched) | 16..31 x_t[r] fp16
// The in-kernel forms build the same entries from xraw.
template <int T, int VW, bool A16, int MODE, bool BULK, bool SEG2>
__global__ void __launch_bounds__(VW * 32, 1)
vmm_kernel(int K, int N, int Sx, int fused, int bmax, const uint32_t* __restrict__ planes, const __half* __restrict__ scales,
           const __half* __restrict__ zeros, const uint32_t* __restrict__ gsched, const uint8_t* __restrict__ gcnt_ge,
           const uint16_t* __restrict__ xraw, CutParams cp, float* __restrict__ part, int* __restrict__ tickets,
           float* __restrict__ y) {
    using C = Cfg<T, VW>;
    constexpr int RING = C::RING, NT = C::NT;
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ uint32_t s_glist[GLC][GQ_G];  // lists of the first GLC groups of this CTA's range
    __shared__ __align__(16) TokenCuts s_tc[T];
    __shared__ SelectScratch s_sel;
    __shared__ int s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, sx = blockIdx.y;
    const int words = N >> 5;
    const int word = tile * 32 + lane;
    const bool active = word < words;
    // bytes of one row of one plane (or of one 2-bit segment: twice as many), and of one whole plane / segment
    const uint32_t rowbytes = (uint32_t)words * (SEG2 ? 8u : 4u);
    const size_t pbytes = (size_t)K * rowbytes;
    static_assert(!SEG2 || (T == 1 && A16 && !BULK), "the 2-bit-segment store: one token, aligned rows, cp.async copies");
    const int groups = K / GQ_G;
    const int nd = cp.nd;

    uint8_t* wbase = smem + warp * C::WARP_BYTES;
    const uint8_t* ring = wbase + C::RING_OFF;
    float* yacc = reinterpret_cast<float*>(wbase + C::YACC_OFF);
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(wbase + C::RING_OFF);
    uint16_t* s_tie = reinterpret_cast<uint16_t*>(smem + C::BASE_BYTES);  // [T][groups][8] ordered tie offsets

#ifdef GQ_TIMING
    unsigned long long gt0, gt2 = 0;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(gt0));
    long long stamp[16];
    int nst = 0;
#define GQ_STAMP() stamp[nst++] = clock64()
#else
#define GQ_STAMP()
#endif
    GQ_STAMP();
    pdl_launch_dependents();

    // ================================================================== prologue: the cuts and the ordered tie offsets
    if (MODE == MODE_SCHED) {
        pdl_wait();  // nothing global is touched before the previous kernel has finished
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
                // ---- a cut splits a run of equal keys: per group the number of keys equal to each such cut (thread =
                //      8 consecutive keys, 16 threads = one group: a half-warp reduction), then their exclusive prefix
                //      over the groups = the ordered tie offsets (ties go to the lower index)
                uint16_t* tie = s_tie + (size_t)t * groups * 8;
#pragma unroll 1
                for (int c0 = warp * 32; c0 < (K >> 3); c0 += NT) {  // (warp-uniform bounds: every lane shuffles)
                    const int c = c0 + lane;
                    const bool valid = c < (K >> 3);
                    const uint4 kv = valid ? reinterpret_cast<const uint4*>(skeys)[c] : make_uint4(~0u, ~0u, ~0u, ~0u);
                    const uint32_t kw[4] = {kv.x, kv.y, kv.z, kv.w};
                    uint32_t pk[2] = {0u, 0u};  // equal counts of cuts 0..3 and 4..7, 8 bits each (a group has 128 keys)
#pragma unroll
                    for (int d = 0; d < 8; ++d) {
                        if (d < nd) {  // uniform
                            const uint32_t th = (uint32_t)s_tc[t].thr[d];
                            uint32_t ce = 0;
#pragma unroll
                            for (int j = 0; j < 8; ++j) ce += (((kw[j >> 1] >> (16 * (j & 1))) & 0x7FFFu) == th) ? 1u : 0u;
                            pk[d >> 2] += ce << (8 * (d & 3));
                        }
                    }
#pragma unroll
                    for (int o = 8; o >= 1; o >>= 1) {  // the 16 lanes of a group
                        pk[0] += __shfl_xor_sync(0xffffffffu, pk[0], o);
                        if (nd > 4) pk[1] += __shfl_xor_sync(0xffffffffu, pk[1], o);
                    }
                    if (valid && (lane & 15) < 8) {
                        const int d = lane & 15;
                        tie[(c >> 4) * 8 + d] = (uint16_t)((pk[d >> 2] >> (8 * (d & 3))) & 0xFFu);
                    }
                }
                __syncthreads();
#pragma unroll 1
                for (int d = warp; d < nd; d += VW) {  // (up to 8 rounds of 32 groups: independent scans, then the carries)
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
    }

    // ================================================================== the warp's range of the tile's slots
    // Group g owns slots 128 g .. 128 g + 127; slot s holds position brev7(s) of the group's (width desc, index asc)
    // list, so ANY run of consecutive slots sees the group's width mix (and its share of the b = 0 rows, which are
    // skipped): warp slot ws of the tile's S = Sx * VW warps takes slots [ws K / S, (ws + 1) K / S) — balanced without
    // knowing a single width, so nothing has to be counted or scanned before the first row can be fetched.
    const int S = Sx * VW, ws = sx * VW + warp;
    const int slot_lo = (int)(((uint32_t)K * (uint32_t)ws) / (uint32_t)S);        // K <= 2^15, S < 2^17
    const int slot_hi = (int)(((uint32_t)K * (uint32_t)(ws + 1)) / (uint32_t)S);
    const int G0 = (int)(((uint32_t)K * (uint32_t)(sx * VW)) / (uint32_t)S) >> 7;  // first group of the CTA's range
    if (T == 1 && MODE != MODE_SCHED) {
        // ---- the lists of the first GLC groups of the CTA's range are made once, by one warp each (every warp of the
        //      CTA walks one or two of the same few groups)
        const int cta_hi = (int)(((uint32_t)K * (uint32_t)((sx + 1) * VW)) / (uint32_t)S);
#pragma unroll 1
        for (int gi = warp; gi < GLC; gi += VW) {
            const int g = G0 + gi;
            if (g >= groups || g * GQ_G >= cta_hi) break;
            const uint2 xv = (MODE == MODE_RANK)
                                 ? *reinterpret_cast<const uint2*>(reinterpret_cast<const uint16_t*>(smem + C::KEYS_OFF) +
                                                                   g * GQ_G + 4 * lane)
                                 : *reinterpret_cast<const uint2*>(xraw + g * GQ_G + 4 * lane);
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
    GQ_STAMP();
    __syncthreads();  // from here on the warp regions belong to their warps
    GQ_STAMP();

    // per-lane copy geometry: lane copies chunk `seg` (16 B) of plane pj (and pj + 4); pjx = 99 disables the lane.
    // 2-bit segments: a segment row of the tile is 256 B: lanes 16 j .. 16 j + 15 copy segment j (and j + 2).
    const int pj = SEG2 ? (lane >> 4) : (lane >> 3), seg = SEG2 ? (lane & 15) : (lane & 7);
    const bool chunk_ok = SEG2 ? (tile * 64 + seg * 4 < 2 * words) : A16 ? (tile * 32 + seg * 4 < words) : active;
    const int pjx = chunk_ok ? (A16 ? pj : 0) : 99;
    const uint8_t* lane_src = reinterpret_cast<const uint8_t*>(planes) +
                              (SEG2 ? (size_t)pj * pbytes + (size_t)(tile * 64 + seg * 4) * 4
                               : A16 ? (size_t)pj * pbytes + (size_t)(tile * 32 + seg * 4) * 4
                                     : (size_t)word * 4);
    const uint32_t lane_dst = SEG2 ? ring_s + pj * 256 + seg * 16 : A16 ? ring_s + pj * 128 + seg * 16 : ring_s + lane * 4;
    const size_t hi_off = (SEG2 ? 2 : 4) * pbytes;  // planes 4..7 (segments 2, 3) of the same row
    // 2-bit segments with b_max < 8: the codes are left-aligned in the byte, so everything is 2^(8 - b_max) too large
    const float code_scale = SEG2 ? CODE_SCALE / (float)(1 << (8 - bmax)) : CODE_SCALE;
    // bulk-copy form: lane j copies the whole 128-byte segment of plane j with one cp.async.bulk; slot v mod RING has
    // its own mbarrier (one arrival = the expect_tx of lane 0, then the bytes)
    const uint32_t mbar_s = (uint32_t)__cvta_generic_to_shared(wbase + C::MBAR_OFF);
    const uint32_t segbytes = (uint32_t)min(128, max(0, (int)rowbytes - tile * 128));
    const uint8_t* bulk_src = reinterpret_cast<const uint8_t*>(planes) + (size_t)lane * pbytes + (size_t)tile * 128;
    if (BULK) {
        if (lane == 0) {
#pragma unroll 1
            for (int i = 0; i < RING; ++i) mbar_init(mbar_s + i * 8, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncwarp();
    }

    // ================================================================== list: pieces of group segments appended ahead of the copies
    // entry = {word, byte offset of the row inside a plane}; word of a row: the gsched format; word of a scale/zero
    // chunk: ENTRY_SZ | chunk L (bits 0..1) | group (bits 8..15) | X/Phi slot (bits 16..19).
    constexpr int LN = C::LISTN;
    uint2* list = reinterpret_cast<uint2*>(wbase + C::LIST_OFF);              // [LN]
    uint32_t* tok = reinterpret_cast<uint32_t*>(wbase + C::LIST_OFF + LN * 8);  // [T-1][LN] words of tokens 1..T-1
    float2* xphi = reinterpret_cast<float2*>(wbase + C::XPHI_OFF);            // [16][T] {X, Phi} of the segments in flight
    int app = 0;                  // list entries appended so far
    int iv = 0, cv = 0;           // next entry to issue / to consume
    int seg_s = slot_lo;          // next slot to append (a piece = the slots of one half of one group's positions)
    int seg_half = 0, segj = 0;
    bool seg_rows = false;        // the current segment has appended at least one row
    uint32_t gw[T][4];            // the current group: words of the lane's 4 rows / positions, their positions,
    int gpos[4], gnz = 0;         // whether they are in the warp's slots, rows with b > 0
    bool gin[4];
    float Xrun[T], Prun[T];       // X = sum x, Phi = sum x phi_b over the segment's rows appended so far
#pragma unroll
    for (int t = 0; t < T; ++t) Xrun[t] = Prun[t] = 0.f;

    auto more_rows = [&]() { return seg_s < slot_hi; };

    // appends the warp's rows of the current group whose positions lie in half `seg_half` (positions 64 h .. 64 h + 63),
    // in position order (so width classes stay together), + the 4 chunk entries after the second half
    auto append_piece = [&]() {
        const int g = seg_s >> 7;
        const int a = seg_s & 127, b_ = min(slot_hi - g * GQ_G, GQ_G);  // the warp's slots of this group: [a, b_)
        // lane l looks at positions 4 l .. 4 l + 3: brev7(4 l + i) = (brev2(i) << 5) | brev5(l)
        const bool direct = MODE == MODE_SCHED || (T == 1 && g - G0 < GLC);  // the list exists: position = 4 lane + i
        if (seg_half == 0) {  // the group's words are fetched / made once and kept for both halves
            if (direct) {
                const int rl = (int)(__brev((uint32_t)lane) >> 27);
                const int sl[4] = {rl, 64 + rl, 32 + rl, 96 + rl};
                // (rows with b = 0 sit at the end of the list and say so themselves: no count is needed)
                gnz = GQ_G;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    gpos[i] = 4 * lane + i;
                    bool in = sl[i] >= a && sl[i] < b_;
#pragma unroll
                    for (int t = 0; t < T; ++t)
                        gw[t][i] = !in ? 0u
                                   : (MODE == MODE_SCHED) ? gsched[(size_t)t * K + g * GQ_G + gpos[i]]
                                                          : s_glist[g - G0][gpos[i]];
                    gin[i] = in && ((gw[0][i] >> 12) & 15u) != 0u;
                }
            } else {
                uint2 xv[T];
                int bt[T][4], bu[4], ge[10];
#pragma unroll
                for (int i = 0; i < 4; ++i) bu[i] = 0;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    xv[t] = *reinterpret_cast<const uint2*>(xraw + (size_t)t * K + g * GQ_G + 4 * lane);
                    int m[4];
                    keys4(xv[t], m);
                    widths4(m, &s_tc[t], cp.mult, nd, s_tie + ((size_t)t * groups + g) * 8, lane, bt[t]);
#pragma unroll
                    for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], bt[t][i]);
                }
                partition128(bu, lane, gpos, ge);
                gnz = ge[1];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int s_ = (int)(__brev((uint32_t)gpos[i]) >> 25);
                    gin[i] = s_ >= a && s_ < b_ && gpos[i] < gnz;
#pragma unroll
                    for (int t = 0; t < T; ++t) {
                        const uint32_t xs = (i == 0) ? (xv[t].x & 0xFFFFu) : (i == 1) ? (xv[t].x >> 16)
                                            : (i == 2) ? (xv[t].y & 0xFFFFu) : (xv[t].y >> 16);
                        gw[t][i] = (uint32_t)(4 * lane + i) | ((uint32_t)bt[t][i] << 8) | ((uint32_t)bu[i] << 12) | (xs << 16);
                    }
                }
            }
        }
        bool have[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) have[i] = gin[i] && (gpos[i] >> 6) == seg_half;
        // ---- rank of every kept position among the kept positions of this half.  inc[i] = kept positions of the form
        //      4 l' + i (bit l'), the same on every lane: position p = 4 q + r is preceded by those with l' < q, plus
        //      l' = q for i < r.
        uint32_t inc[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            bool k;  // is position 4 lane + i kept?
            if (direct) {
                k = have[i];
            } else {
                const int p = 4 * lane + i;
                const int s_ = (int)(__brev((uint32_t)p) >> 25);
                k = s_ >= a && s_ < b_ && p < gnz && (p >> 6) == seg_half;
            }
            inc[i] = __ballot_sync(0xffffffffu, k);
        }
        const int n = __popc(inc[0]) + __popc(inc[1]) + __popc(inc[2]) + __popc(inc[3]);
        const uint32_t gbase = (uint32_t)g * GQ_G * rowbytes;
        float Xp[T], Pp[T];
#pragma unroll
        for (int t = 0; t < T; ++t) Xp[t] = Pp[t] = 0.f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (have[i]) {
                const int q = gpos[i] >> 2, r = gpos[i] & 3;
                const uint32_t below = (1u << q) - 1u, upto = below | (1u << q);
                const int rank = __popc(inc[0] & (r > 0 ? upto : below)) + __popc(inc[1] & (r > 1 ? upto : below)) +
                                 __popc(inc[2] & (r > 2 ? upto : below)) + __popc(inc[3] & below);
                const int idx = (app + rank) & (LN - 1);
                list[idx] = make_uint2(gw[0][i], gbase + (gw[0][i] & 0x7Fu) * rowbytes);
#pragma unroll
                for (int t = 1; t < T; ++t) tok[(t - 1) * LN + idx] = gw[t][i];
            }
        }
        __syncwarp();
        // ---- this piece's share of the segment's X and Phi, summed in list order by every form (same bits)
#pragma unroll 1
        for (int i = lane; i < n; i += 32) {
            const int idx = (app + i) & (LN - 1);
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const uint32_t ww = (t == 0) ? list[idx].x : tok[(t - 1) * LN + idx];
                const int b = (ww >> 8) & 15;
                if (b > 0) {
                    const float xf = __half2float(__ushort_as_half((uint16_t)(ww >> 16)));
                    Xp[t] += xf;
                    // phi_b = 2^(7-b), phi_8 = 0; 2-bit segments: in the left-aligned byte, 0 at b = b_max
                    const float ph = SEG2 ? ((b == bmax) ? 0.f : (float)(0x80 >> b) / (float)(1 << (8 - bmax)))
                                          : (float)(0x80 >> b);
                    Pp[t] = fmaf(xf, ph, Pp[t]);
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
        seg_rows = seg_rows || n > 0;
        if (seg_half == 0) {
            seg_half = 1;
        } else {  // the group is done for this warp: scale/zero chunks, X and Phi (if it had rows at all), next group
            if (seg_rows) {
                const int slot = segj & 15;
                if (lane < 4)
                    list[(app + lane) & (LN - 1)] =
                        make_uint2(ENTRY_SZ | (uint32_t)lane | ((uint32_t)g << 8) | ((uint32_t)slot << 16), 0u);
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
                app += 4;
                ++segj;
            }
#pragma unroll
            for (int t = 0; t < T; ++t) Xrun[t] = Prun[t] = 0.f;
            seg_rows = false;
            seg_half = 0;
            seg_s = (g + 1) * GQ_G;
        }
        __syncwarp();
    };

    // issues list entry iv into ring slot iv mod RING (one cp.async group, empty past the end of the list; or bulk
    // copies completing on the slot's mbarrier)
    auto issue_one = [&]() {
        if (iv < app) {
            const uint2 e = list[iv & (LN - 1)];
            const uint32_t so = (uint32_t)(iv & (RING - 1)) * SLOT_BYTES;
            if (BULK) {
                const uint32_t mb = mbar_s + (uint32_t)(iv & (RING - 1)) * 8;
                if (!(e.x & ENTRY_SZ)) {
                    const uint32_t b = (e.x >> 12) & 15;
                    if (lane == 0) mbar_arrive_expect_tx(mb, b * segbytes);
                    if ((uint32_t)lane < b && segbytes) bulk_g2s(ring_s + so + lane * 128, bulk_src + e.y, segbytes, mb);
                } else {
                    const uint32_t nact = (uint32_t)min(32, max(0, words - tile * 32));
                    if (lane == 0) mbar_arrive_expect_tx(mb, nact * 32);
                    if (active) {
                        const size_t gn = (size_t)((e.x >> 8) & 0xFFu) * N + (size_t)word * 32 + 8 * (e.x & 3u);
                        bulk_g2s(ring_s + so + lane * 16, scales + gn, 16, mb);
                        bulk_g2s(ring_s + so + 512 + lane * 16, zeros + gn, 16, mb);
                    }
                }
                ++iv;
                return;
            }
            if (!(e.x & ENTRY_SZ)) {
                const int b = (e.x >> 12) & 15;
                const uint8_t* src = lane_src + e.y;
                const uint32_t dst = lane_dst + so;
                if (SEG2) {
                    if (2 * pjx < b) cp_async16(dst, src);
                    if (2 * pjx + 4 < b) cp_async16(dst + 512, src + hi_off);
                } else if (A16) {
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
        if (!BULK) cp_async_commit();
    };
    // entry v has landed in its slot
    auto wait_entry = [&](int v) {
        if (BULK) {
            mbar_wait(mbar_s + (uint32_t)(v & (RING - 1)) * 8, (uint32_t)(v / RING) & 1u);
        } else {
            cp_async_wait<RING - 3>();
        }
        __syncwarp();
    };

    GQ_STAMP();
    while (app - iv < RING && more_rows()) append_piece();
    GQ_STAMP();
#pragma unroll 1
    for (int i = 0; i < RING - 2; ++i) issue_one();
    GQ_STAMP();
    // the warp's accumulator tile starts at zero (cleared while the first rows are on their way)
    {
        float4* yz = reinterpret_cast<float4*>(yacc);
#pragma unroll 1
        for (int i = lane; i < T * YSLOT / 4; i += 32) yz[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }

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

    // one row of the 2-bit-segment store: NS segments of 2 x 16 columns -> 32 left-aligned codes -> 32 FMAs
    auto consume2 = [&](auto ns_tag, uint32_t m, int v) {
        constexpr int NS = decltype(ns_tag)::value;
        const uint2* slot = reinterpret_cast<const uint2*>(ring + (uint32_t)(v & (RING - 1)) * SLOT_BYTES) + lane;
        uint32_t a0[4] = {0u, 0u, 0u, 0u}, a1[4] = {0u, 0u, 0u, 0u}, X0[4], X1[4];
#pragma unroll
        for (int sg = 0; sg < NS; ++sg) {
            const uint2 w = slot[sg * 32];
            a0[sg] = w.x;
            a1[sg] = w.y;
        }
        gather_seg2<NS>(a0, X0);
        gather_seg2<NS>(a1, X1);
        const uint16_t xh = (uint16_t)(m >> 16);
#pragma unroll
        for (int r = 0; r < 8; ++r) {  // column r of the half = byte r >> 2 of X[r & 3], column 8 + r = byte (r >> 2) + 2
            const uint32_t h01 = (r < 4) ? __byte_perm(X0[r & 3], 0u, 0x4240) : __byte_perm(X0[r & 3], 0u, 0x4341);
            const uint32_t h23 = (r < 4) ? __byte_perm(X1[r & 3], 0u, 0x4240) : __byte_perm(X1[r & 3], 0u, 0x4341);
            fhfma_lo(acc[0][4 * r + 0], h01, xh);
            fhfma_hi(acc[0][4 * r + 1], h01, xh);
            fhfma_lo(acc[0][4 * r + 2], h23, xh);
            fhfma_hi(acc[0][4 * r + 3], h23, xh);
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
                    *dst = fmaf(zf[r], X[t], fmaf(sf[r], fmaf(acc[t][4 * r + L], code_scale, Phi[t]), *dst));
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
                    wait_entry(cv);
                    issue_one();
                    if constexpr (SEG2) consume2(integral_constant<int, (B >= 2 ? B / 2 : 1)>{}, e, cv);
                    else consume(b_tag, e, cv);
                    ++cv;
                    e = list[cv & (LN - 1)].x;
                } while (cv < stop && !(e & ENTRY_SZ) &&
                         (B != 0 ? (int)((e >> 12) & 15) == B
                                 : ((e >> 12) & 15) != 8 && ((e >> 12) & 15) != 4 && ((e >> 12) & 15) != 2));
            };
            if (e & ENTRY_SZ) {
                wait_entry(cv);
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
                else if constexpr (SEG2) run(integral_constant<int, 6>{});  // (widths are 2, 4, 6, 8 there)
                else run(integral_constant<int, 0>{});
            }
        }
    }
    if (!BULK) cp_async_wait<0>();
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
        GQ_STAMP();
        __syncthreads();  // the CTA's partial is complete ...
        GQ_STAMP();
        if (tid == 0) {
            // ... and released device-wide with the ticket: ONE acq_rel atomic (release: the CTA's partial, ordered
            // before it by the barrier; acquire: the other CTAs' partials for the last one) instead of a sequentially
            // consistent fence on either side of a relaxed atomic
            int old;
            asm volatile("atom.add.acq_rel.gpu.global.s32 %0, [%1], 1;" : "=r"(old) : "l"(tickets + tile) : "memory");
            s_last = (old == Sx - 1);
        }
        GQ_STAMP();
        __syncthreads();
        GQ_STAMP();
        if (s_last) {
            // float2 columns spread over all the CTA's threads, 32 partials per column in flight, added in the fixed
            // order s = 0..Sx-1
            constexpr int BATCH = 32;
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
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(gt2));
    GQ_STAMP();
    if (tid == 0 && (s_last == 1 || blockIdx.y == 0) && blockIdx.x == 0) {
        if (false) {
            printf("select:");
            for (int i = 1; i < g_sel_n; ++i) printf(" %lld", g_sel_stamp[i] - g_sel_stamp[0]);
            printf("\n");
        }
        printf("blk %3d last %d entries %3d:", blockIdx.y, s_last, cv);
        for (int i = 1; i < nst; ++i) printf(" %6lld", stamp[i] - stamp[0]);
        printf("\n");
    }
#endif
}

// y[t][n] = sum_{s=0}^{S-1} part[s][t][n], sequentially in s: the same order as the fused second pass, so the
// two-launch form returns the same bits.
__global__ void __launch_bounds__(256)
vmm_reduce_kernel(const float* __restrict__ part, int S, int T, int N, float* __restrict__ y);

template <int T, int VW, bool A16, int MODE, bool BULK = false, bool SEG2 = false>
static int launch_impl(const VmmArgs& a, const VmmPlan& pl) {
    using C = Cfg<T, VW>;
    const size_t smem = (size_t)C::BASE_BYTES + (MODE == MODE_SCHED ? 0 : (size_t)T * (a.K / GQ_G) * 16);
    // the attribute belongs to the device: set it on every launch (cheap, legal during stream capture)
    if (cudaFuncSetAttribute(vmm_kernel<T, VW, A16, MODE, BULK, SEG2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
        cudaSuccess)
        return GRINQH_ERR_CUDA;
    dim3 grid(pl.col_tiles, pl.Sx);
    const cudaError_t e =
        launch_pdl(vmm_kernel<T, VW, A16, MODE, BULK, SEG2>, grid, dim3(C::NT), smem, a.st, a.K, a.N, pl.Sx, a.fused, a.bmax,
                   a.planes,
                   (const __half*)a.scales, (const __half*)a.zeros, a.gsched, a.gcnt_ge, a.xraw, a.cp,
                   (float*)((char*)a.workspace + TICKET_BYTES), (int*)a.workspace, a.y);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

int launch_vmm_multi(const VmmArgs& a, const VmmPlan& pl);  // vmm_multi.cu: T = 2..4

}  // namespace gq
