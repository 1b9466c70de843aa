// vmm_items.cu — the item kernel behind grinqh_vmm / grinqh_vmm_rank / grinqh_vmm_thresholds (1-bit plane store).
// PAPER.md:85 (reconstruction), :51 (only the needed planes are fetched), :61-65 / :271 (assignment), :440-444
// (prior-art kernel).
//
// Work item = (column tile of 1024 columns, group g of 128 rows, sub-chunk q of Q): the positions
// q, q+Q, q+2Q, ... of the group's (width desc, index asc) list, so every item of a group sees the same
// width mix.  A WARP owns `ipw` consecutive items of one column tile and is fully independent of the other
// warps until the CTA epilogue (no __syncthreads in the row loop):
//
//   prologue lanes stage the item's schedule entries (row | widths | x) and row byte offsets in shared memory; the
//            warp reduces the item's scalars X = sum_{b_k>0} x_k, Phi = sum x_k phi_{b_k}.  The entries come from
//            gsched (grinqh_assign ran before) or are made on the spot from x and the launch's cuts (threshold / rank
//            form: widths4 + partition128 in two ring slots).
//   stream   a warp-private ring of RING 1-KB slots in shared memory, filled by cp.async (LDGSTS.128):
//            one instruction fetches 4 planes x 128 B of a row (lanes 8j..8j+7 copy plane j), so a 4-bit
//            row costs one and an 8-bit row two; RING-2 rows are in flight while a row is consumed; the
//            group's scales and zeros follow the rows through the same ring.
//   expand   rows are walked in width-class runs (compile-time b = 8 / 4 / 2, generic otherwise); lane l reads
//            its plane words (columns 32l..32l+31 of the tile), rebuilds the 32 truncated codes in byte lanes
//            (gather.cuh, SIMD 8x8 bit transpose) and does 32 mixed-precision FMAs
//            acc[c] += half(code_c) * half(x_k)   (exact product, fp32 accumulate).
//   item end y_n += s_gn * (A_n + Phi) + z_gn * X  — s and z are applied once per (item, column) and
//            summed into the warp's shared-memory accumulator.
// CTA epilogue: the warps' accumulators are added in fixed order and written as one split-K partial
// part[sx][t][n]; the last CTA of the tile (ticket) sums the Sx partials in fixed order.  Deterministic.
//
// Rank form inside the launch (grinqh_vmm_rank): before the items, every CTA selects the cut keys of x itself
// (select.cuh: one shared-memory atomic per key into a 15-bit histogram, block scan, the owning warp scans the cut's
// bins) and, when a cut splits a run of equal keys, the ordered tie offsets of every group; the item prologue then
// makes the widths with widths4.  Why this kernel and not the stream kernel for the plane store: at the shapes of the
// configs a warp of the stream kernel gets 6-45 rows and pays ~1500-2000 instructions of its own (range, lists,
// chunks, run transitions) for them; here half as many warps run items of 14-22 rows with ~600 (profiles/r02_kernels.md).
#include <cstdlib>
#include <type_traits>

#include "common.cuh"
#include "gather.cuh"
#include "select.cuh"
#include "vmm_args.cuh"

namespace gq {
namespace items {

constexpr int VW = 8;  // warps per CTA (16 in the wide variant: half as many split-K partials, 1 CTA per SM)
constexpr int TILE_COLS = 1024;
constexpr int SLOT_BYTES = 1024;   // 8 planes x 128 B
constexpr int YSLOT = 32 * 33;     // one warp's 1024 sums, padded: column 32*l + c lives at c*33 + l

template <int T>
struct Cfg {
    static constexpr int RING = (T == 1) ? 8 : 4;
    // per-warp shared memory: ring | yacc[T] | item[128] {entry, row byte offset} | tok[T-1][128] entries
    static constexpr int RING_OFF = 0;
    static constexpr int YACC_OFF = RING * SLOT_BYTES;
    static constexpr int ITEM_OFF = YACC_OFF + T * YSLOT * 4;
    static constexpr int TOK_OFF = ITEM_OFF + 1024;
    static constexpr int WARP_BYTES = TOK_OFF + (T - 1) * 512;
    static constexpr int SMEM = VW * WARP_BYTES;  // x2 for the 16-warp variant
    static_assert(WARP_BYTES % 16 == 0, "warp regions stay 16-byte aligned");
};

struct VmmPlan {
    int col_tiles;  // ceil(N / 1024)
    int Q;          // sub-chunks per group
    int Sx;         // CTAs (= split-K partials) per column tile
    int ipw;        // items per warp; warp slot ws owns items [ws*ipw, min(I, (ws+1)*ipw)), I = (K/128)*Q
    int vw;         // warps per CTA: 8 (2 CTAs per SM) or 16 (1 CTA per SM, half the partials)
};

// Static plan from the shape only (the workspace size depends on it).  Cost model in "rows": a warp does
// ipw * (rows per item + item overhead), and the launch ends with the last CTA's second pass over Sx partials;
// pick (warps per CTA, Q in 1..8) that minimises the sum under the residency limit (16 warps per SM either way).
//
// ONE plan per shape for every form of the launch (schedule, threshold, rank, two-launch): the forms promise the same
// bits, and the bits depend on the item partition.  So the plan obeys the rank form's limits — the select's histogram
// and keys (128 KB) alias the warp regions: one CTA per SM whatever the width, and the 16-warp variant only where its
// regions plus the tie table fit.
constexpr int SMEM_LIMIT = 232448 - 1024;  // 227 KB per CTA, static shared memory included (cuts, scratch: < 1 KB)
static inline int warp_bytes(int T) {
    return T == 1 ? Cfg<1>::WARP_BYTES : T == 2 ? Cfg<2>::WARP_BYTES : T == 3 ? Cfg<3>::WARP_BYTES : Cfg<4>::WARP_BYTES;
}
static inline int smem_bytes(int T, int vw, int K, bool rank) {
    const int base = warp_bytes(T) * vw;
    return rank ? (base > 2 * 65536 ? base : 2 * 65536) + T * (K / GQ_G) * 16 : base;
}

static inline VmmPlan vmm_plan(int T, int K, int N) {
    VmmPlan best{};
    const int CT = (N + TILE_COLS - 1) / TILE_COLS;
    const int groups = K / GQ_G;
    double best_cost = 1e30;
    for (int vw = 8; vw <= ((T <= 2) ? 16 : 8); vw *= 2) {
        if (vw == 16 && smem_bytes(T, vw, K, true) > SMEM_LIMIT) continue;
        const int resident = num_sms();
        const int sx_max = resident / CT > 0 ? resident / CT : 1;
        for (int Q = 1; Q <= 16; ++Q) {
            const int I = groups * Q;
            int Sx = (I + vw - 1) / vw;
            if (Sx > sx_max) Sx = sx_max;
            const int ipw = (I + vw * Sx - 1) / (vw * Sx);
            Sx = (I + vw * ipw - 1) / (vw * ipw);
            // (item overhead 12 rows: measured on this kernel — a sweep of the constant over the configs' shapes, 6 -> 12:
            // layer step 83.9 -> 82.5 us, the 70B shapes up to 13 % faster in the rank form; profiles/r02_kernels.md)
            const double cost = ipw * (112.0 / Q + 12.0) + 4.0 + 0.12 * Sx;  // + second pass, in row units (~0.45 us)
            if (cost < best_cost - 1e-9) {
                best_cost = cost;
                best = VmmPlan{CT, Q, Sx, ipw, vw};
            }
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

// A16: every plane row is 16-byte aligned (N % 128 == 0) -> LDGSTS.128, 4 planes per instruction;
// otherwise each lane copies its own word of every plane with 4-byte cp.async.
//
// gsched[t][g*128 + p] (written by grinqh_assign) is position p of group g's list for token t:
//   bits 0..7 local row r | 8..11 b_t (token's width) | 12..15 b (union width = planes fetched) | 16..31 x_t[r] fp16
//
// fused: the last CTA of a column tile to finish (ticket counter in the workspace, reset to 0 by that CTA) sums the
// tile's Sx partials in the fixed order s = 0..Sx-1 and writes y: still deterministic, one launch instead of two.
template <int T, int VWT, bool A16>
__global__ void __launch_bounds__(VWT * 32, 1)
vmm_items_kernel(int K, int N, int Q, uint32_t rq, int ipw, int Sx, int fused, int mode, const uint32_t* __restrict__ planes,
                const __half* __restrict__ scales, const __half* __restrict__ zeros,
                const uint32_t* __restrict__ gsched, const uint8_t* __restrict__ gcnt_ge,
                float* __restrict__ part, int* __restrict__ tickets, float* __restrict__ y,
                const uint16_t* __restrict__ xraw, CutParams cp) {
    using C = Cfg<T>;
    constexpr int RING = C::RING;
    extern __shared__ __align__(16) uint8_t smem[];
    __shared__ __align__(16) TokenCuts s_tc[T];
    __shared__ SelectScratch s_sel;
    __shared__ int s_cuts[16];  // Cd[8] | mult[8], read with run-time indices (as kernel parameters every thread would copy
                                // them to local memory at kernel entry, schedule form included)
    __shared__ int s_last;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x, sx = blockIdx.y;
    const int words = N >> 5;
    const int word = tile * 32 + lane;
    const bool active = word < words;
    const uint32_t rowbytes = (uint32_t)words * 4u;
    const size_t pbytes = (size_t)K * rowbytes;  // one plane
    const int I = (K / GQ_G) * Q;

    uint8_t* wbase = smem + warp * C::WARP_BYTES;
    const uint8_t* ring = wbase + C::RING_OFF;
    float* yacc = reinterpret_cast<float*>(wbase + C::YACC_OFF);
    uint2* s_item = reinterpret_cast<uint2*>(wbase + C::ITEM_OFF);
    uint32_t* s_tok = reinterpret_cast<uint32_t*>(wbase + C::TOK_OFF);
    const uint32_t ring_s = (uint32_t)__cvta_generic_to_shared(wbase + C::RING_OFF);

    // per-lane copy geometry: lane copies chunk `seg` (16 B) of plane pj (and pj + 4); pjx = 99 disables the lane
    const int pj = lane >> 3, seg = lane & 7;
    const bool chunk_ok = A16 ? (tile * 32 + seg * 4 < words) : active;
    const int pjx = chunk_ok ? (A16 ? pj : 0) : 99;
    const uint8_t* lane_src = reinterpret_cast<const uint8_t*>(planes) +
                              (A16 ? (size_t)pj * pbytes + (size_t)(tile * 32 + seg * 4) * 4 : (size_t)word * 4);
    const uint32_t lane_dst = A16 ? ring_s + pj * 128 + seg * 16 : ring_s + lane * 4;

    const int groups = K / GQ_G, nd = cp.nd;
    uint16_t* s_tie = reinterpret_cast<uint16_t*>(smem + max(VWT * C::WARP_BYTES, 2 * 65536));  // [T][groups][8]

    pdl_launch_dependents();
    if (xraw == nullptr) {
        pdl_wait();  // nothing global (schedule, partials, tickets) is touched before the previous kernel has finished
    } else {
        // ---- the assignment is made in this launch: the cuts of every token (rank form: selected here; threshold
        //      form: given) and, where a cut splits a run of equal keys, the ordered tie offsets of every group.  The
        //      histogram and the token's keys alias the warp regions, which nobody uses before the barrier below.
        constexpr int NT = VWT * 32;
        uint32_t* hist = reinterpret_cast<uint32_t*>(smem);
        uint16_t* skeys = reinterpret_cast<uint16_t*>(smem + 65536);
        if (tid == 0) {
#pragma unroll
            for (int d = 0; d < 8; ++d) s_cuts[d] = cp.Cd[d];
        } else if (tid == 32) {
#pragma unroll
            for (int d = 0; d < 8; ++d) s_cuts[8 + d] = cp.mult[d];
        } else if (tid == 64 && mode != MODE_RANK) {
#pragma unroll
            for (int t = 0; t < T; ++t) {
#pragma unroll
                for (int d = 0; d < 8; ++d) {
                    s_tc[t].thr[d] = cp.thr[d];
                    s_tc[t].take[d] = 0;
                    s_tc[t].hh[d] = 0;
                }
                s_tc[t].split = 0;
                s_tc[t].nd = nd;
            }
        }
        if (mode == MODE_RANK) {  // cleared while the previous kernel is still running
            uint4* z = reinterpret_cast<uint4*>(hist);
            for (int i = tid; i < 4096; i += NT) z[i] = make_uint4(0, 0, 0, 0);
        }
        __syncthreads();
        pdl_wait();
#pragma unroll 1
        for (int t = 0; t < T; ++t) {
            if (mode == MODE_RANK)
                rank_select<NT>(xraw + (size_t)t * K, skeys, K, nd, s_cuts, hist, t + 1 < T, &s_sel, &s_tc[t]);
            const uint32_t split = s_tc[t].split;
            if (split) {
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
                for (int d = warp; d < nd; d += VWT) {  // (up to 8 rounds of 32 groups: independent scans, then the carries)
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
        __syncthreads();  // from here on the warp regions belong to their warps
    }

    const int ws = sx * VWT + warp;
    const int it0 = ws * ipw;
    const int it1 = min(I, it0 + ipw);
    bool first = true;

    for (int it = it0; it < it1; ++it) {
        const int g = (int)(((uint32_t)it * rq) >> 16), q = it - g * Q;  // it / Q (rq = ceil(65536 / Q), it < 8192)
        __syncwarp();
        // ---- item prologue: lane l stages item rows l, l+32, ... and the warp reduces X, Phi
        auto rows_ge = [&](uint32_t c) -> int {  // rows of this item among the first c list positions
            return ((int)c > q) ? (int)(((c - q + Q - 1) * rq) >> 16) : 0;
        };
        uint4 cv;
        uint32_t ev[T][4];
        if (xraw == nullptr) {
            // the schedule entries are fetched speculatively (position < 128), in flight together with the counts
            cv = *reinterpret_cast<const uint4*>(gcnt_ge + g * GQ_GCNT);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const int pos = q + (lane + 32 * jj) * Q;
#pragma unroll
                for (int t = 0; t < T; ++t) ev[t][jj] = (pos < GQ_G) ? gsched[(size_t)t * K + g * GQ_G + pos] : 0u;
            }
        } else {
            // grinqh_vmm_thresholds / grinqh_vmm_rank: the warp makes the group's schedule itself from x and the launch's
            // cuts — widths4 (ties by index), union over tokens, partition128 — in the two ring slots
            // the item prologue does not fill; no assignment kernel, no schedule in global memory.
            uint32_t* s_list = reinterpret_cast<uint32_t*>(wbase + C::RING_OFF + (RING - 2) * SLOT_BYTES);
            uint2 xv[T];
#pragma unroll
            for (int t = 0; t < T; ++t) xv[t] = *reinterpret_cast<const uint2*>(xraw + (size_t)t * K + g * GQ_G + 4 * lane);
            int bt[T][4], bu[4] = {0, 0, 0, 0}, pos[4], ge[10];
#pragma unroll
            for (int t = 0; t < T; ++t) {
                int m[4];
                keys4(xv[t], m);
                widths4(m, &s_tc[t], s_cuts + 8, nd, s_tie + ((size_t)t * groups + g) * 8, lane, bt[t]);
#pragma unroll
                for (int i = 0; i < 4; ++i) bu[i] = max(bu[i], bt[t][i]);
            }
            partition128(bu, lane, pos, ge);
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const uint32_t xs[4] = {xv[t].x & 0xFFFFu, xv[t].x >> 16, xv[t].y & 0xFFFFu, xv[t].y >> 16};
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    s_list[t * GQ_G + pos[i]] = (uint32_t)(4 * lane + i) | ((uint32_t)bt[t][i] << 8) |
                                                ((uint32_t)bu[i] << 12) | (xs[i] << 16);
            }
            cv.x = (uint32_t)ge[0] | ((uint32_t)ge[1] << 8) | ((uint32_t)ge[2] << 16) | ((uint32_t)ge[3] << 24);
            cv.y = (uint32_t)ge[4] | ((uint32_t)ge[5] << 8) | ((uint32_t)ge[6] << 16) | ((uint32_t)ge[7] << 24);
            cv.z = (uint32_t)ge[8];
            cv.w = 0;
            __syncwarp();
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const int pos_i = q + (lane + 32 * jj) * Q;
#pragma unroll
                for (int t = 0; t < T; ++t) ev[t][jj] = (pos_i < GQ_G) ? s_list[t * GQ_G + pos_i] : 0u;
            }
            __syncwarp();  // the list is consumed before the ring slots are handed to the copies
        }
        const int n_rows = rows_ge((cv.x >> 8) & 0xFF);
        float X[T], Phi[T];
#pragma unroll
        for (int t = 0; t < T; ++t) X[t] = Phi[t] = 0.f;
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            const int i = lane + 32 * jj;
            if (i < n_rows) {
                const uint32_t e0 = ev[0][jj];
                s_item[i] = make_uint2(e0, (e0 & 0xFFu) * rowbytes);
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const uint32_t e = ev[t][jj];
                    if (t > 0) s_tok[(t - 1) * GQ_G + i] = e;
                    const int bt = (e >> 8) & 15;
                    if (bt > 0) {
                        const float xf = __half2float(__ushort_as_half((uint16_t)(e >> 16)));
                        X[t] += xf;
                        Phi[t] = fmaf(xf, (float)(0x80 >> bt), Phi[t]);  // phi_b = 2^(7-b), phi_8 = 0
                    }
                }
            }
        }
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                X[t] += __shfl_xor_sync(0xffffffffu, X[t], d);
                Phi[t] += __shfl_xor_sync(0xffffffffu, Phi[t], d);
            }
        __syncwarp();
        const uint8_t* item_src = lane_src + (size_t)g * GQ_G * rowbytes;

        float acc[T][32];
#pragma unroll
        for (int t = 0; t < T; ++t)
#pragma unroll
            for (int c = 0; c < 32; ++c) acc[t][c] = 0.f;

        // copy of item row ii into ring slot at byte offset `so`; HI = the row may have more than 4 planes
        auto issue = [&](int ii, uint32_t so, auto hi_tag) {
            constexpr bool HI = decltype(hi_tag)::value;
            const uint2 m = s_item[ii];
            const int b = (m.x >> 12) & 15;
            const uint8_t* src = item_src + m.y;
            const uint32_t dst = lane_dst + so;
            if (A16) {
                if (pjx < b) cp_async16(dst, src);
                if (HI && pjx + 4 < b) cp_async16(dst + 512, src + 4 * pbytes);
            } else {
#pragma unroll
                for (int j = 0; j < (HI ? 8 : 4); ++j)
                    if (pjx + j < b) cp_async4(dst + j * 128, src + j * pbytes);
            }
        };
        using HiT = std::integral_constant<bool, true>;
        using LoT = std::integral_constant<bool, false>;

        // The group's scales and zeros (64 B + 64 B per lane) ride the ring too, as "virtual rows" n_rows .. n_rows+3
        // behind the item's rows: chunk c = the lane's 16-byte piece c of both.  Virtual row v always lives in slot
        // v mod RING, and every issue is one cp.async group, so group index == virtual row index.
        const size_t gn = (size_t)g * N + (size_t)word * 32;
        int next_v = 0;  // next virtual row to issue
        auto issue_next = [&](auto hi_tag) {
            const uint32_t slot_off = (uint32_t)(next_v & (RING - 1)) * SLOT_BYTES;
            if (next_v < n_rows) {
                issue(next_v, slot_off, hi_tag);
            } else if (next_v < n_rows + 4 && active) {
                const int c = next_v - n_rows;
                cp_async16(ring_s + slot_off + lane * 16, scales + gn + 8 * c);
                cp_async16(ring_s + slot_off + 512 + lane * 16, zeros + gn + 8 * c);
            }
            cp_async_commit();
            ++next_v;
        };
        // lean form when the virtual row is known to be a real row (no scale/zero chunk, no bounds): the common case
        auto issue_row = [&](auto hi_tag) {
            issue(next_v, (uint32_t)(next_v & (RING - 1)) * SLOT_BYTES, hi_tag);
            cp_async_commit();
            ++next_v;
        };
        const int n_lean = max(0, n_rows - (RING - 2));  // rows i < n_lean prefetch a real row (i + RING - 2 < n_rows)
        if (n_lean > 0) {
#pragma unroll
            for (int i = 0; i < RING - 2; ++i) issue_row(HiT{});
        } else {
#pragma unroll
            for (int i = 0; i < RING - 2; ++i) issue_next(HiT{});
        }

        // one row: plane words of its ring slot -> 32 truncated codes -> 32 FMAs per token
        auto consume = [&](auto b_tag, int i) {
            constexpr int B = decltype(b_tag)::value;
            const uint32_t m = s_item[i].x;
            const uint32_t* slot = reinterpret_cast<const uint32_t*>(ring + (uint32_t)(i & (RING - 1)) * SLOT_BYTES) + lane;
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
                const int b = (m >> 12) & 15;
#pragma unroll
                for (int j = 0; j < 8; ++j) Wd[j] = (j < b) ? slot[j * 32] : 0u;
                gather<8>(Wd, V);
            }
            if (T == 1) {
                accumulate_row(V, (uint16_t)(m >> 16), acc[0]);
            } else if (T == 2) {
                const int b = (m >> 12) & 15;
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const uint32_t e = (t == 0) ? m : s_tok[(t - 1) * GQ_G + i];
                    const int bt = (e >> 8) & 15;  // this token's own width (<= b, the union)
                    if (bt == 0) continue;         // warp-uniform
                    if (bt == b) {
                        accumulate_row(V, (uint16_t)(e >> 16), acc[t]);
                    } else {
                        const uint32_t mask = 0x01010101u * ((0xFF00u >> bt) & 0xFFu);
                        uint32_t Vm[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) Vm[j] = V[j] & mask;
                        accumulate_row(Vm, (uint16_t)(e >> 16), acc[t]);
                    }
                }
            } else {
                // 3 or 4 tokens: the bytes are widened to fp16 lanes once per row; a token narrower than the union
                // masks the 16-bit lanes instead of the bytes (no further byte permutes): -12 % at T = 4 (at T = 2 the
                // 16 extra registers spill, so it keeps the byte form)
                const int b = (m >> 12) & 15;
                uint32_t H[16];
#pragma unroll
                for (int r = 0; r < 8; ++r) {
                    H[2 * r] = __byte_perm(V[r], 0u, 0x4140);
                    H[2 * r + 1] = __byte_perm(V[r], 0u, 0x4342);
                }
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    const uint32_t e = (t == 0) ? m : s_tok[(t - 1) * GQ_G + i];
                    const int bt = (e >> 8) & 15;
                    if (bt == 0) continue;
                    const uint16_t xh = (uint16_t)(e >> 16);
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
        };

        // rows [i0, i1) of the item, all of width B (B = 0: any width, read from the schedule)
        auto run = [&](auto b_tag, auto hi_tag, int i0, int i1) {
            int i = i0;
            for (const int ie = min(i1, n_lean); i < ie; ++i) {  // steady state: one row in, one row out
                cp_async_wait<RING - 3>();
                __syncwarp();
                issue_row(hi_tag);
                consume(b_tag, i);
            }
            for (; i < i1; ++i) {  // the item's last RING-2 rows: scale/zero chunks (or nothing) follow the rows
                cp_async_wait<RING - 3>();
                __syncwarp();
                issue_next(hi_tag);
                consume(b_tag, i);
            }
        };
        {
            using std::integral_constant;
            const int r8 = rows_ge(cv.z & 0xFF), r5 = rows_ge((cv.y >> 8) & 0xFF), r4 = rows_ge(cv.y & 0xFF);
            const int r3 = rows_ge(cv.x >> 24), r2 = rows_ge((cv.x >> 16) & 0xFF);
            run(integral_constant<int, 8>{}, HiT{}, 0, r8);
            run(integral_constant<int, 0>{}, HiT{}, r8, r5);
            run(integral_constant<int, 4>{}, LoT{}, r5, r4);
            run(integral_constant<int, 0>{}, LoT{}, r4, r3);
            run(integral_constant<int, 2>{}, LoT{}, r3, r2);
            run(integral_constant<int, 0>{}, LoT{}, r2, n_rows);
        }
        if (n_rows > 0 && next_v < n_rows + 4) {  // scale/zero chunks that found no iteration (short items)
            __syncwarp();
            while (next_v < n_rows + 4) issue_next(LoT{});
        }
        cp_async_wait<0>();

        // ---- item end: s and z once per (item, column), into the warp's accumulator
        if (active) {
#pragma unroll
            for (int L = 0; L < 4; ++L) {
                float sf[8], zf[8];
                if (n_rows > 0) {
                    const uint8_t* sz = ring + (uint32_t)((n_rows + L) & (RING - 1)) * SLOT_BYTES + lane * 16;
                    const uint4 sv = *reinterpret_cast<const uint4*>(sz);
                    const uint4 zv = *reinterpret_cast<const uint4*>(sz + 512);
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
                        if (n_rows > 0) v = fmaf(zf[r], X[t], fmaf(sf[r], fmaf(acc[t][4 * r + L], CODE_SCALE, Phi[t]), v));
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

    // ---- CTA epilogue: fixed-order sum over the 8 warps -> one split-K partial (or y itself when Sx == 1)
    float* out = (fused && Sx == 1) ? y : part + (size_t)sx * T * N;
#pragma unroll
    for (int t = 0; t < T; ++t)
#pragma unroll
        for (int i = 0; i < TILE_COLS / (VWT * 32); ++i) {
            const int c = tid + VWT * 32 * i;  // column inside the tile
            const int n = tile * TILE_COLS + c;
            if (n < N) {
                const int idx = (c & 31) * 33 + (c >> 5);
                float A = 0.f;
#pragma unroll
                for (int w = 0; w < VWT; ++w)
                    A += *reinterpret_cast<const float*>(smem + w * C::WARP_BYTES + C::YACC_OFF + (t * YSLOT + idx) * 4);
                out[(size_t)t * N + n] = A;
            }
        }
    if (fused && Sx > 1) {
        __syncthreads();  // the CTA's partial is complete ...
        if (tid == 0) {
            // ... and released device-wide with the ticket: one acq_rel atomic (release: the CTA's partial, ordered
            // before it by the barrier; acquire: the other CTAs' partials for the last one)
            int old;
            asm volatile("atom.add.acq_rel.gpu.global.s32 %0, [%1], 1;" : "=r"(old) : "l"(tickets + tile) : "memory");
            s_last = (old == Sx - 1);
        }
        __syncthreads();
        if (s_last) {
            // every thread takes TILE_COLS / threads columns (4 with 8 warps, 2 with 16): the same bytes spread over
            // all the CTA's threads, so one batch holds 16 or 32 partials per column in flight
            constexpr int CPT = TILE_COLS / (VWT * 32);
            constexpr int BATCH = (CPT == 2) ? 32 : 16;
            using Vec = typename std::conditional<CPT == 2, float2, float4>::type;
            const int n = tile * TILE_COLS + CPT * tid;
            if (n < N) {
#pragma unroll
                for (int t = 0; t < T; ++t) {
                    float a[CPT];
#pragma unroll
                    for (int c = 0; c < CPT; ++c) a[c] = 0.f;
                    for (int s0 = 0; s0 < Sx; s0 += BATCH) {  // BATCH loads in flight, added in the fixed order
                        Vec v[BATCH];
#pragma unroll
                        for (int j = 0; j < BATCH; ++j)
                            if (s0 + j < Sx)
                                v[j] = __ldcg(reinterpret_cast<const Vec*>(part + ((size_t)(s0 + j) * T + t) * N + n));
#pragma unroll
                        for (int j = 0; j < BATCH; ++j)
                            if (s0 + j < Sx) {
                                const float* f = reinterpret_cast<const float*>(&v[j]);
#pragma unroll
                                for (int c = 0; c < CPT; ++c) a[c] += f[c];
                            }
                    }
                    Vec o;
                    float* fo = reinterpret_cast<float*>(&o);
#pragma unroll
                    for (int c = 0; c < CPT; ++c) fo[c] = a[c];
                    *reinterpret_cast<Vec*>(y + (size_t)t * N + n) = o;
                }
            }
            if (tid == 0) tickets[tile] = 0;  // ready for the next launch on this workspace
        }
    }
}


template <int T, int VWT, bool A16>
static int launch_items_impl(const VmmArgs& a, const VmmPlan& pl) {
    const bool rank = a.mode == MODE_RANK;
    const int smem = smem_bytes(T, VWT, a.K, rank);
    // (set on every launch: the attribute belongs to the current device's copy of the function, and the call is cheap)
    if (cudaFuncSetAttribute(vmm_items_kernel<T, VWT, A16>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) !=
        cudaSuccess)
        return GRINQH_ERR_CUDA;
    dim3 grid(pl.col_tiles, pl.Sx);
    const uint32_t rq = (65536u + pl.Q - 1) / pl.Q;
    const cudaError_t e = launch_pdl(vmm_items_kernel<T, VWT, A16>, grid, dim3(VWT * 32), (size_t)smem, a.st, a.K, a.N, pl.Q,
                                     rq, pl.ipw, pl.Sx, a.fused, a.mode, a.planes, (const __half*)a.scales,
                                     (const __half*)a.zeros, a.gsched, a.gcnt_ge,
                                     (float*)((char*)a.workspace + TICKET_BYTES), (int*)a.workspace, a.y, a.xraw, a.cp);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

}  // namespace items

int items_sx(int T, int K, int N) { return items::vmm_plan(T, K, N).Sx; }

int launch_vmm_items(const VmmArgs& a) {
    using namespace items;
    const VmmPlan pl = vmm_plan(a.T, a.K, a.N);
#define GQ_LAUNCH_W(TT, WW) \
    return (a.N % 128 == 0) ? launch_items_impl<TT, WW, true>(a, pl) : launch_items_impl<TT, WW, false>(a, pl)
    if (pl.vw == 16) {  // only planned for T <= 2 (registers)
        if (a.T == 1) { GQ_LAUNCH_W(1, 16); }
        GQ_LAUNCH_W(2, 16);
    }
    switch (a.T) {
        case 1: GQ_LAUNCH_W(1, 8);
        case 2: GQ_LAUNCH_W(2, 8);
        case 3: GQ_LAUNCH_W(3, 8);
        default: GQ_LAUNCH_W(4, 8);
    }
#undef GQ_LAUNCH_W
}

}  // namespace gq
