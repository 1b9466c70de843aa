// vmm.cu — grinqh_vmm: split-K vector-matrix multiply over the bit-planar store.
// PAPER.md:85 (reconstruction), :51 (only the needed planes are fetched), :440-444 (prior-art kernel).
//
// Work item = (column tile of 1024 columns, group g of 128 rows, sub-chunk q of Q): the positions
// q, q+Q, q+2Q, ... of the group's (width desc, index asc) list, so every item of a group sees the same
// width mix.  A WARP owns `ipw` consecutive items of one column tile and is fully independent of the other
// warps until the CTA epilogue (no __syncthreads in the row loop):
//
//   prologue lanes stage the item's schedule entries (gsched: row | widths | x) and row byte offsets in shared
//            memory; the warp reduces the item's scalars X = sum_{b_k>0} x_k, Phi = sum x_k phi_{b_k}.
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
// CTA epilogue: the 8 warps' accumulators are added in fixed order and written as one split-K partial
// part[sx][t][n]; the last CTA of the tile (ticket) sums the Sx partials in fixed order.  Deterministic.
#include "common.cuh"
#include <type_traits>

#include "gather.cuh"

namespace gq {

constexpr int VW = 8;  // warps per CTA (16 in the wide variant: half as many split-K partials, 1 CTA per SM)
constexpr int VTHREADS = VW * 32;
constexpr int TILE_COLS = 1024;
constexpr int SLOT_BYTES = 1024;   // 8 planes x 128 B
constexpr int YSLOT = 32 * 33;     // one warp's 1024 sums, padded: column 32*l + c lives at c*33 + l
constexpr int NUM_SMS = 148;
constexpr int ctas_per_sm(int T) { return T <= 2 ? 2 : 1; }  // register / shared-memory budget

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
static inline VmmPlan vmm_plan(int T, int K, int N) {
    VmmPlan best{};
    const int CT = (N + TILE_COLS - 1) / TILE_COLS;
    const int groups = K / GQ_G;
    double best_cost = 1e30;
    for (int vw = 8; vw <= ((T <= 2) ? 16 : 8); vw *= 2) {
        const int resident = NUM_SMS * (vw == 8 ? ctas_per_sm(T) : 1);
        const int sx_max = resident / CT > 0 ? resident / CT : 1;
        for (int Q = 1; Q <= 16; ++Q) {
            const int I = groups * Q;
            int Sx = (I + vw - 1) / vw;
            if (Sx > sx_max) Sx = sx_max;
            const int ipw = (I + vw * Sx - 1) / (vw * Sx);
            Sx = (I + vw * ipw - 1) / (vw * ipw);
            const double cost = ipw * (112.0 / Q + 6.0) + 4.0 + 0.12 * Sx;  // + second pass, in row units (~0.45 us)
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

// threshold assignment done inside the VMM (grinqh_vmm_thresholds): distinct cut keys and how many widths share each
struct ThrParams {
    int thr[8];   // magnitude pattern of distinct cut d (0x8000 = unused: no key reaches it)
    int mult[8];  // widths sharing the cut: b = sum_d mult[d] * [key >= thr[d]]
};

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
// FUSED: the last CTA of a column tile to finish (ticket counter in the workspace, reset to 0 by that CTA) sums the
// tile's Sx partials in the fixed order s = 0..Sx-1 and writes y: still deterministic, one launch instead of two.
template <int T, int VWT, bool A16, bool FUSED>
__global__ void __launch_bounds__(VWT * 32, VWT == 8 ? ctas_per_sm(T) : 1)
vmm_main_kernel(int K, int N, int Q, uint32_t rq, int ipw, int Sx, const uint32_t* __restrict__ planes,
                const __half* __restrict__ scales, const __half* __restrict__ zeros,
                const uint32_t* __restrict__ gsched, const uint8_t* __restrict__ gcnt_ge,
                float* __restrict__ part, int* __restrict__ tickets, float* __restrict__ y,
                const uint16_t* __restrict__ xraw, ThrParams tp) {
    using C = Cfg<T>;
    constexpr int RING = C::RING;
    extern __shared__ __align__(16) uint8_t smem[];

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

    pdl_launch_dependents();
    pdl_wait();  // nothing global (schedule, partials, tickets) is touched before the previous kernel has finished

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
            // grinqh_vmm_thresholds: the warp makes the group's schedule itself from x and the thresholds
            // — widths by comparison, union over tokens, partition128 — in the two ring slots the
            // item prologue does not fill; no assignment kernel, no schedule in global memory.
            uint32_t* s_list = reinterpret_cast<uint32_t*>(wbase + C::RING_OFF + (RING - 2) * SLOT_BYTES);
            uint2 xv[T];
#pragma unroll
            for (int t = 0; t < T; ++t) xv[t] = *reinterpret_cast<const uint2*>(xraw + (size_t)t * K + g * GQ_G + 4 * lane);
            int bt[T][4], bu[4] = {0, 0, 0, 0}, pos[4], ge[10];
#pragma unroll
            for (int t = 0; t < T; ++t) {
                const int m[4] = {(int)(xv[t].x & 0x7FFF), (int)((xv[t].x >> 16) & 0x7FFF), (int)(xv[t].y & 0x7FFF),
                                  (int)((xv[t].y >> 16) & 0x7FFF)};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    int b = 0;
#pragma unroll
                    for (int d = 0; d < 8; ++d) b += (m[i] >= tp.thr[d]) ? tp.mult[d] : 0;
                    bt[t][i] = b;
                    bu[i] = max(bu[i], b);
                }
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
    float* out = (FUSED && Sx == 1) ? y : part + (size_t)sx * T * N;
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
    if (FUSED && Sx > 1) {
        __shared__ int s_last;
        __syncthreads();  // the CTA's partial is complete ...
        if (tid == 0) {
            __threadfence();  // ... and (fence cumulativity over the barrier) visible device-wide before its ticket
            const int last = (atomicAdd(&tickets[tile], 1) == Sx - 1);
            if (last) __threadfence();  // acquire side: the other CTAs' partials, read below with ld.global.cg
            s_last = last;
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

// y[t][n] = sum_{s=0}^{S-1} part[s][t][n], sequentially in s: the same order as the fused second pass, so the
// two-launch form returns the same bits.
__global__ void __launch_bounds__(VTHREADS)
vmm_reduce_kernel(const float* __restrict__ part, int S, int T, int N, float* __restrict__ y) {
    const int t = blockIdx.y;
    const int n = (blockIdx.x * VTHREADS + threadIdx.x) * 4;
    if (n >= N) return;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < S; ++s) {
        const float4 v = *reinterpret_cast<const float4*>(part + ((size_t)s * T + t) * N + n);
        a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
    }
    *reinterpret_cast<float4*>(y + (size_t)t * N + n) = a;
}

constexpr size_t TICKET_BYTES = 16384;  // head of the workspace: one int per column tile, zero between launches

template <int T, int VWT, bool A16, bool FUSED>
static int launch_main_impl(int K, int N, const VmmPlan& pl, const uint32_t* planes, const void* scales,
                            const void* zeros, const uint32_t* gsched, const uint8_t* gcnt_ge, void* workspace,
                            float* y, cudaStream_t st, const uint16_t* xraw, const ThrParams& tp) {
    constexpr int smem = Cfg<T>::WARP_BYTES * VWT;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(vmm_main_kernel<T, VWT, A16, FUSED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 smem) != cudaSuccess)
            return GRINQH_ERR_CUDA;
        configured = true;
    }
    dim3 grid(pl.col_tiles, pl.Sx);
    const uint32_t rq = (65536u + pl.Q - 1) / pl.Q;
    const cudaError_t e = launch_pdl(vmm_main_kernel<T, VWT, A16, FUSED>, grid, dim3(VWT * 32), (size_t)smem, st, K, N,
                                     pl.Q, rq, pl.ipw, pl.Sx, planes, (const __half*)scales, (const __half*)zeros,
                                     gsched, gcnt_ge, (float*)((char*)workspace + TICKET_BYTES), (int*)workspace, y,
                                     xraw, tp);
    return e == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

template <bool FUSED>
static int launch_main(int T, int K, int N, const VmmPlan& pl, const uint32_t* planes, const void* scales,
                       const void* zeros, const uint32_t* gsched, const uint8_t* gcnt_ge, void* ws, float* y,
                       cudaStream_t st, const uint16_t* xraw = nullptr, const ThrParams& tp = ThrParams{}) {
#define GQ_LAUNCH_W(TT, WW)                                                                                              \
    return (N % 128 == 0)                                                                                                \
               ? launch_main_impl<TT, WW, true, FUSED>(K, N, pl, planes, scales, zeros, gsched, gcnt_ge, ws, y, st, xraw, tp) \
               : launch_main_impl<TT, WW, false, FUSED>(K, N, pl, planes, scales, zeros, gsched, gcnt_ge, ws, y, st, xraw, tp)
    if (pl.vw == 16) {  // only planned for T <= 2 (registers)
        if (T == 1) { GQ_LAUNCH_W(1, 16); }
        GQ_LAUNCH_W(2, 16);
    }
#define GQ_LAUNCH(TT) GQ_LAUNCH_W(TT, 8)
    switch (T) {
        case 1: GQ_LAUNCH(1);
        case 2: GQ_LAUNCH(2);
        case 3: GQ_LAUNCH(3);
        default: GQ_LAUNCH(4);
    }
#undef GQ_LAUNCH_W
#undef GQ_LAUNCH
}

static int check_vmm_args(int T, int K, int N, int group) {
    if (group != GQ_G || T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32 || K > GQ_MAX_K)
        return GRINQH_ERR_SHAPE;  // (K <= 32768 as for grinqh_assign: the item arithmetic assumes <= 4096 items per tile)
    if ((size_t)((N + TILE_COLS - 1) / TILE_COLS) * sizeof(int) > TICKET_BYTES) return GRINQH_ERR_SHAPE;
    return GRINQH_OK;
}

static int check_vmm_ptrs(int T, int K, int N, int group, const void* planes, const void* scales, const void* zeros,
                          const void* gsched, const void* gcnt_ge, const void* workspace, size_t workspace_bytes) {
    if (!planes || !scales || !zeros || !gsched || !gcnt_ge || !workspace) return GRINQH_ERR_NULL;
    const int rc = check_vmm_args(T, K, N, group);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)planes | (uintptr_t)scales | (uintptr_t)zeros | (uintptr_t)gsched | (uintptr_t)gcnt_ge |
         (uintptr_t)workspace) & 15)
        return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    return GRINQH_OK;
}

}  // namespace gq

extern "C" size_t grinqh_vmm_workspace_bytes(int T, int K, int N) {
    if (gq::check_vmm_args(T, K, N, GQ_G) != GRINQH_OK) return 0;
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    return gq::TICKET_BYTES + (size_t)pl.Sx * T * N * sizeof(float);
}

extern "C" int grinqh_vmm_workspace_init(void* workspace, size_t workspace_bytes, void* stream) {
    if (!workspace) return GRINQH_ERR_NULL;
    if ((uintptr_t)workspace & 15) return GRINQH_ERR_ALIGN;
    if (workspace_bytes < gq::TICKET_BYTES) return GRINQH_ERR_WORKSPACE;
    return cudaMemsetAsync(workspace, 0, gq::TICKET_BYTES, (cudaStream_t)stream) == cudaSuccess ? GRINQH_OK
                                                                                                : GRINQH_ERR_CUDA;
}

extern "C" int grinqh_vmm(int T, int K, int N, int group, const uint32_t* planes, const void* scales_f16,
                          const void* zeros_f16, const uint32_t* gsched, const uint8_t* gcnt_ge, float* y,
                          void* workspace, size_t workspace_bytes, void* stream) {
    if (!y) return GRINQH_ERR_NULL;
    if ((uintptr_t)y & 15) return GRINQH_ERR_ALIGN;
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, gsched, gcnt_ge, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    return gq::launch_main<true>(T, K, N, gq::vmm_plan(T, K, N), planes, scales_f16, zeros_f16, gsched, gcnt_ge,
                                 workspace, y, (cudaStream_t)stream);
}

extern "C" int grinqh_vmm_main(int T, int K, int N, int group, const uint32_t* planes, const void* scales_f16,
                               const void* zeros_f16, const uint32_t* gsched, const uint8_t* gcnt_ge,
                               void* workspace, size_t workspace_bytes, void* stream) {
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, gsched, gcnt_ge, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    return gq::launch_main<false>(T, K, N, gq::vmm_plan(T, K, N), planes, scales_f16, zeros_f16, gsched, gcnt_ge,
                                  workspace, nullptr, (cudaStream_t)stream);
}

extern "C" int grinqh_vmm_reduce(int T, int K, int N, float* y, const void* workspace, size_t workspace_bytes,
                                 void* stream) {
    if (!y || !workspace) return GRINQH_ERR_NULL;
    int rc = gq::check_vmm_args(T, K, N, GQ_G);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)y | (uintptr_t)workspace) & 15) return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    dim3 grid((N + 4 * gq::VTHREADS - 1) / (4 * gq::VTHREADS), T);
    gq::vmm_reduce_kernel<<<grid, gq::VTHREADS, 0, (cudaStream_t)stream>>>(
        (const float*)((const char*)workspace + gq::TICKET_BYTES), pl.Sx, T, N, y);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

// SURVEY.md 8f4 (assignment fused into the consumer): the paper's threshold assignment made inside
// the VMM launch — every warp derives its group's widths and list from x and theta; one launch per projection and
// no assignment kernel.  y equals grinqh_assign_thresholds + grinqh_vmm bit for bit.
extern "C" int grinqh_vmm_thresholds(const void* x_f16, int T, int K, int N, int group, const uint16_t theta[9],
                                     const uint32_t* planes, const void* scales_f16, const void* zeros_f16, float* y,
                                     void* workspace, size_t workspace_bytes, void* stream) {
    if (!y || !x_f16 || !theta) return GRINQH_ERR_NULL;
    if (((uintptr_t)y | (uintptr_t)x_f16) & 15) return GRINQH_ERR_ALIGN;
    // (the schedule pointers are unused in this mode; pass the planes pointer to satisfy the shared checks)
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, planes, planes, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    for (int w = 1; w <= 8; ++w)
        if (theta[w] > 0x8000 || (w > 1 && theta[w] < theta[w - 1])) return GRINQH_ERR_MIX;
    gq::ThrParams tp;
    int nd = 0;
    for (int d = 0; d < 8; ++d) {
        tp.thr[d] = 0x8000;
        tp.mult[d] = 0;
    }
    for (int w = 1; w <= 8; ++w) {  // distinct reachable thresholds
        if (theta[w] == 0x8000) continue;
        int d = 0;
        while (d < nd && tp.thr[d] != (int)theta[w]) ++d;
        if (d == nd) tp.thr[nd++] = (int)theta[w];
        tp.mult[d]++;
    }
    return gq::launch_main<true>(T, K, N, gq::vmm_plan(T, K, N), planes, scales_f16, zeros_f16, nullptr, nullptr,
                                 workspace, y, (cudaStream_t)stream, (const uint16_t*)x_f16, tp);
}
