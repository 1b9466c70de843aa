// gather.cuh — plane words -> truncated codes in byte lanes (SIMD-in-register 8x8 bit transpose).
//
// A lane holds one 32-bit word per fetched plane of a weight row: W[j] bit p = code bit (7-j) of column p
// of the lane's 32-column block (the b-bit code is the top b planes).  gather<B> runs
// the three butterfly stages of an 8x8 bit-matrix transpose on all four byte lanes at once and returns
// V[r], r = 0..7, with   byte L of V[r] = truncated code (top B bits, low bits 0) of column 8 L + r.
// Planes j >= B are treated as zero, so stages that would only move zeros fold away at compile time:
// 36 + 12, 20 + 8 and 15 + 7 ops for B = 8, 4, 2 per 32 weights (logic or right shift on the half-rate pipe + left
// shifts that the compiler issues as IMAD.SHL on the FMA pipe).
//
// Plain C++ on uint32_t so that the same code is unit-tested on the host (tests/test_host_logic.py).
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define GQ_HD __host__ __device__ __forceinline__
#else
#define GQ_HD inline
#endif

namespace gq {

// transpose step on the pair (lo, hi) = (row i, row i+s) of every 8x8 byte-lane block:
//   lo' = (lo & m) | ((hi & m) << s),   hi' = ((lo >> s) & m) | (hi & ~m),   m = low s bits of each 2s.
//   LOZ: lo is known to be zero (its planes are not fetched), so the step is a shift and two masks.
template <int S, bool LOZ>
GQ_HD void tstep(uint32_t& lo, uint32_t& hi) {
    constexpr uint32_t m = (S == 1) ? 0x55555555u : (S == 2) ? 0x33333333u : 0x0F0F0F0Fu;
    if (LOZ) {
        lo = (hi << S) & ~m;
        hi = hi & ~m;
        return;
    }
    // two bit-selects under the one mask m (m << S == ~m): one LOP3 each after its shift.  The compiler rewrites the
    // C form into and + or-and (2 LOP3 per output on the half-rate pipe), so the device path spells the LOP3 out.
    const uint32_t H = hi << S, L = lo >> S;
#if defined(__CUDA_ARCH__)
    uint32_t nlo, nhi;
    asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(nlo) : "r"(lo), "r"(H), "r"(m));  // (lo & m) | (H & ~m)
    asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(nhi) : "r"(L), "r"(hi), "r"(m));  // (L & m) | (hi & ~m)
#else
    const uint32_t nlo = (lo & m) | (H & ~m);
    const uint32_t nhi = (L & m) | (hi & ~m);
#endif
    lo = nlo;
    hi = nhi;
}

// W[j], j < B: plane words (W[j] for j >= B is ignored).  V[r]: byte L = code of column 8L + r.
template <int B>
GQ_HD void gather(const uint32_t (&W)[8], uint32_t (&V)[8]) {
    static_assert(B == 2 || B == 4 || B == 8, "gather is instantiated for 2, 4 or 8 planes");
    // a[i] carries code bit i = plane 7 - i
#pragma unroll
    for (int i = 0; i < 8; ++i) V[i] = (7 - i < B) ? W[7 - i] : 0u;
    tstep<1, false>(V[6], V[7]);
    if (B > 2) tstep<1, false>(V[4], V[5]);
    if (B > 4) {
        tstep<1, false>(V[0], V[1]);
        tstep<1, false>(V[2], V[3]);
    }
    tstep<2, (B <= 2)>(V[4], V[6]);
    tstep<2, (B <= 2)>(V[5], V[7]);
    if (B > 4) {
        tstep<2, false>(V[0], V[2]);
        tstep<2, false>(V[1], V[3]);
    }
    tstep<4, (B <= 4)>(V[0], V[4]);
    tstep<4, (B <= 4)>(V[1], V[5]);
    tstep<4, (B <= 4)>(V[2], V[6]);
    tstep<4, (B <= 4)>(V[3], V[7]);
}

// ---- 2-bit-segment store.  a[sg], sg < NS: the segment words of one 16-column
// half (column c's pair at bits 2c + 1, 2c; segment 0 = the most significant pair).  X[j], j = 0..3: byte i = the code
// of column 4 i + j, left-aligned in the byte (segment sg at bits 7 - 2 sg, 6 - 2 sg), missing segments zero.  Two
// stages of a 4 x 4 transpose of 2-bit elements: the first butterfly stage of the 1-bit store is already in the layout.
template <int NS>
GQ_HD void gather_seg2(const uint32_t (&a)[4], uint32_t (&X)[4]) {
    static_assert(NS >= 1 && NS <= 4, "1 to 4 segments");
    constexpr uint32_t M2 = 0x33333333u, M4 = 0x0F0F0F0Fu;
    // nibble j of pe / po = (a0 element << 2) | a1 element of columns 2 j / 2 j + 1; qe / qo the same of a2, a3
    const uint32_t pe = (NS >= 2) ? (((a[0] << 2) & ~M2) | (a[1] & M2)) : ((a[0] << 2) & ~M2);
    const uint32_t po = (NS >= 2) ? ((a[0] & ~M2) | ((a[1] >> 2) & M2)) : (a[0] & ~M2);
    const uint32_t qe = (NS >= 4) ? (((a[2] << 2) & ~M2) | (a[3] & M2)) : (NS == 3) ? ((a[2] << 2) & ~M2) : 0u;
    const uint32_t qo = (NS >= 4) ? ((a[2] & ~M2) | ((a[3] >> 2) & M2)) : (NS == 3) ? (a[2] & ~M2) : 0u;
    X[0] = ((pe & M4) << 4) | (qe & M4);
    X[2] = (pe & ~M4) | ((qe >> 4) & M4);
    X[1] = ((po & M4) << 4) | (qo & M4);
    X[3] = (po & ~M4) | ((qo >> 4) & M4);
}

}  // namespace gq
