// prefill.cu — grinqh_prefill_gemm: the paper's prefill path ("unpacking the weights at full b_max precision
// and performing dense matrix-matrix multiplication", :182 "efficient unpacking and kernel fusion"; Table 2 :158-166;
// SURVEY.md 8f3) as ONE kernel: Y[M, N] = X[M, K] . W_hat[K, N], W_hat = s * q + z rounded once to fp16 (the value
// grinqh_unpack writes), with the unpack fused into the operand staging of a tcgen05 GEMM.  HBM sees 1 byte per weight
// (the 8 planes) instead of 1 + 2 + 2 (unpack's read and write, then the GEMM's read of the fp16 matrix).
//
// One CTA = one 256 x 256 tile of Y (two 128-row accumulators of 256 fp32 columns: all 512 TMEM columns), K in blocks
// of 64, STAGES-deep shared-memory ring.  Warp roles (no role waits inside another's critical section):
//   warps 0-15 B producers, then epilogue.  Per stage each lane takes one (row k, 32-column word) unit: 8 plane words
//              from the raw buffer (LDS, conflict-free) -> SIMD 8x8 bit transpose (gather.cuh) -> bytes widened to fp16 subnormals by PRMT,
//              x 2^15 (exact), HFMA2 with (s 2^9, z): the correctly rounded s q + z -> four 16-byte chunks into the
//              stage's B tile in the canonical MN-major SWIZZLE_128B layout (64 columns x 8 k-rows per 1-KB atom).
//              The 32 columns of a word are stored in the order the transpose leaves them (a fixed permutation inside
//              the word); the epilogue undoes it on registers.  fence.proxy.async, then the warp arrives on `full`.
//   warp 16    TMA producer: the stage's two 128 x 64 X boxes (K-major, SWIZZLE_128B) with complete_tx on `full`.
//   warp 17    TMA producer for the plane words: one 3-D box per k block (8 planes x 64 rows x 32 bytes) into a raw double
//              buffer [plane][row][8 words] (`rawfull` / `rawempty`).  Per-lane global loads stalled the producers: 1024
//              sectors in flight per SM are more than the L1 miss path tracks (profiles/r02_prefill.md).
//   warp 18    MMA issuer: one lane issues 2 x 4 tcgen05.mma (M 128, N 256, K 16, fp16 x fp16 -> fp32 in TMEM) per stage,
//              tcgen05.commit -> `empty` (frees the stage) and, after the last block, -> `accum`.
//   epilogue   warps 0-15 (TMEM lane quarter = warp % 4, accumulator and column half from warp / 4): tcgen05.ld 32 columns, un-permute,
//              fp32 -> fp16, 64 contiguous bytes per row and word to Y.
// Every mbarrier wait is bounded (a trap instead of a hang if a count is ever wrong).
#include <cuda.h>

#include <cstdlib>
#include <mutex>

#include "common.cuh"
#include "gather.cuh"

namespace gq {
namespace prefill {

constexpr int BM = 128;  // rows per accumulator (UMMA M)
constexpr int MT = 2;    // accumulators per CTA
constexpr int BN = 256;  // columns per CTA (UMMA N)
constexpr int BK = 64;   // k per stage: one 128-byte swizzle row of fp16
constexpr int UK = 16;   // k per tcgen05.mma (fp16)
constexpr int STAGES = 3;
constexpr int A_TILE = BM * BK * 2;         // 16 KB: one TMA box
constexpr int A_STAGE = MT * A_TILE;        // 32 KB
constexpr int B_STAGE = BK * BN * 2;        // 32 KB
constexpr int STAGE_BYTES = A_STAGE + B_STAGE;
constexpr int NPROD = 16;                   // producer / epilogue warps
constexpr int THREADS = (NPROD + 3) * 32;   // + TMA warp for X, TMA warp for the planes, MMA warp
constexpr int RAW_BYTES = 8 * BK * (BN / 32) * 4;  // 16 KB: the stage's plane words, [plane][row][8 words]
constexpr int RAW_BUFS = 2;
constexpr int RAW_OFF = STAGES * STAGE_BYTES;
constexpr int BAR_OFF = RAW_OFF + RAW_BUFS * RAW_BYTES;
constexpr int SMEM_BYTES = BAR_OFF + 1024 /* alignment slack */ + 256 /* barriers */;
constexpr uint32_t TMEM_COLS = MT * BN;     // 512

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// bounded wait: ~2 s of polling, then a trap (an error the host sees) instead of a hung GPU
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok = 0;
#pragma unroll 1
    for (uint32_t spin = 0; spin < (1u << 26); ++spin) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.b32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity), "r"(2000u)  // suspend-time hint (ns): a waiting warp sleeps instead of polling
            : "memory");
        if (ok) return;
    }
    __trap();
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
        : "memory");
}

// shared-memory matrix descriptor (tcgen05): start address, leading / stride byte offsets in 16-byte units, version 1
// (Blackwell) at bit 46, layout type SWIZZLE_128B (= 2) at bits 61-63
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor, kind::f16: D fp32 (bits 4-5 = 1), A and B fp16 (0), A K-major (bit 15 = 0), B MN-major
// (bit 16 = 1), N / 8 at bits 17-22, M / 16 at bits 24-28
constexpr uint32_t IDESC = (1u << 4) | (1u << 16) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);

__device__ __forceinline__ void mma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "r"(IDESC), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

__device__ __forceinline__ uint32_t h2_mul(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t h2_fma(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}

// Position p (0..31) of a word's 32 columns in the B tile / the accumulator <-> column c of the word: the order in
// which the bit transpose leaves the codes (V[r] byte i = column 8 i + r).  Chunk jj = p / 8 holds V[2 jj], V[2 jj + 1]:
// half2 q = (p / 2) % 4: r = 2 jj + q / 2, bytes i = 2 (q % 2) + p % 2.
__host__ __device__ constexpr int col_of_pos(int p) {
    return 8 * (2 * (((p >> 1) & 3) & 1) + (p & 1)) + 2 * (p >> 3) + (((p >> 1) & 3) >> 1);
}
__host__ __device__ constexpr int pos_of_col(int c) {
    // c = 8 i + r:  jj = r / 2,  q = 2 (r % 2) + i / 2,  h = i % 2
    return 8 * ((c & 7) >> 1) + 2 * (2 * ((c & 7) & 1) + ((c >> 3) >> 1)) + ((c >> 3) & 1);
}

__global__ void __launch_bounds__(THREADS, 1)
prefill_kernel(const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap pmap, int M, int K, int N,
               const __half* __restrict__ scales, const __half* __restrict__ zeros, __half* __restrict__ Y, int dbg_arg) {
#ifdef GQ_PREFILL_DBG
    const int dbg = dbg_arg;  // measurement build only: legs of the kernel switched off (results are then wrong on purpose)
#else
    constexpr int dbg = 0;
    (void)dbg_arg;
#endif
    extern __shared__ uint8_t smem_raw[];
    const uint32_t raw = smem_u32(smem_raw);
    const uint32_t base = (raw + 1023u) & ~1023u;  // the swizzle atoms are 1 KB
    uint8_t* sm = smem_raw + (base - raw);
    const uint32_t bars = base + BAR_OFF;
    auto full = [&](int s) { return bars + 8u * s; };
    auto empty = [&](int s) { return bars + 8u * (STAGES + s); };
    const uint32_t accum = bars + 8u * (2 * STAGES);
    auto rawfull = [&](int i) { return bars + 8u * (2 * STAGES + 2 + i); };
    auto rawempty = [&](int i) { return bars + 8u * (2 * STAGES + 2 + RAW_BUFS + i); };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(sm + BAR_OFF + 8 * (2 * STAGES + 1));

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n0 = blockIdx.x * BN, m0 = blockIdx.y * (MT * BM);
    const int KB = K / BK;

    if (warp == NPROD + 2 && lane == 0) {
        for (int i = 0; i < RAW_BUFS; ++i) {
            mbar_init(rawfull(i), 1);       // the plane TMA thread's arrive.expect_tx
            mbar_init(rawempty(i), NPROD);  // every producer warp has taken its words
        }
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full(s), NPROD + 1);  // the producer warps + the TMA thread's arrive.expect_tx
            mbar_init(empty(s), 1);         // one tcgen05.commit
        }
        mbar_init(accum, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_proxy_async();
    }
    if (warp == NPROD && lane == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&xmap) : "memory");
    if (warp == NPROD + 1 && lane == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&pmap) : "memory");
    if (warp == 0) {  // the whole warp allocates all 512 TMEM columns (one CTA per SM: nobody else asks)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         bars + 8u * (2 * STAGES + 1)),
                     "r"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp < NPROD) {
        // ================================================================ B producers
        // lane -> (row, word): the 8 lanes of a store phase take 4 rows x 2 words (8 distinct swizzled chunks: no bank
        // conflict) and a warp's plane load covers 4 rows x the tile's 8 words = whole 32-byte sectors
        const int word = lane >> 2;                     // the lane's 32-column word of the tile, fixed for the whole K loop
        const int katom = warp >> 1;                    // the lane's k atom (8 rows) of every stage
        const int kk = 4 * (warp & 1) + (lane & 3);     // row inside the atom
        // the lane's word of plane j in the raw tile [plane][row][8 words]: the 32 lanes of a warp hit 32 distinct banks
        const uint32_t raw_off = RAW_OFF + (uint32_t)(katom * 8 + kk) * 32u + (uint32_t)word * 4u;
        const uint32_t b_off = A_STAGE + (uint32_t)(word >> 1) * 8192u + (uint32_t)katom * 1024u + (uint32_t)kk * 128u;
        const uint32_t j0 = (uint32_t)(word & 1) * 4u;
        const uint32_t K15 = 0x78007800u;  // 2^15 | 2^15
        const uint32_t K9 = 0x60006000u;   // 2^9 | 2^9
        const __half* sz_s = scales + n0 + word * 32;
        const __half* sz_z = zeros + n0 + word * 32;

        uint32_t S2[8][2], Z2[8][2];  // {s[r], s[8+r]} 2^9, {s[16+r], s[24+r]} 2^9 and the zeros in the same pairing
        auto load_sz = [&](int g) {   // group g's scales and zeros of the lane's 32 columns
            const size_t gn = (size_t)g * N;
            uint32_t sr[16], zr[16];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint4 a = __ldg(reinterpret_cast<const uint4*>(sz_s + gn + 8 * i));
                const uint4 b = __ldg(reinterpret_cast<const uint4*>(sz_z + gn + 8 * i));
                sr[4 * i] = a.x; sr[4 * i + 1] = a.y; sr[4 * i + 2] = a.z; sr[4 * i + 3] = a.w;
                zr[4 * i] = b.x; zr[4 * i + 1] = b.y; zr[4 * i + 2] = b.z; zr[4 * i + 3] = b.w;
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const uint32_t sel = (r & 1) ? 0x7632u : 0x5410u;  // the odd or the even halves of the two registers
                S2[r][0] = h2_mul(__byte_perm(sr[r >> 1], sr[(8 + r) >> 1], sel), K9);
                S2[r][1] = h2_mul(__byte_perm(sr[(16 + r) >> 1], sr[(24 + r) >> 1], sel), K9);
                Z2[r][0] = __byte_perm(zr[r >> 1], zr[(8 + r) >> 1], sel);
                Z2[r][1] = __byte_perm(zr[(16 + r) >> 1], zr[(24 + r) >> 1], sel);
            }
            if ((g + 1) * 2 < KB) {  // the next group's lines are asked for now
                asm volatile("prefetch.global.L2 [%0];" ::"l"(sz_s + gn + N));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(sz_z + gn + N));
            }
        };
        // one stage: the lane's unit of k block kb
        auto produce = [&](int kb) {
            const int s = kb % STAGES;
            const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
            const int rb = kb % RAW_BUFS;
            uint32_t W[8], V[8], H[8][2];
            mbar_wait(rawfull(rb), (uint32_t)(kb / RAW_BUFS) & 1u);  // the stage's plane words have landed (TMA)
#pragma unroll
            for (int j = 0; j < 8; ++j)
                asm volatile("ld.shared.b32 %0, [%1];" : "=r"(W[j]) : "r"(base + raw_off + (uint32_t)rb * RAW_BYTES + (uint32_t)j * 2048u));
            gather<8>(W, V);
            __syncwarp();
            if (lane == 0) mbar_arrive(rawempty(rb));  // the warp's loads have returned (their values are consumed above)
            if (dbg & 1) {
                mbar_wait(empty(s), ph ^ 1u);
                __syncwarp();
                if (lane == 0) mbar_arrive(full(s) + (V[0] == 0x12345678u ? 1u : 0u));
                return;
            }
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                // bytes -> fp16 subnormals q 2^-24 (PRMT with zero), x 2^15 (exact), then q 2^-9 * s 2^9 + z: one rounding
                H[r][0] = h2_fma(h2_mul(__byte_perm(V[r], 0u, 0x4140), K15), S2[r][0], Z2[r][0]);
                H[r][1] = h2_fma(h2_mul(__byte_perm(V[r], 0u, 0x4342), K15), S2[r][1], Z2[r][1]);
            }
            mbar_wait(empty(s), ph ^ 1u);
            const uint32_t dst = base + (uint32_t)s * STAGE_BYTES + b_off;
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const uint32_t a = dst + (((j0 + jj) ^ (uint32_t)kk) << 4);
                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(H[2 * jj][0]), "r"(H[2 * jj][1]),
                             "r"(H[2 * jj + 1][0]), "r"(H[2 * jj + 1][1])
                             : "memory");
            }
            if (!(dbg & 8)) fence_proxy_async();  // the tile is read by the tensor core through the async proxy
            __syncwarp();
            if (lane == 0) mbar_arrive(full(s));
        };
#pragma unroll 1
        for (int kb = 0; kb < KB; ++kb) {
            if ((kb & 1) == 0) load_sz(kb >> 1);  // a new group of 128 rows
            produce(kb);
        }
    } else if (warp == NPROD) {
        // ================================================================ TMA producer (X)
        if (lane == 0) {
#pragma unroll 1
            for (int kb = 0; kb < KB; ++kb) {
                const int s = kb % STAGES;
                const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
                mbar_wait(empty(s), ph ^ 1u);
                mbar_arrive_expect_tx(full(s), A_STAGE);
                const uint32_t a = base + (uint32_t)s * STAGE_BYTES;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) tma_load_2d(a + mt * A_TILE, &xmap, (dbg & 4) ? 0 : kb * BK, m0 + mt * BM, full(s));
            }
        }
    } else if (warp == NPROD + 1) {
        // ================================================================ TMA producer (plane words): one 3-D box per k block,
        // 8 planes x 64 rows x 32 bytes, into the raw double buffer; no L1 miss tracking, no registers, no address arithmetic
        if (lane == 0) {
#pragma unroll 1
            for (int kb = 0; kb < KB; ++kb) {
                const int rb = kb % RAW_BUFS;
                mbar_wait(rawempty(rb), ((uint32_t)(kb / RAW_BUFS) & 1u) ^ 1u);
                mbar_arrive_expect_tx(rawfull(rb), RAW_BYTES);
                if (!(dbg & 16)) tma_load_3d(base + RAW_OFF + (uint32_t)rb * RAW_BYTES, &pmap, n0 >> 5, kb * BK, 0, rawfull(rb));
                else asm volatile("mbarrier.complete_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(rawfull(rb)), "r"((uint32_t)RAW_BYTES) : "memory");
            }
        }
    } else {
        // ================================================================ MMA issuer
#pragma unroll 1
        for (int kb = 0; kb < KB; ++kb) {
            const int s = kb % STAGES;
            const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
            mbar_wait(full(s), ph);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t a = base + (uint32_t)s * STAGE_BYTES, b = a + A_STAGE;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                    for (int k4 = 0; k4 < BK / UK; ++k4) {
                        // A: K-major, 128-byte rows, 8-row atoms 1 KB apart; 16 k = 32 bytes further along the row
                        const uint64_t ad = smem_desc(a + mt * A_TILE + k4 * (UK * 2), 16, 1024);
                        // B: MN-major atoms of 64 columns x 8 k: column atoms 8 KB apart, k atoms 1 KB apart; 16 k = 2 atoms
                        const uint64_t bd = smem_desc(b + k4 * 2048, 8192, 1024);
                        if (!(dbg & 2)) mma_f16(tmem + (uint32_t)(mt * BN), ad, bd, (uint32_t)((kb | k4) != 0));
                    }
                mma_commit(empty(s));
                if (kb == KB - 1) mma_commit(accum);
            }
            __syncwarp();
        }
    }

    if (warp < NPROD) {
        // ================================================================ epilogue
        mbar_wait(accum, 0);
        tc_fence_after();
        const int quarter = warp & 3, mt = (warp >> 2) & 1, chalf = warp >> 3;  // 16 warps: 2 accumulators x 2 column halves
        const int m = m0 + mt * BM + quarter * 32 + lane;
#pragma unroll 1
        for (int cb = chalf * (BN / 64); cb < (chalf + 1) * (BN / 64); ++cb) {
            uint32_t v[32];
            tmem_ld32(tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(mt * BN + cb * 32), v);
            if (m < M) {
                uint32_t o[16];
#pragma unroll
                for (int c = 0; c < 32; c += 2) {
                    const __half2 h = __floats2half2_rn(__uint_as_float(v[pos_of_col(c)]), __uint_as_float(v[pos_of_col(c + 1)]));
                    o[c >> 1] = *reinterpret_cast<const uint32_t*>(&h);
                }
                uint4* dst = reinterpret_cast<uint4*>(Y + (size_t)m * N + n0 + cb * 32);
#pragma unroll
                for (int i = 0; i < 4; ++i) dst[i] = make_uint4(o[4 * i], o[4 * i + 1], o[4 * i + 2], o[4 * i + 3]);
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(TMEM_COLS) : "memory");
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    });
    return fn;
}

}  // namespace prefill
}  // namespace gq

extern "C" int grinqh_prefill_gemm(const void* x_f16, int M, int K, int N, int group, const uint32_t* planes,
                                   const void* scales_f16, const void* zeros_f16, void* y_f16, void* stream) {
    using namespace gq::prefill;
    if (!x_f16 || !planes || !scales_f16 || !zeros_f16 || !y_f16) return GRINQH_ERR_NULL;
    if (group != GQ_G || M <= 0 || K <= 0 || N <= 0 || K % GQ_G || N % BN) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_f16 | (uintptr_t)planes | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16 | (uintptr_t)y_f16) & 15)
        return GRINQH_ERR_ALIGN;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return GRINQH_ERR_CUDA;
    CUtensorMap xmap;
    const cuuint64_t dims[2] = {(cuuint64_t)K, (cuuint64_t)M};       // innermost first
    const cuuint64_t strides[1] = {(cuuint64_t)K * 2};               // bytes between rows
    const cuuint32_t box[2] = {(cuuint32_t)BK, (cuuint32_t)BM};      // 64 k (128 bytes) x 128 rows
    const cuuint32_t estr[2] = {1, 1};
    if (enc(&xmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(x_f16), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return GRINQH_ERR_CUDA;
    CUtensorMap pmap;  // planes as [8 planes][K rows][N/32 words] u32, box = 8 words x 64 rows x 8 planes
    const cuuint64_t pdims[3] = {(cuuint64_t)(N / 32), (cuuint64_t)K, 8};
    const cuuint64_t pstrides[2] = {(cuuint64_t)(N / 8), (cuuint64_t)K * (cuuint64_t)(N / 8)};
    const cuuint32_t pbox[3] = {(cuuint32_t)(BN / 32), (cuuint32_t)BK, 8};
    const cuuint32_t pestr[3] = {1, 1, 1};
    if (enc(&pmap, CU_TENSOR_MAP_DATA_TYPE_UINT32, 3, const_cast<uint32_t*>(planes), pdims, pstrides, pbox, pestr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return GRINQH_ERR_CUDA;
    int dbg = 0;
#ifdef GQ_PREFILL_DBG  // GQ_NVCC_EXTRA=-DGQ_PREFILL_DBG: 1 no unpack, 2 no MMA, 4 X from k = 0, 8 no proxy fence, 16 no plane loads
    if (const char* e = getenv("GRINQH_PREFILL_DBG")) dbg = atoi(e);
#endif
    if (cudaFuncSetAttribute(prefill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess)
        return GRINQH_ERR_CUDA;
    dim3 grid(N / BN, (M + MT * BM - 1) / (MT * BM));
    prefill_kernel<<<grid, THREADS, SMEM_BYTES, (cudaStream_t)stream>>>(xmap, pmap, M, K, N, (const __half*)scales_f16,
                                                                         (const __half*)zeros_f16, (__half*)y_f16, dbg);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}
