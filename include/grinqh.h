/*
 * grinqh.h — C ABI of the B200-native GRINQH decode hot path.
 *
 * Method: GRINQH (arxiv/paper_2606_23419).  Citations are PAPER.md:LINE of the
 * paper text this build was written from.
 *
 *   y[t, n] = sum_k  x[t, k] * w_hat(k, n; b_tk)
 *
 * over a bit-planar, nested 8-bit weight store.  Every decode
 * step each input channel k of the current vector gets a bit width b_k in
 * {0..8} from the rank of |x_k| (top-p form of :271) and only
 * the top b_k bit planes of weight row k are fetched; the truncated code is
 * reconstructed with the paper's midpoint bias
 *
 *   w_hat = s * (q_b * 2^(8-b) + phi_b) + z ,   phi_b = 2^(8-b-1)
 *
 * with phi_8 = 0 and a b = 0 row contributing exactly nothing (DESIGN.md
 * readings #5, #7).
 *
 * Conventions for every call below
 *   - "dev" pointers are DEVICE pointers owned by the caller; "host" pointers
 *     are ordinary host memory.  The library never allocates, frees or keeps a
 *     pointer after the call returns.
 *   - Every call only ENQUEUES work on `stream` (a cudaStream_t passed as
 *     void*; NULL = the legacy default stream).  Nothing synchronises.  All
 *     device entry points are CUDA-graph capturable.
 *   - Return value: GRINQH_OK (0) or a negative grinqh_status.  On error
 *     nothing has been enqueued.
 *   - W is [K, N] row-major fp16: K = d_in rows (input channels), N = d_out.
 *     group = 128 consecutive input channels of one output column
 *     ("group size G=128").  Required: K % 128 == 0, K <= 32768, N % 32 == 0,
 *     1 <= T <= 4, all base pointers 16-byte aligned.
 *   - Plane j (j = 0 is the MSB, code bit 7) is planes[j][k][n >> 5], column n
 *     sits at bit (n & 31) of that word.  planes is one allocation of
 *     8 * K * (N/32) uint32.
 */
#ifndef GRINQH_H
#define GRINQH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GRINQH_OK = 0,
    GRINQH_ERR_NULL = -1,      /* a required pointer is NULL                              */
    GRINQH_ERR_SHAPE = -2,     /* K % 128, N % 32, T outside 1..4, group != 128, K > max  */
    GRINQH_ERR_ALIGN = -3,     /* a base pointer is not 16-byte aligned                   */
    GRINQH_ERR_MIX = -4,       /* sum(counts) != K                                        */
    GRINQH_ERR_WORKSPACE = -5, /* workspace_bytes smaller than *_workspace_bytes()        */
    GRINQH_ERR_CUDA = -6,      /* a CUDA launch failed; see cudaGetLastError              */
    GRINQH_ERR_STATIC_LIMIT = -7 /* grinqh_vmm_rank_static: the shape needs more scratch than the static array holds */
} grinqh_status;

#define GRINQH_GROUP 128
#define GRINQH_MAX_T 4
#define GRINQH_MAX_K 32768      /* the 15-bit key histogram and one token's keys live in one CTA's shared memory */
#define GRINQH_GCNT_STRIDE 16   /* bytes per group in gcnt_ge (entries 0..9 used)        */

/* Static strings, never freed. */
const char* grinqh_status_string(int status);
/* major*10000 + minor*100 + patch */
int grinqh_version(void);

/*
 * Host helper (Eq. 1: precision distribution P on the simplex).
 * frac[w] = share of input channels that get w bits, w = 0..8.  Cumulative
 * rounding from the top width: C_w = floor(K * sum_{v>=w} frac[v] + 0.5),
 * counts[w] = C_w - C_{w+1}, C_0 forced to K — always sums to K
 * (reading #3).  Returns GRINQH_ERR_MIX if |sum(frac) - 1| > 1e-6
 * or any frac < 0.
 */
int grinqh_mix_to_counts(int K, const double frac[9], uint32_t counts[9]);

/*
 * grinqh_pack — offline, once per weight.
 * Per (group g, column n): lo/hi = min/max of the 128 fp16 values;
 * s = fp16_rn((float(hi) - float(lo)) / 255), z = lo; if s == 0 all codes are 0,
 * else q = clamp(rint((float(w) - float(z)) / float(s)), 0, 255), IEEE fp32,
 * round-half-even, no FMA contraction (reading #8).  Code bit (7-j)
 * goes to plane j.
 *   W_f16      dev  [K, N] fp16, read only
 *   planes     dev  [8][K][N/32] uint32, written
 *   scales_f16 dev  [K/128][N] fp16, written
 *   zeros_f16  dev  [K/128][N] fp16, written
 */
int grinqh_pack(const void* W_f16, int K, int N, int group,
                uint32_t* planes, void* scales_f16, void* zeros_f16, void* stream);

/*
 * grinqh_unpack — the first half of the paper's prefill path ("unpack at b_max, dense GEMM";
 * stage decoupling :51).  Rebuilds the full 8-bit codes from the 8 planes and writes W_hat = s * q + z as fp16: the
 * fp64 value rounded once (round-to-nearest-even).  The dense GEMM that follows is an ordinary library GEMM on W_f16.
 *   planes, scales_f16, zeros_f16   dev   as written by grinqh_pack
 *   W_f16      dev  [K, N] fp16, written
 */
int grinqh_unpack(const uint32_t* planes, const void* scales_f16, const void* zeros_f16, int K, int N, int group,
                  void* W_f16, void* stream);

/*
 * grinqh_assign — every decode step, once per input vector
 * (PAPER.md:61-65 assignment, :271 top-p partition of the live vector).
 * Per token t: order channels by (|x_tk| descending, k ascending) on the 15
 * magnitude bits of the fp16 pattern; with C_w = sum_{v>=w} counts[v] the
 * channel at rank r gets b = max{w : r < C_w} (0 if r >= C_1).
 *   x_f16       dev   [T, K] fp16
 *   counts      HOST  [9], counts[w] = rows at width w, sum = K; read during the call
 *   bits        dev   [T][K] uint8       per-token widths
 *   bits_union  dev   [K] uint8          max over tokens (the planes actually fetched)
 *   rows        dev   [K] int32          all channels sorted by (bits_union desc, k asc):
 *                                        rows[0 : cnt_ge[j+1]] are exactly the rows needing plane j
 *   cnt_ge      dev   [10] int32         cnt_ge[w] = #{k : bits_union[k] >= w}; cnt_ge[0]=K, cnt_ge[9]=0
 *   grows       dev   [K] uint8          per 128-row group g, grows[128 g + i] = local index (0..127) of
 *                                        the i-th row of the group in (bits_union desc, k asc) order
 *   gcnt_ge     dev   [K/128][16] uint8  gcnt_ge[g][w] = #{k in group g : bits_union[k] >= w}, w = 0..9
 *                                        (entries 10..15 are zero)
 *   gsched      dev   [T][K] uint32      the per-group schedule grinqh_vmm walks: entry [t][128 g + i] describes
 *                                        the i-th row of group g's list, r = grows[128 g + i], k = 128 g + r:
 *                                          bits 0..7 r | 8..11 bits[t][k] | 12..15 bits_union[k] | 16..31 x[t][k] (fp16 pattern)
 *                                        a pure re-indexing of the outputs above (bit-exact against the oracle's)
 *   workspace   dev   unused: grinqh_assign_workspace_bytes returns 0 (everything lives in shared memory); the
 *                     arguments are kept for ABI stability and may be NULL / 0
 * Any of the seven output pointers may be NULL: that output is skipped (grinqh_vmm reads gsched only).
 */
size_t grinqh_assign_workspace_bytes(int T, int K);
int grinqh_assign(const void* x_f16, int T, int K, const uint32_t counts[9],
                  uint8_t* bits, uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge,
                  uint8_t* grows, uint8_t* gcnt_ge, uint32_t* gsched,
                  void* workspace, size_t workspace_bytes, void* stream);

/*
 * grinqh_assign_thresholds — the paper's own run-time form (b_i = b_k if |x_i| in
 * [theta_k, theta_{k+1}); "negligible latency", :73).  No ranking: b = max{w : m >= theta[w]} on the 15 magnitude
 * bits m of the fp16 pattern; the effective bits then float around the calibration target instead of hitting it
 * exactly.  Everything after the widths (union, rows, cnt_ge, grows, gcnt_ge, gsched) is as in grinqh_assign.
 *   theta   HOST [9] fp16 magnitude patterns, theta[w] (w = 1..8) = smallest magnitude that still gets >= w bits,
 *           non-decreasing in w, 0x8000 = width w unreachable; theta[0] ignored.  GRINQH_ERR_MIX if not monotone.
 *
 * grinqh_calibrate_thresholds — offline HOST helper (Eq. 2): for each of the S calibration
 * vectors the magnitude that separates the levels under the rank partition `counts` (the C_w-th largest |x|),
 * averaged in fp64, rounded to fp32 then fp16 (round-to-nearest-even); C_w == 0 -> 0x8000.
 *   x_host_f16  HOST [S, K] fp16      counts HOST [9], sum = K      theta HOST [9], written
 */
int grinqh_assign_thresholds(const void* x_f16, int T, int K, const uint16_t theta[9],
                             uint8_t* bits, uint8_t* bits_union, int32_t* rows, int32_t* cnt_ge,
                             uint8_t* grows, uint8_t* gcnt_ge, uint32_t* gsched, void* stream);
int grinqh_calibrate_thresholds(const void* x_host_f16, int S, int K, const uint32_t counts[9], uint16_t theta[9]);

/*
 * grinqh_vmm — per projection (PAPER.md:85 reconstruction, :51 selective fetch).
 * ONE launch: split-K main kernel (warps walk their slots of the per-group schedule and fetch only planes
 * j < bits_union[k] of row k) whose last-finishing CTA per column tile runs the deterministic second pass: it sums the tile's split-K
 * partials in the fixed order s = 0..S-1 (the result does not depend on which CTA is last).  fp32 accumulation.
 * For T > 1 each token is truncated to its own bits[t][k]; y[t] equals the T = 1 result of token t alone.
 * The activations enter through gsched (x values, widths and row order of the assignment).
 *   gsched, gcnt_ge   dev   as written by grinqh_assign for this [T, K] input (gcnt_ge is not read any more:
 *                           rows with b = 0 are recognised from their schedule entries; any non-NULL pointer will do)
 *   y          dev  [T, N] fp32, written
 *   workspace  dev  >= grinqh_vmm_workspace_bytes(T, K, N) bytes, 16-byte aligned.  Its first 16 KB hold the
 *                   per-tile tickets: call grinqh_vmm_workspace_init ONCE after allocating it (and again only
 *                   after an aborted launch); every launch leaves them zero.  One workspace may serve calls of
 *                   different shapes as long as they are ordered on one stream (size it for the largest).
 * grinqh_vmm_main / grinqh_vmm_reduce are the same computation as two launches (main writes the split-K partials
 * into workspace, reduce sums them into y in the same fixed order); they do not use the tickets.
 */
size_t grinqh_vmm_workspace_bytes(int T, int K, int N);
int grinqh_vmm_workspace_init(void* workspace, size_t workspace_bytes, void* stream);
int grinqh_vmm(int T, int K, int N, int group,
               const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
               const uint32_t* gsched, const uint8_t* gcnt_ge,
               float* y, void* workspace, size_t workspace_bytes, void* stream);
int grinqh_vmm_main(int T, int K, int N, int group,
                    const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                    const uint32_t* gsched, const uint8_t* gcnt_ge,
                    void* workspace, size_t workspace_bytes, void* stream);
int grinqh_vmm_reduce(int T, int K, int N, float* y,
                      const void* workspace, size_t workspace_bytes, void* stream);

/*
 * grinqh_vmm_thresholds — the threshold assignment made inside the VMM launch (SURVEY.md 8f4:
 * assignment fused into its consumer).  Every warp derives the widths, the union and the (width desc, index asc)
 * list of its 128-row group from x and theta; no assignment kernel runs and no schedule is written.  y is bit-identical
 * to grinqh_assign_thresholds followed by grinqh_vmm.  Arguments as in those two calls.
 */
int grinqh_vmm_thresholds(const void* x_f16, int T, int K, int N, int group, const uint16_t theta[9],
                          const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                          float* y, void* workspace, size_t workspace_bytes, void* stream);

/*
 * grinqh_vmm_rank — the rank assignment of grinqh_assign (PAPER.md:271 top-p partition of the live vector,
 * :61-65; ties to the lower index) made inside the VMM launch.  Every CTA selects the cut keys of x
 * itself (a 5+5+5-bit radix select in shared memory), resolves ties in index order, and builds the lists of the
 * groups it walks; no assignment kernel runs and no schedule is written.  y is bit-identical to grinqh_assign
 * followed by grinqh_vmm.
 *   x_f16   dev  [T, K] fp16        counts HOST [9], sum = K (GRINQH_ERR_MIX otherwise), read during the call
 *   other arguments as in grinqh_vmm.
 */
int grinqh_vmm_rank(const void* x_f16, int T, int K, int N, int group, const uint32_t counts[9],
                    const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                    float* y, void* workspace, size_t workspace_bytes, void* stream);

/*
 * grinqh_vmm_rank_static — grinqh_vmm_rank (same launch, same bits) for callers that cannot allocate: code under
 * CUDA graph capture, serving loops and harnesses that forbid cudaMalloc.  The scratch of the launch (ticket counters
 * + split-K partials, PAPER.md:85 / SURVEY.md 8a4) lives in a file-scope device array of the library instead of a
 * caller-provided workspace; the call makes no cudaMalloc, cudaFree or allocating library call.
 *   limit      the array is GRINQH_STATIC_SCRATCH_BYTES of device memory on every GPU that loads the library, held
 *              until exit; a shape with grinqh_vmm_workspace_bytes(T, K, N) above it returns GRINQH_ERR_STATIC_LIMIT
 *              (nothing is enqueued) — use grinqh_vmm_rank with a workspace there.
 *   sharing    every call on a device uses the same array: calls that overlap on the GPU (two streams, graph
 *              branches without a dependency) RACE; calls ordered on one stream do not.  The tickets are cleared on
 *              `stream` before every launch; stale partials are never read.
 *   arguments  as grinqh_vmm_rank without workspace / workspace_bytes; all pointers dev except counts (HOST).
 * grinqh_static_scratch_bytes returns GRINQH_STATIC_SCRATCH_BYTES as built into the library.
 */
#define GRINQH_STATIC_SCRATCH_BYTES (4u << 20)
size_t grinqh_static_scratch_bytes(void);
int grinqh_vmm_rank_static(const void* x_f16, int T, int K, int N, int group, const uint32_t counts[9],
                           const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                           float* y, void* stream);

/*
 * The paper's own storage granularity ("decomposed into discrete 2-bit segments",
 * :95 b_max in {4, 6, 8}, :442 sixteen 2-bit chunks per uint32): b_max-bit asymmetric group codes (the quantiser of
 * grinqh_pack with 2^b_max - 1 steps) split into b_max / 2 two-bit significance segments.
 *   segs  dev  [b_max/2][K][N/16] uint32: segment 0 is the most significant pair; column n's pair sits at bits
 *              2 (n & 15) + 1 and 2 (n & 15) of word n >> 4.
 * grinqh_pack_seg2: offline, once per weight (scales / zeros as in grinqh_pack).
 * grinqh_vmm_rank_seg2: grinqh_vmm_rank over that store: widths in {0, 2, .., b_max} (counts[w] must be 0 for odd w
 * and for w > b_max: GRINQH_ERR_MIX), a row of width b fetches its first b / 2 segments, reconstruction
 * w_hat = s * (q_b * 2^(b_max - b) + 2^(b_max - b - 1)) + z (no bias at b = b_max).  One token (T = 1),
 * N % 128 == 0 (GRINQH_ERR_SHAPE otherwise); workspace as for grinqh_vmm.
 */
int grinqh_pack_seg2(const void* W_f16, int K, int N, int group, int bmax,
                     uint32_t* segs, void* scales_f16, void* zeros_f16, void* stream);
int grinqh_vmm_rank_seg2(const void* x_f16, int T, int K, int N, int group, int bmax, const uint32_t counts[9],
                         const uint32_t* segs, const void* scales_f16, const void* zeros_f16,
                         float* y, void* workspace, size_t workspace_bytes, void* stream);

/*
 * grinqh_prefill_gemm — the paper's prefill path ("unpacking the weights at full b_max precision and
 * performing dense matrix-matrix multiplication", :182 kernel fusion) in one launch:
 *   Y[M, N] = X[M, K] . W_hat[K, N],  W_hat = s * q + z rounded once to fp16 (exactly what grinqh_unpack writes),
 * fp16 x fp16 products accumulated in fp32 on the tensor cores (tcgen05, accumulators in TMEM), Y rounded to fp16.
 * The planes are unpacked inside the kernel into the shared-memory operand tile: HBM sees 1 byte per weight.
 *   x_f16   dev [M, K] fp16 row-major (any M >= 1; rows beyond M are not read)    y_f16  dev [M, N] fp16 row-major
 *   planes / scales_f16 / zeros_f16  as written by grinqh_pack
 * Needs N % 256 == 0, K % 128 == 0, group == 128 (GRINQH_ERR_SHAPE), 16-byte aligned pointers (GRINQH_ERR_ALIGN) and
 * scales below 128 (weight range per group < 32640: the kernel holds s * 2^9 in fp16).  Enqueued on `stream`; the
 * tensor map for X is encoded on the host during the call.
 */
int grinqh_prefill_gemm(const void* x_f16, int M, int K, int N, int group,
                        const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                        void* y_f16, void* stream);

/*
 * Host-buffer decode call (the end-to-end entry): x comes from HOST memory, the rank assignment and the VMM run in
 * one launch (grinqh_vmm_rank), y ends in HOST memory, all enqueued on `stream`.  x is staged with one
 * cudaMemcpyAsync (every CTA reads all of x for its rank selection).  With a pinned (page-locked) y_host the VMM's
 * second pass writes y straight into host memory; a pageable buffer, or GRINQH_FORCE_COPIES, is staged through y_dev
 * with cudaMemcpyAsync.  The packed weights stay resident on the device.  The caller synchronises the stream before
 * reading y_host.  All arguments are validated before anything is enqueued.
 *   x_host_f16  HOST [T, K] fp16       y_host  HOST [T, N] fp32       counts HOST [9], sum = K
 *   x_dev_f16   dev  [T, K] fp16 staging, y_dev dev [T, N] fp32 staging
 *   vmm_ws      dev  workspace of grinqh_vmm_workspace_bytes(T, K, N) bytes (tickets initialised)
 */
#define GRINQH_FORCE_COPIES 2   /* always stage y through y_dev with cudaMemcpyAsync */
int grinqh_decode_host(const void* x_host_f16, int T, int K, int N, int group,
                       const uint32_t counts[9],
                       const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                       void* x_dev_f16, float* y_dev, void* vmm_ws, size_t vmm_ws_bytes,
                       float* y_host, int flags, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GRINQH_H */
