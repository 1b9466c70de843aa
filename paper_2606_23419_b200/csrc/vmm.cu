// vmm.cu — C ABI of the VMM (grinqh_vmm, grinqh_vmm_rank, grinqh_vmm_thresholds, the two-launch form, the 2-bit-segment
// form), the routing between the two kernel families (vmm_args.cuh), the stream kernel's shape-only plan and its
// one-token instantiations (vmm_kernel.cuh).
#include <algorithm>
#include <cstdlib>

#include "vmm_kernel.cuh"

namespace gq {

__global__ void __launch_bounds__(256)
vmm_reduce_kernel(const float* __restrict__ part, int S, int T, int N, float* __restrict__ y) {
    const int t = blockIdx.y;
    const int n = (blockIdx.x * 256 + threadIdx.x) * 4;
    if (n >= N) return;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int s = 0; s < S; ++s) {
        const float4 v = *reinterpret_cast<const float4*>(part + ((size_t)s * T + t) * N + n);
        a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
    }
    *reinterpret_cast<float4*>(y + (size_t)t * N + n) = a;
}

int num_sms() {
    static int cached[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    if (cached[dev] == 0) {
        int n = 0;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cached[dev] = n;
    }
    return cached[dev];
}

// Shape-only plan (the workspace size depends on it): one CTA per SM, as many split-K slices as fit.
static inline VmmPlan vmm_plan(int T, int K, int N) {
    VmmPlan pl;
    pl.col_tiles = (N + TILE_COLS - 1) / TILE_COLS;
    int sx = num_sms() / pl.col_tiles;
    const int cap = K / 64 > 0 ? K / 64 : 1;
    if (sx > cap) sx = cap;
    if (sx < 1) sx = 1;
    // Among the few largest split factors take the one sharing the largest factor with the number of groups: the CTAs'
    // slot ranges then line up with group boundaries more often (fewer warps straddle two groups and pay two sets of
    // scale/zero chunks).  Measured (profiles/r02_kernels.md): 4096 x 4096 36 slices 13.1 us against 14.6 us with 37;
    // 14336 x 4096 35 slices 19.1 us against 20.7 us with 37.
    {
        auto gcd = [](int a, int b) {
            while (b) {
                const int t = a % b;
                a = b;
                b = t;
            }
            return a;
        };
        const int groups = K / GQ_G;
        int best = sx, best_g = gcd(groups, sx);
        for (int c = sx - 1; c >= 1 && c * 100 >= sx * 94; --c)
            if (gcd(groups, c) > best_g) {
                best = c;
                best_g = gcd(groups, c);
            }
        sx = best;
    }
    if (const char* f = getenv("GRINQH_SX")) {  // measurement override
        const int v = atoi(f);
        if (v >= 1 && v <= sx) sx = v;
    }
    pl.Sx = sx;
    pl.vw = 8;
    if (T == 1) {
        pl.vw = 16;  // measured: 16 warps win at every shape (4 and 8 leave the schedulers without enough warps)
        if (const char* f = getenv("GRINQH_VW")) {  // measurement override
            const int v = atoi(f);
            if (v == 4 || v == 8 || v == 16) pl.vw = v;
            if (pl.vw == 4 && K > 16384) pl.vw = 8;
        }
    }
    return pl;
}

// Measurement switch: GRINQH_BULK=1 selects the cp.async.bulk (TMA, SASS UBLKCP) + mbarrier form of the row copies.
// It is correct and twice as slow as the cp.async (LDGSTS) form on B200 — a 128-byte bulk copy costs the TMA unit
// ~24 cycles per SM (profiles/r02_bulk_ab.md) — so the default is LDGSTS.
static bool use_bulk() {
    static int v = -1;
    if (v < 0) {
        const char* f = getenv("GRINQH_BULK");
        v = (f && atoi(f) == 1) ? 1 : 0;
    }
    return v != 0;
}

template <int VW, int MODE>
static int launch_a16(const VmmArgs& a, const VmmPlan& pl) {
    return use_bulk() ? launch_impl<1, VW, true, MODE, true>(a, pl) : launch_impl<1, VW, true, MODE, false>(a, pl);
}

template <int MODE>
static int launch_t1(const VmmArgs& a, const VmmPlan& pl) {
    if (a.N % 128 != 0) return launch_impl<1, 8, false, MODE>(a, pl);  // ragged rows: 4-byte copies, 8 warps only
    switch (pl.vw) {
        case 4: return launch_a16<4, MODE>(a, pl);
        case 16: return launch_a16<16, MODE>(a, pl);
        default: return launch_a16<8, MODE>(a, pl);
    }
}

int stream_sx(int T, int K, int N) { return vmm_plan(T, K, N).Sx; }

int launch_vmm_stream(const VmmArgs& a) {
    const VmmPlan pl = vmm_plan(a.T, a.K, a.N);
    if (a.T > 1) return launch_vmm_multi(a, pl);
    switch (a.mode) {
        case MODE_SCHED: return launch_t1<MODE_SCHED>(a, pl);
        case MODE_THR: return launch_t1<MODE_THR>(a, pl);
        default: return launch_t1<MODE_RANK>(a, pl);
    }
}

// The 1-bit plane store goes to the item kernel (vmm_items.cu): at every shape of the configs it is the faster of the
// two (profiles/r02_kernels.md).  GRINQH_STREAM=1 (read once) routes it to the stream kernel instead — the A/B switch
// of that table, and what GRINQH_BULK=1 needs.
static bool use_stream() {
    static int v = -1;
    if (v < 0) {
        const char* f = getenv("GRINQH_STREAM");
        v = ((f && atoi(f) == 1) || use_bulk()) ? 1 : 0;
    }
    return v != 0;
}

static int launch_vmm(const VmmArgs& a) { return use_stream() ? launch_vmm_stream(a) : launch_vmm_items(a); }

// split-K partials per column tile of the launch (the two-launch form reads it back)
static int active_sx(int T, int K, int N) { return use_stream() ? stream_sx(T, K, N) : items_sx(T, K, N); }

static int check_vmm_args(int T, int K, int N, int group) {
    if (group != GQ_G || T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32 || K > GQ_MAX_K)
        return GRINQH_ERR_SHAPE;
    if ((size_t)((N + TILE_COLS - 1) / TILE_COLS) * sizeof(int) > TICKET_BYTES) return GRINQH_ERR_SHAPE;
    return GRINQH_OK;
}

static int check_vmm_ptrs(int T, int K, int N, int group, const void* planes, const void* scales, const void* zeros,
                          const void* a, const void* b, const void* workspace, size_t workspace_bytes) {
    if (!planes || !scales || !zeros || !a || !b || !workspace) return GRINQH_ERR_NULL;
    const int rc = check_vmm_args(T, K, N, group);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)planes | (uintptr_t)scales | (uintptr_t)zeros | (uintptr_t)a | (uintptr_t)b |
         (uintptr_t)workspace) & 15)
        return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    return GRINQH_OK;
}

}  // namespace gq

extern "C" size_t grinqh_vmm_workspace_bytes(int T, int K, int N) {
    if (gq::check_vmm_args(T, K, N, GQ_G) != GRINQH_OK) return 0;
    // one workspace serves every entry point: the largest split-K factor of the plans behind them
    int sx = gq::stream_sx(T, K, N);
    sx = std::max(sx, gq::items_sx(T, K, N));
    return gq::TICKET_BYTES + (size_t)sx * T * N * sizeof(float);
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
    gq::VmmArgs a{T, K, N, 1, gq::MODE_SCHED, 8, planes, scales_f16, zeros_f16, gsched, gcnt_ge, nullptr, gq::CutParams{},
                  workspace, y, (cudaStream_t)stream};
    return gq::launch_vmm(a);
}

extern "C" int grinqh_vmm_main(int T, int K, int N, int group, const uint32_t* planes, const void* scales_f16,
                               const void* zeros_f16, const uint32_t* gsched, const uint8_t* gcnt_ge,
                               void* workspace, size_t workspace_bytes, void* stream) {
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, gsched, gcnt_ge, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    gq::VmmArgs a{T, K, N, 0, gq::MODE_SCHED, 8, planes, scales_f16, zeros_f16, gsched, gcnt_ge, nullptr, gq::CutParams{},
                  workspace, nullptr, (cudaStream_t)stream};
    return gq::launch_vmm(a);
}

extern "C" int grinqh_vmm_reduce(int T, int K, int N, float* y, const void* workspace, size_t workspace_bytes,
                                 void* stream) {
    if (!y || !workspace) return GRINQH_ERR_NULL;
    int rc = gq::check_vmm_args(T, K, N, GQ_G);
    if (rc != GRINQH_OK) return rc;
    if (((uintptr_t)y | (uintptr_t)workspace) & 15) return GRINQH_ERR_ALIGN;
    if (workspace_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    dim3 grid((N + 4 * 256 - 1) / (4 * 256), T);
    gq::vmm_reduce_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(
        (const float*)((const char*)workspace + gq::TICKET_BYTES), gq::active_sx(T, K, N), T, N, y);
    return cudaGetLastError() == cudaSuccess ? GRINQH_OK : GRINQH_ERR_CUDA;
}

// SURVEY.md 8f4 (assignment fused into the consumer): the paper's threshold assignment made inside
// the VMM launch — every warp derives its groups' widths and lists from x and theta; one launch per projection and
// no assignment kernel.  y equals grinqh_assign_thresholds + grinqh_vmm bit for bit.
extern "C" int grinqh_vmm_thresholds(const void* x_f16, int T, int K, int N, int group, const uint16_t theta[9],
                                     const uint32_t* planes, const void* scales_f16, const void* zeros_f16, float* y,
                                     void* workspace, size_t workspace_bytes, void* stream) {
    if (!y || !x_f16 || !theta) return GRINQH_ERR_NULL;
    if (((uintptr_t)y | (uintptr_t)x_f16) & 15) return GRINQH_ERR_ALIGN;
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, x_f16, x_f16, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    for (int w = 1; w <= 8; ++w)
        if (theta[w] > 0x8000 || (w > 1 && theta[w] < theta[w - 1])) return GRINQH_ERR_MIX;
    gq::VmmArgs a{T, K, N, 1, gq::MODE_THR, 8, planes, scales_f16, zeros_f16, nullptr, nullptr, (const uint16_t*)x_f16,
                  gq::cuts_from_thetas(theta), workspace, y, (cudaStream_t)stream};
    return gq::launch_vmm(a);
}

// The north star's rank assignment (PAPER.md:271 top-p partition of the live vector; readings #2-#4) made
// inside the VMM launch: every CTA selects the cut keys of x itself.  y equals grinqh_assign + grinqh_vmm bit for bit.
extern "C" int grinqh_vmm_rank(const void* x_f16, int T, int K, int N, int group, const uint32_t counts[9],
                               const uint32_t* planes, const void* scales_f16, const void* zeros_f16, float* y,
                               void* workspace, size_t workspace_bytes, void* stream) {
    if (!y || !x_f16 || !counts) return GRINQH_ERR_NULL;
    if (((uintptr_t)y | (uintptr_t)x_f16) & 15) return GRINQH_ERR_ALIGN;
    const int rc = gq::check_vmm_ptrs(T, K, N, group, planes, scales_f16, zeros_f16, x_f16, x_f16, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    gq::VmmArgs a{T, K, N, 1, gq::MODE_RANK, 8, planes, scales_f16, zeros_f16, nullptr, nullptr, (const uint16_t*)x_f16,
                  gq::cuts_from_counts(counts), workspace, y, (cudaStream_t)stream};
    return gq::launch_vmm(a);
}

// the same launch over the paper's own store — b_max-bit codes in 2-bit significance segments
// (grinqh_pack_seg2), widths in {0, 2, .., b_max}.  One token, N % 128 == 0.
extern "C" int grinqh_vmm_rank_seg2(const void* x_f16, int T, int K, int N, int group, int bmax, const uint32_t counts[9],
                                    const uint32_t* segs, const void* scales_f16, const void* zeros_f16, float* y,
                                    void* workspace, size_t workspace_bytes, void* stream) {
    if (!y || !x_f16 || !counts) return GRINQH_ERR_NULL;
    if (((uintptr_t)y | (uintptr_t)x_f16) & 15) return GRINQH_ERR_ALIGN;
    if (T != 1 || N % 128 || (bmax != 4 && bmax != 6 && bmax != 8)) return GRINQH_ERR_SHAPE;
    const int rc = gq::check_vmm_ptrs(T, K, N, group, segs, scales_f16, zeros_f16, x_f16, x_f16, workspace,
                                      workspace_bytes);
    if (rc != GRINQH_OK) return rc;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) {
        total += counts[w];
        if (counts[w] && ((w & 1) || w > bmax)) return GRINQH_ERR_MIX;  // widths are 0, 2, .., b_max
    }
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    gq::VmmArgs a{T, K, N, 1, gq::MODE_RANK, bmax, segs, scales_f16, zeros_f16, nullptr, nullptr, (const uint16_t*)x_f16,
                  gq::cuts_from_counts(counts), workspace, y, (cudaStream_t)stream};
    const gq::VmmPlan pl = gq::vmm_plan(T, K, N);
    return gq::launch_impl<1, 16, true, gq::MODE_RANK, false, true>(a, pl);
}
