// api.cu — host-side entry points of the C ABI that launch no kernel of their own.
#include <math.h>

#include <algorithm>
#include <functional>
#include <vector>

#include "common.cuh"

extern "C" const char* grinqh_status_string(int status) {
    switch (status) {
        case GRINQH_OK: return "ok";
        case GRINQH_ERR_NULL: return "null pointer";
        case GRINQH_ERR_SHAPE: return "unsupported shape (need K % 128 == 0, N % 32 == 0, 1 <= T <= 4, group == 128, K <= 32768 for assign)";
        case GRINQH_ERR_ALIGN: return "pointer not 16-byte aligned";
        case GRINQH_ERR_MIX: return "level mix does not sum to K (or fractions do not sum to 1)";
        case GRINQH_ERR_WORKSPACE: return "workspace too small";
        case GRINQH_ERR_CUDA: return "CUDA launch failed";
        case GRINQH_ERR_STATIC_LIMIT:
            return "shape needs more scratch than the library's static array (GRINQH_STATIC_SCRATCH_BYTES); use the "
                   "workspace form";
        default: return "unknown status";
    }
}

extern "C" int grinqh_version(void) { return 300; /* 0.3.0: grinqh_vmm_rank, slot-striped VMM, histogram select */ }

// PAPER.md:262-266 (Eq. 1): precision distribution P -> integer row counts; reading #3.
extern "C" int grinqh_mix_to_counts(int K, const double frac[9], uint32_t counts[9]) {
    if (!frac || !counts) return GRINQH_ERR_NULL;
    if (K <= 0) return GRINQH_ERR_SHAPE;
    double sum = 0.0;
    for (int w = 0; w < 9; ++w) {
        if (!(frac[w] >= 0.0)) return GRINQH_ERR_MIX;
        sum += frac[w];
    }
    if (fabs(sum - 1.0) > 1e-6) return GRINQH_ERR_MIX;
    long long C[10];
    C[9] = 0;
    double F = 0.0;
    for (int w = 8; w >= 1; --w) {
        F += frac[w];
        long long c = (long long)floor(F * (double)K + 0.5);
        if (c < C[w + 1]) c = C[w + 1];
        if (c > K) c = K;
        C[w] = c;
    }
    C[0] = K;
    for (int w = 0; w < 9; ++w) counts[w] = (uint32_t)(C[w] - C[w + 1]);
    return GRINQH_OK;
}

// PAPER.md:69-73, :271-273 (Eq. 2): thresholds = per-vector level-separating magnitudes under the rank partition,
// averaged over the calibration vectors.  Offline host helper (like grinqh_mix_to_counts): fp64 mean of the C_w-th
// largest |x| of every vector, rounded to fp32 then fp16 (RN-even); C_w == 0 -> 0x8000 (width w unreachable).
extern "C" int grinqh_calibrate_thresholds(const void* x_host_f16, int S, int K, const uint32_t counts[9],
                                           uint16_t theta[9]) {
    if (!x_host_f16 || !counts || !theta) return GRINQH_ERR_NULL;
    if (S < 1 || K <= 0) return GRINQH_ERR_SHAPE;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    long long C[10];
    C[9] = 0;
    for (int w = 8; w >= 0; --w) C[w] = C[w + 1] + counts[w];
    const uint16_t* x = (const uint16_t*)x_host_f16;
    std::vector<uint16_t> m((size_t)K);
    double sum[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int s = 0; s < S; ++s) {
        for (int k = 0; k < K; ++k) m[k] = x[(size_t)s * K + k] & 0x7FFFu;
        for (int w = 1; w <= 8; ++w) {
            if (C[w] == 0) continue;
            std::nth_element(m.begin(), m.begin() + (C[w] - 1), m.end(), std::greater<uint16_t>());
            __half_raw r;
            r.x = m[C[w] - 1];
            sum[w] += (double)__half2float(__half(r));
        }
    }
    theta[0] = 0;
    for (int w = 1; w <= 8; ++w) {
        if (C[w] == 0) {
            theta[w] = 0x8000;
        } else {
            const __half_raw r = __float2half_rn((float)(sum[w] / S));
            theta[w] = r.x;
        }
    }
    return GRINQH_OK;
}

namespace gq {
// x from pinned host memory to its device staging buffer: ONE small CTA reads the few KB over PCIe (host-mapped
// access), so that the 148 CTAs of the VMM read x from L2.  A kernel, not a copy node: it chains to its neighbours with
// programmatic dependent launch like every other launch of the step.
__global__ void __launch_bounds__(512) stage_x_kernel(const uint4* __restrict__ src, uint4* __restrict__ dst, int n16) {
    pdl_launch_dependents();
    pdl_wait();
    for (int i = threadIdx.x; i < n16; i += 512) dst[i] = src[i];
}
}  // namespace gq

extern "C" int grinqh_decode_host(const void* x_host_f16, int T, int K, int N, int group, const uint32_t counts[9],
                                  const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                                  void* x_dev_f16, float* y_dev, void* vmm_ws, size_t vmm_ws_bytes, float* y_host,
                                  int flags, void* stream) {
    // every argument is checked before the first enqueue: on error nothing has been enqueued
    if (!x_host_f16 || !x_dev_f16 || !y_dev || !y_host || !counts || !planes || !scales_f16 || !zeros_f16 || !vmm_ws)
        return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32 || group != GQ_G || K > GQ_MAX_K)
        return GRINQH_ERR_SHAPE;
    if (((uintptr_t)x_dev_f16 | (uintptr_t)y_dev | (uintptr_t)planes | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16 |
         (uintptr_t)vmm_ws) & 15)
        return GRINQH_ERR_ALIGN;
    const size_t need = grinqh_vmm_workspace_bytes(T, K, N);
    if (need == 0) return GRINQH_ERR_SHAPE;
    if (vmm_ws_bytes < need) return GRINQH_ERR_WORKSPACE;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;
    cudaStream_t st = (cudaStream_t)stream;
    // x: one small copy to the device (every CTA of the VMM reads all of x for its rank selection: that traffic
    // belongs in L2, not on PCIe) — by a one-CTA kernel reading the pinned buffer directly, else by cudaMemcpyAsync.  y: with a pinned (page-locked) host buffer the VMM's second pass writes the result
    // straight into host memory — no copy node; a pageable buffer (or GRINQH_FORCE_COPIES) is staged through y_dev.
    float* yv = nullptr;
    if (!(flags & GRINQH_FORCE_COPIES)) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, y_host) == cudaSuccess) {
            if (a.type == cudaMemoryTypeHost && a.devicePointer && !((uintptr_t)a.devicePointer & 15))
                yv = (float*)a.devicePointer;
        } else {
            (void)cudaGetLastError();
        }
    }
    const void* xv = nullptr;  // device view of a pinned x_host
    if (!(flags & GRINQH_FORCE_COPIES)) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, x_host_f16) == cudaSuccess) {
            if (a.type == cudaMemoryTypeHost && a.devicePointer && !((uintptr_t)a.devicePointer & 15)) xv = a.devicePointer;
        } else {
            (void)cudaGetLastError();
        }
    }
    if (xv) {
        if (gq::launch_pdl(gq::stage_x_kernel, dim3(1), dim3(512), 0, st, (const uint4*)xv, (uint4*)x_dev_f16,
                           T * K / 8) != cudaSuccess)
            return GRINQH_ERR_CUDA;
    } else if (cudaMemcpyAsync(x_dev_f16, x_host_f16, (size_t)T * K * 2, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        return GRINQH_ERR_CUDA;
    }
    const int rc = grinqh_vmm_rank(x_dev_f16, T, K, N, group, counts, planes, scales_f16, zeros_f16, yv ? yv : y_dev,
                                   vmm_ws, vmm_ws_bytes, stream);
    if (rc != GRINQH_OK) return rc;
    if (!yv && cudaMemcpyAsync(y_host, y_dev, (size_t)T * N * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return GRINQH_ERR_CUDA;
    return GRINQH_OK;
}
