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
        default: return "unknown status";
    }
}

extern "C" int grinqh_version(void) { return 200; /* 0.2.0: gsched schedule, fused second pass, threshold assignment */ }

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

extern "C" int grinqh_decode_host(const void* x_host_f16, int T, int K, int N, int group, const uint32_t counts[9],
                                  const uint32_t* planes, const void* scales_f16, const void* zeros_f16,
                                  void* x_dev_f16, uint8_t* bits, uint8_t* bits_union, int32_t* rows,
                                  int32_t* cnt_ge, uint8_t* grows, uint8_t* gcnt_ge, uint32_t* gsched,
                                  void* assign_ws, size_t assign_ws_bytes, float* y_dev, void* vmm_ws, size_t vmm_ws_bytes,
                                  float* y_host, int flags, void* stream) {
    if (!x_host_f16 || !x_dev_f16 || !y_dev || !y_host || !gsched) return GRINQH_ERR_NULL;
    if (T < 1 || T > GRINQH_MAX_T || K <= 0 || N <= 0 || K % GQ_G || N % 32 || group != GQ_G || K > GQ_MAX_K)
        return GRINQH_ERR_SHAPE;
    if (vmm_ws_bytes < grinqh_vmm_workspace_bytes(T, K, N)) return GRINQH_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = GRINQH_OK;
    // Pinned (page-locked) host buffers are visible to the device under unified addressing: the assignment kernel
    // then reads x straight from host memory (8-57 KB, once) and the VMM's second pass writes y straight into it —
    // no copy nodes, no staging.  Pageable buffers (or GRINQH_FORCE_COPIES) go through cudaMemcpyAsync + staging.
    auto device_view = [&](const void* host) -> void* {
        if (flags & GRINQH_FORCE_COPIES) return nullptr;
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, host) != cudaSuccess) {
            (void)cudaGetLastError();
            return nullptr;
        }
        return (a.type == cudaMemoryTypeHost && a.devicePointer && !((uintptr_t)a.devicePointer & 15)) ? a.devicePointer
                                                                                                     : nullptr;
    };
    if (!(flags & GRINQH_REUSE_ASSIGNMENT)) {
        const void* xv = device_view(x_host_f16);
        if (!xv) {
            if (cudaMemcpyAsync(x_dev_f16, x_host_f16, (size_t)T * K * 2, cudaMemcpyHostToDevice, st) != cudaSuccess)
                return GRINQH_ERR_CUDA;
            xv = x_dev_f16;
        }
        rc = grinqh_assign(xv, T, K, counts, bits, bits_union, rows, cnt_ge, grows, gcnt_ge, gsched, assign_ws,
                           assign_ws_bytes, stream);
        if (rc != GRINQH_OK) return rc;
    }
    float* yv = (float*)device_view(y_host);
    rc = grinqh_vmm(T, K, N, group, planes, scales_f16, zeros_f16, gsched, gcnt_ge, yv ? yv : y_dev, vmm_ws,
                    vmm_ws_bytes, stream);
    if (rc != GRINQH_OK) return rc;
    if (!yv && cudaMemcpyAsync(y_host, y_dev, (size_t)T * N * 4, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return GRINQH_ERR_CUDA;
    return GRINQH_OK;
}
