// vmm_static.cu — grinqh_vmm_rank_static: grinqh_vmm_rank for callers that cannot allocate (code under CUDA graph
// capture, serving loops and harnesses that forbid cudaMalloc).  The launch is the same one (vmm_items.cu: rank select,
// selective plane fetch, deterministic split-K second pass); only the scratch differs: the ticket counters and the
// split-K partials live in a file-scope __device__ array instead of a caller-provided workspace.
//
//   * The array is GRINQH_STATIC_SCRATCH_BYTES (4 MiB) of device memory per GPU that loads the library, held until the
//     process exits.  A shape whose grinqh_vmm_workspace_bytes(T, K, N) is larger is rejected (GRINQH_ERR_STATIC_LIMIT);
//     4 MiB covers every projection of the configs at T <= 4 (largest: 4 x 4096 x 37 partials = 2.4 MB).
//   * No cudaMalloc / cudaFree / allocating library call on this path: cudaGetSymbolAddress once per device, then one
//     memset node for the tickets and the kernel launch per call.
//   * EVERY call on a device shares the one array.  It keeps the previous call's partials (harmless: every partial
//     that is read was written by the same launch) and tickets (must be zero at launch: cleared on the stream before
//     every launch, so an aborted launch cannot poison the next one).  Two calls that overlap on the GPU — different
//     streams, or graph branches without a dependency — RACE on it: serialise them, or use grinqh_vmm_rank with one
//     workspace per stream.
#include <mutex>

#include "vmm_args.cuh"

namespace gq {

// (the name below is a host-side stand-in in host code, not a device address: host code takes the address with
// cudaGetSymbolAddress, device code could name the array directly)
static __device__ __align__(256) unsigned char g_static_scratch[GRINQH_STATIC_SCRATCH_BYTES];

// device address of the array on the CURRENT device, looked up once per device
static int static_scratch_ptr(void** out) {
    static void* ptrs[64];
    static std::mutex mu;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return GRINQH_ERR_CUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (ptrs[dev] == nullptr) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || p == nullptr) {
            (void)cudaGetLastError();
            return GRINQH_ERR_CUDA;
        }
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return GRINQH_OK;
}

}  // namespace gq

extern "C" size_t grinqh_static_scratch_bytes(void) { return (size_t)GRINQH_STATIC_SCRATCH_BYTES; }

extern "C" int grinqh_vmm_rank_static(const void* x_f16, int T, int K, int N, int group, const uint32_t counts[9],
                                      const uint32_t* planes, const void* scales_f16, const void* zeros_f16, float* y,
                                      void* stream) {
    if (!y || !x_f16 || !counts || !planes || !scales_f16 || !zeros_f16) return GRINQH_ERR_NULL;
    const size_t need = grinqh_vmm_workspace_bytes(T, K, N);  // 0: the shape itself is unsupported
    if (need == 0) return GRINQH_ERR_SHAPE;
    if (group != GQ_G) return GRINQH_ERR_SHAPE;
    if (((uintptr_t)y | (uintptr_t)x_f16 | (uintptr_t)planes | (uintptr_t)scales_f16 | (uintptr_t)zeros_f16) & 15)
        return GRINQH_ERR_ALIGN;
    if (need > (size_t)GRINQH_STATIC_SCRATCH_BYTES) return GRINQH_ERR_STATIC_LIMIT;
    unsigned long long total = 0;
    for (int w = 0; w < 9; ++w) total += counts[w];
    if (total != (unsigned long long)K) return GRINQH_ERR_MIX;

    void* ws = nullptr;
    const int rc = gq::static_scratch_ptr(&ws);
    if (rc != GRINQH_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the tickets of this shape's column tiles start at zero, whatever the previous call on the array left behind
    const size_t tiles = (size_t)((N + 1023) / 1024);
    if (cudaMemsetAsync(ws, 0, (tiles * sizeof(int) + 255) & ~(size_t)255, st) != cudaSuccess) return GRINQH_ERR_CUDA;
    gq::VmmArgs a{T, K, N, 1, gq::MODE_RANK, 8, planes, scales_f16, zeros_f16, nullptr, nullptr, (const uint16_t*)x_f16,
                  gq::cuts_from_counts(counts), ws, y, st};
    return gq::launch_vmm_items(a);
}
