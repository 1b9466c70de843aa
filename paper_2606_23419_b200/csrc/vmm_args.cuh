// vmm_args.cuh — what the VMM's C ABI (vmm.cu) hands to the two kernel families behind it:
//   vmm_items.cu   the item kernel: a warp owns whole (group, sub-chunk) items; fewer, fatter warps — the faster one for
//                  the 1-bit plane store at every shape measured, and the one grinqh_vmm / _rank / _thresholds launch;
//   vmm_kernel.cuh the stream kernel: slot-striped row stream with per-warp lists — carries the 2-bit-segment store
//                  (grinqh_vmm_rank_seg2) and the cp.async.bulk A/B (GRINQH_STREAM=1 routes the plane store to it too).
#pragma once
#include "common.cuh"
#include "select.cuh"

namespace gq {

constexpr size_t TICKET_BYTES = 16384;  // head of the workspace: one int per column tile, zero between launches

enum { MODE_SCHED = 0, MODE_THR = 1, MODE_RANK = 2 };

struct VmmArgs {
    int T, K, N, fused, mode;
    int bmax;  // 8 for the 1-bit plane store; 4 / 6 / 8 for the 2-bit-segment store
    const uint32_t* planes;
    const void *scales, *zeros;
    const uint32_t* gsched;
    const uint8_t* gcnt_ge;
    const uint16_t* xraw;
    CutParams cp;
    void* workspace;
    float* y;
    cudaStream_t st;
};

int num_sms();                              // of the current device
int items_sx(int T, int K, int N);          // split-K partials per column tile of the item kernel's plan
int launch_vmm_items(const VmmArgs& a);     // vmm_items.cu
int stream_sx(int T, int K, int N);         // ... of the stream kernel's plan
int launch_vmm_stream(const VmmArgs& a);    // vmm.cu / vmm_multi.cu

}  // namespace gq
