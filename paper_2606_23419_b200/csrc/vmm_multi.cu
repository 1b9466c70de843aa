// vmm_multi.cu — instantiations of the VMM kernel for 2..4 tokens (a translation unit of its own: build time).
#include "vmm_kernel.cuh"

namespace gq {

template <int T, int MODE>
static int launch_a16(const VmmArgs& a, const VmmPlan& pl) {
    return (a.N % 128 == 0) ? launch_impl<T, 8, true, MODE>(a, pl) : launch_impl<T, 8, false, MODE>(a, pl);
}

template <int MODE>
static int launch_t(const VmmArgs& a, const VmmPlan& pl) {
    switch (a.T) {
        case 2: return launch_a16<2, MODE>(a, pl);
        case 3: return launch_a16<3, MODE>(a, pl);
        default: return launch_a16<4, MODE>(a, pl);
    }
}

int launch_vmm_multi(const VmmArgs& a, const VmmPlan& pl) {
    switch (a.mode) {
        case MODE_SCHED: return launch_t<MODE_SCHED>(a, pl);
        case MODE_THR: return launch_t<MODE_THR>(a, pl);
        default: return launch_t<MODE_RANK>(a, pl);
    }
}

}  // namespace gq
