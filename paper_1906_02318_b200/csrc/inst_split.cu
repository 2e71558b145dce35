// inst_split.cu -- instantiates the row-split second-pass kernels (rollout_split.cuh) for one MPMI_NOISE.
#include "rollout_split.cuh"
using namespace mpmi;
#ifndef MPMI_NOISE
#define MPMI_NOISE 0
#endif
#if MPMI_NOISE
#define FN mpmi_pick_splitn_32
#else
#define FN mpmi_pick_split_32
#endif

template <int RS>
static KernFn pick_m(int M) {
    switch (M) {
        case 1: return rollout_split_kernel<32, 1, RS, (MPMI_NOISE != 0)>;
        case 2: return rollout_split_kernel<32, 2, RS, (MPMI_NOISE != 0)>;
        case 3: return rollout_split_kernel<32, 3, RS, (MPMI_NOISE != 0)>;
        case 4: return rollout_split_kernel<32, 4, RS, (MPMI_NOISE != 0)>;
    }
    return nullptr;
}
// rs = lanes per candidate pair (2, 4, 8 or 16)
KernFn FN(int M, int rs) { return rs == 2 ? pick_m<2>(M) : rs == 4 ? pick_m<4>(M) : rs == 8 ? pick_m<8>(M) : rs == 16 ? pick_m<16>(M) : nullptr; }
