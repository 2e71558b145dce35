// inst_relift.cu -- instantiates the re-lift rollout kernel (rollout_relift.cuh) for padded physical dims 4, 8, 16.
#include "rollout_relift.cuh"
using namespace mpmi;

KernFn mpmi_pick_relift(int n, int mode) {
    const bool t = mode == MODE_TICK;
    if (n <= 4) return t ? rollout_relift_kernel<4, MODE_TICK> : rollout_relift_kernel<4, MODE_BATCH>;
    if (n <= 8) return t ? rollout_relift_kernel<8, MODE_TICK> : rollout_relift_kernel<8, MODE_BATCH>;
    if (n <= 16) return t ? rollout_relift_kernel<16, MODE_TICK> : rollout_relift_kernel<16, MODE_BATCH>;
    return nullptr;
}
