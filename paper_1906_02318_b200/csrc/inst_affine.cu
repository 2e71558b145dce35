// inst_affine.cu -- instantiates the affine-in-u fast path (rollout_affine.cuh).
#include "rollout_affine.cuh"
using namespace mpmi;

KernFn mpmi_pick_affine_base(int D) {
    switch (D) {
        case 8: return affine_base_kernel<8>;
        case 16: return affine_base_kernel<16>;
        case 32: return affine_base_kernel<32>;
        case 64: return affine_base_kernel<64>;
        case 128: return affine_base_kernel<128>;
    }
    return nullptr;
}
KernFn mpmi_pick_affine(int np, int mode) {
    const bool t = mode == MODE_TICK;
    if (np == 4) return t ? rollout_affine_kernel<4, MODE_TICK> : rollout_affine_kernel<4, MODE_BATCH>;
    if (np == 8) return t ? rollout_affine_kernel<8, MODE_TICK> : rollout_affine_kernel<8, MODE_BATCH>;
    if (np == 16) return t ? rollout_affine_kernel<16, MODE_TICK> : rollout_affine_kernel<16, MODE_BATCH>;
    return nullptr;
}
