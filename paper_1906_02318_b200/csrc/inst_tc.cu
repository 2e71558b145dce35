// inst_tc.cu -- instantiates the tensor-core (tcgen05) rollout kernel for one MPMI_MODE: D = 128 and D = 32, with and without noise.
#include "rollout_tc.cuh"
#ifndef MPMI_MODE
#error "compile with -DMPMI_MODE=0|1"
#endif
using namespace mpmi;
template <int D, int MODE>
static KernFn pick(int *smem, int *threads, int *ctas_per_sm, int noise) {
    *smem = TcGeom<D>::kSmemBytes; *threads = TcGeom<D>::kThreads; *ctas_per_sm = TcGeom<D>::kCtasPerSm;
    return noise ? rollout_tc_kernel<D, MODE, true> : rollout_tc_kernel<D, MODE, false>;
}
#if MPMI_MODE == 0
KernFn mpmi_pick_tc_tick(int D, int *smem, int *threads, int *ctas_per_sm, int noise) {
    return D == 128 ? pick<128, MODE_TICK>(smem, threads, ctas_per_sm, noise) : D == 32 ? pick<32, MODE_TICK>(smem, threads, ctas_per_sm, noise) : nullptr;
}
#else
KernFn mpmi_pick_tc_batch(int D, int *smem, int *threads, int *ctas_per_sm, int noise) {
    return D == 128 ? pick<128, MODE_BATCH>(smem, threads, ctas_per_sm, noise) : D == 32 ? pick<32, MODE_BATCH>(smem, threads, ctas_per_sm, noise) : nullptr;
}
#endif
