// inst_tc.cu -- instantiates the tensor-core (tcgen05) rollout kernel for one MPMI_MODE, with and without noise.
#include "rollout_tc.cuh"
#ifndef MPMI_MODE
#error "compile with -DMPMI_MODE=0|1"
#endif
using namespace mpmi;
#if MPMI_MODE == 0
KernFn mpmi_pick_tc_tick(int *smem, int *threads, int noise) {
    *smem = kTcSmemBytes; *threads = kTcThreads;
    return noise ? rollout_tc_kernel<MODE_TICK, true> : rollout_tc_kernel<MODE_TICK, false>;
}
#else
KernFn mpmi_pick_tc_batch(int *smem, int *threads, int noise) {
    *smem = kTcSmemBytes; *threads = kTcThreads;
    return noise ? rollout_tc_kernel<MODE_BATCH, true> : rollout_tc_kernel<MODE_BATCH, false>;
}
#endif
