// inst_tc.cu -- instantiates the tensor-core (tcgen05) rollout kernel for one MPMI_MODE.
#include "rollout_tc.cuh"
#ifndef MPMI_MODE
#error "compile with -DMPMI_MODE=0|1"
#endif
using namespace mpmi;
#if MPMI_MODE == 0
KernFn mpmi_pick_tc_tick(int *smem, int *threads) {
    *smem = kTcSmemBytes; *threads = kTcThreads;
    return rollout_tc_kernel<MODE_TICK>;
}
#else
KernFn mpmi_pick_tc_batch(int *smem, int *threads) {
    *smem = kTcSmemBytes; *threads = kTcThreads;
    return rollout_tc_kernel<MODE_BATCH>;
}
#endif
