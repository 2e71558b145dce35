// inst_lat.cu -- instantiates the latency-oriented tick kernels (rollout_lat.cuh) for one MPMI_D.
#include "rollout_lat.cuh"
#ifndef MPMI_D
#error "compile with -DMPMI_D=8|16|32"
#endif
using namespace mpmi;
#define FN(D) mpmi_pick_lat_##D
#define FN2(D) FN(D)

template <int R>
static KernFn pick_m(int M) {
    switch (M) {
        case 1: return rollout_lat_kernel<MPMI_D, 1, R>;
        case 2: return rollout_lat_kernel<MPMI_D, 2, R>;
        case 3: return rollout_lat_kernel<MPMI_D, 3, R>;
        case 4: return rollout_lat_kernel<MPMI_D, 4, R>;
    }
    return nullptr;
}
KernFn FN2(MPMI_D)(int M, int R) { return R == 2 ? pick_m<2>(M) : R == 4 ? pick_m<4>(M) : nullptr; }
