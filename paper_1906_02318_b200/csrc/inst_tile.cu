// inst_tile.cu -- instantiates the CTA-tile kernels for one (MPMI_D, MPMI_MODE); see inst_reg.cu.
#include "rollout_tile.cuh"
#ifndef MPMI_D
#error "compile with -DMPMI_D=64|128 -DMPMI_MODE=0|1"
#endif
using namespace mpmi;
#ifndef MPMI_NOISE
#define MPMI_NOISE 0
#endif
#if MPMI_MODE == 0 && !MPMI_NOISE
#define FN(D) mpmi_pick_tile_##D##_tick
#elif !MPMI_NOISE
#define FN(D) mpmi_pick_tile_##D##_batch
#elif MPMI_MODE == 0
#define FN(D) mpmi_pick_tilen_##D##_tick
#else
#define FN(D) mpmi_pick_tilen_##D##_batch
#endif
#define FN2(D) FN(D)

KernFn FN2(MPMI_D)(int M, int *smem) {
    switch (M) {
        case 1: *smem = tile_smem_bytes<MPMI_D, 1>(); return rollout_tile_kernel<MPMI_D, 1, MPMI_MODE, (MPMI_NOISE != 0)>;
        case 2: *smem = tile_smem_bytes<MPMI_D, 2>(); return rollout_tile_kernel<MPMI_D, 2, MPMI_MODE, (MPMI_NOISE != 0)>;
        case 3: *smem = tile_smem_bytes<MPMI_D, 3>(); return rollout_tile_kernel<MPMI_D, 3, MPMI_MODE, (MPMI_NOISE != 0)>;
        case 4: *smem = tile_smem_bytes<MPMI_D, 4>(); return rollout_tile_kernel<MPMI_D, 4, MPMI_MODE, (MPMI_NOISE != 0)>;
    }
    return nullptr;
}

#if MPMI_D == 128
// second pass of the verified tensor-core tick / batch: 8-candidate warp batches (rollout_tile.cuh)
#define RCFN3(a) a##_rc
#define RCFN2(a) RCFN3(a)
KernFn RCFN2(FN2(MPMI_D))(int M, int *smem) {
    switch (M) {
        case 1: *smem = tile_smem_bytes<MPMI_D, 1, kTileWCRecheck>(); return rollout_tile_kernel<MPMI_D, 1, MPMI_MODE, (MPMI_NOISE != 0), kTileWCRecheck>;
        case 2: *smem = tile_smem_bytes<MPMI_D, 2, kTileWCRecheck>(); return rollout_tile_kernel<MPMI_D, 2, MPMI_MODE, (MPMI_NOISE != 0), kTileWCRecheck>;
        case 3: *smem = tile_smem_bytes<MPMI_D, 3, kTileWCRecheck>(); return rollout_tile_kernel<MPMI_D, 3, MPMI_MODE, (MPMI_NOISE != 0), kTileWCRecheck>;
        case 4: *smem = tile_smem_bytes<MPMI_D, 4, kTileWCRecheck>(); return rollout_tile_kernel<MPMI_D, 4, MPMI_MODE, (MPMI_NOISE != 0), kTileWCRecheck>;
    }
    return nullptr;
}
#endif
