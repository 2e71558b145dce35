// inst_reg.cu -- instantiates the register-resident kernels for one (MPMI_D, MPMI_MODE); compiled
// once per pair by build.py so that the translation units build in parallel.
#include "rollout_reg.cuh"
#ifndef MPMI_D
#error "compile with -DMPMI_D=8|16|32 -DMPMI_MODE=0|1"
#endif
using namespace mpmi;
#ifndef MPMI_NOISE
#define MPMI_NOISE 0
#endif
#if MPMI_MODE == 0 && !MPMI_NOISE
#define FN(D) mpmi_pick_reg_##D##_tick
#elif !MPMI_NOISE
#define FN(D) mpmi_pick_reg_##D##_batch
#elif MPMI_MODE == 0
#define FN(D) mpmi_pick_regn_##D##_tick
#else
#define FN(D) mpmi_pick_regn_##D##_batch
#endif
#define FN2(D) FN(D)

template <int M>
static KernFn pick_p(int P, int kconst) {
    constexpr int PW = 32 / MPMI_D;                 // wide packing: 2*PW candidates per thread
    if (!kconst) {                               // shared-memory model (small grids, or no free constant slot)
        if (P == 1) return rollout_reg_kernel<MPMI_D, M, 1, MPMI_MODE, (MPMI_NOISE != 0), false>;
        if (P == PW) return rollout_reg_kernel<MPMI_D, M, PW, MPMI_MODE, (MPMI_NOISE != 0), false>;
    }
    if (P == 1) return rollout_reg_kernel<MPMI_D, M, 1, MPMI_MODE, (MPMI_NOISE != 0), true>;
    if (P == PW) return rollout_reg_kernel<MPMI_D, M, PW, MPMI_MODE, (MPMI_NOISE != 0), true>;
    return nullptr;
}
KernFn FN2(MPMI_D)(int M, int P, int kconst) {
    switch (M) {
        case 1: return pick_p<1>(P, kconst);
        case 2: return pick_p<2>(P, kconst);
        case 3: return pick_p<3>(P, kconst);
        case 4: return pick_p<4>(P, kconst);
    }
    return nullptr;
}

#if MPMI_MODE == 0 && MPMI_D == 32
// second pass of the verified tensor-core tick: 2 candidates per thread; model from the constant bank or from shared memory
#if MPMI_NOISE
#define RCFN mpmi_pick_regn_32_recheck
#else
#define RCFN mpmi_pick_reg_32_recheck
#endif
template <bool KC>
static KernFn pick_rc(int M) {
    switch (M) {
        case 1: return rollout_reg_kernel<32, 1, 1, MODE_TICK, (MPMI_NOISE != 0), KC, true>;
        case 2: return rollout_reg_kernel<32, 2, 1, MODE_TICK, (MPMI_NOISE != 0), KC, true>;
        case 3: return rollout_reg_kernel<32, 3, 1, MODE_TICK, (MPMI_NOISE != 0), KC, true>;
        case 4: return rollout_reg_kernel<32, 4, 1, MODE_TICK, (MPMI_NOISE != 0), KC, true>;
    }
    return nullptr;
}
KernFn RCFN(int M, int kconst) { return kconst ? pick_rc<true>(M) : pick_rc<false>(M); }
#endif

// fills constant-memory slot `slot` of THIS translation unit with the context's augmented transposed model
#define SETFN3(a, b) a##b
#define SETFN2(a, b) SETFN3(a, b)
int SETFN2(FN2(MPMI_D), _setmodel)(int slot, const float *kta, int nfloats) {
    if (slot < 0 || slot >= kModelSlots || nfloats > kModelFloats) return (int)cudaErrorInvalidValue;
    return (int)cudaMemcpyToSymbol(c_model, kta, sizeof(float) * nfloats, sizeof(float) * kModelFloats * slot, cudaMemcpyHostToDevice);
}
