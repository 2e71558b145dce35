// rollout_affine.cuh -- affine-in-u fast path for the noise-free linear lifted model.
//
// With z' = K z + B u, the same u held over the horizon and no noise, the physical state
// is affine in the candidate input:
//     x_k = C K^k z_0 + (C S_k B) u = a_k + G_k u,      S_k = sum_{i<k} K^i,   k = 1..H.
// G_k (n x m per step) depends on the model only and is computed once, in FP64, by mpmi_create;
// a_k (n per step) depends on x_t and is produced per tick by affine_base_kernel as (C K^k) Psi(x_t), with the
// n rows of C K^k tabulated in FP64 by mpmi_create as well (H independent n x d products, one CTA each).  The candidate
// kernel then needs n*m FMAs per sample-step instead of d*(d+m): the SAME states, flags and selection
// as Algorithm 2 up to fp32 rounding, at ~d^2/(n m) times less arithmetic.  It is
// an opt-in variant (MPMI_VARIANT_AFFINE) with its own metric; it is invalid with prediction noise or
// the re-lift model, and mpmi_create ignores the flag there.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

// ---- a_k = (C K^k) Psi(x_t), k = 1..H: CTA k, the n rows of C K^k (FP64 at create, cfg.aff_m) times z_0 ----------
// (H dependent mat-vec steps in one CTA took 25 us; H independent n x d products take a launch.)
constexpr int kAffBaseThreads = 128;
template <int D>
__global__ void __launch_bounds__(kAffBaseThreads) affine_base_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    __shared__ float sz[D];
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    for (int f = threadIdx.x; f < D; f += kAffBaseThreads) sz[f] = lift_feature(cfg, f, x0p);
    __syncthreads();
    const int NP = cfg.aff_np, k = blockIdx.x, lane = threadIdx.x & 31;
    for (int q = threadIdx.x >> 5; q < NP; q += kAffBaseThreads / 32) {
        const float *mrow = cfg.aff_m + ((size_t)k * NP + q) * D;
        float s = 0.f;
        for (int c = lane; c < D; c += 32) s = __fmaf_rn(__ldg(mrow + c), sz[c], s);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) cfg.aff_a[k * NP + q] = q < cfg.n ? s : 0.f;
    }
}

constexpr int kAffBlock = 256;

// ---- candidates: x_k = a_k + G_k u, isSafe, first violation, key, argmin (a1, a4-a7; a9 physical dumps) ----
template <int NP, int MODE>
__global__ void __launch_bounds__(kAffBlock) rollout_affine_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    static_assert(NP == 4 || NP == 8 || NP == 16, "padded physical dim");
    constexpr int NB = kMaxN;
    extern __shared__ __align__(16) float sag[];               // [k][1 + m][NP]: a_k, then the m columns of G_k
    const int tid = threadIdx.x;
    const int n = cfg.n, m = cfg.m;
    const int H = (MODE == MODE_TICK) ? cfg.H : a.H;            // a.H <= cfg.H: G_k is tabulated for the context's horizon
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const long long ncand = (MODE == MODE_TICK) ? cfg.shard_count : a.ncand;
    const int stride = (1 + m) * NP;
    for (int e = tid; e < H * stride; e += kAffBlock) {
        const int k = e / stride, c = (e % stride) / NP, j = e % NP;
        sag[e] = c == 0 ? cfg.aff_a[k * NP + j] : cfg.aff_g[(k * m + (c - 1)) * NP + j];
    }
    float u_h[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    bool inputs_ok = true;
    if (MODE == MODE_TICK) {
        inputs_ok = finite_inputs(cfg, x0p, uup);
        clamp_user(cfg, uup, u_h);
    }
    __syncthreads();

    long long li = (long long)blockIdx.x * kAffBlock + tid;
    if (MODE == MODE_TICK && a.perm && li < a.nsamp) li = a.perm[li];               // spatially ordered walk
    const bool valid = li < ncand && inputs_ok;
    bool alive = valid;
    int steps = 0;
    float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    if (li < ncand) {
        if (MODE == MODE_BATCH && a.U) {
#pragma unroll
            for (int j = 0; j < kMaxM; j++) if (j < m) u[j] = a.U[li * m + j];
        } else {
            sample_u(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, tick, u_h, u);
        }
    }
    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const bool dump = (MODE == MODE_BATCH) && a.dump_kind == MPMI_DUMP_PHYS;
    const float qnan = __int_as_float(0x7fc00000);

    int k = 0;
    for (; k < H; k++) {
        if (!__any_sync(0xffffffffu, alive)) break;
        const float *row = sag + k * stride;
        float x[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) x[j] = 0.f;
#pragma unroll
        for (int j = 0; j < NP; j += 4) {
            float4 v = *reinterpret_cast<const float4 *>(row + j);
#pragma unroll
            for (int i = 0; i < kMaxM; i++) {
                if (i < m) {
                    const float4 g = *reinterpret_cast<const float4 *>(row + (1 + i) * NP + j);
                    v.x = __fmaf_rn(g.x, u[i], v.x); v.y = __fmaf_rn(g.y, u[i], v.y);
                    v.z = __fmaf_rn(g.z, u[i], v.z); v.w = __fmaf_rn(g.w, u[i], v.w);
                }
            }
            x[j] = v.x; x[j + 1] = v.y; x[j + 2] = v.z; x[j + 3] = v.w;
        }
        const bool was_alive = alive;
        alive = was_alive && safe_check<NB>(cfg, x, nbox);
        steps += alive ? 1 : 0;
        if (dump && li < ncand) {
#pragma unroll
            for (int j = 0; j < NP; j++)
                if (j < n) a.traj[((long long)k * n + cfg.perm[j]) * ncand + li] = was_alive ? x[j] : qnan;
        }
    }
    if (dump && li < ncand)
        for (; k < H; k++)
            for (int row = 0; row < n; row++) a.traj[((long long)k * n + row) * ncand + li] = qnan;

    if (MODE == MODE_BATCH) {
        if (li < ncand) {
            a.steps[li] = steps;
            if (a.safe) a.safe[li] = steps == H ? 1 : 0;
        }
        return;
    }
    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;
    if (a.steps && li < ncand) a.steps[li] = steps;             // mpmi_step_trace: per-candidate steps of THIS tick kernel
    if (valid) {
        const bool safe = steps == H;
        float d2 = 0.f;
#pragma unroll
        for (int j = 0; j < kMaxM; j++) {
            const float df = __fsub_rn(u[j], u_h[j]);
            d2 = __fmaf_rn(df, df, d2);
        }
        key = make_key(safe, d2, H, steps, cfg.shard_begin + li);
        n_safe = safe ? 1u : 0u;
        n_exec = (unsigned)(steps + 1 < H ? steps + 1 : H);
    }
    block_select_and_finalise<kAffBlock / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq);
}

}  // namespace mpmi
