// bound.cuh -- per-tick bound tau_i(k) on the difference between the 3xTF32 tensor-core rollout and the FP32 rollout
// of the SAME candidate, for the verified tensor-core tick (rollout_tc.cuh).
//
// Both kernels iterate z_{k+1} = K z_k + B u from the same z_0 and u:
//     tensor cores  z~_{k+1} = K z~_k + B u + e~_k,      FP32  z^_{k+1} = K z^_k + B u + e^_k,
// so their difference obeys D_{k+1} = K D_k + (e~_k - e^_k), i.e. for the physical rows x = C z that isSafe reads
//
//     |x~_k - x^_k|_i  <=  sum_{p=0}^{k-1} sum_c |(C K^p)_{ic}| ( |e~_{k-1-p}| + |e^_{k-1-p}| )_c .
// One step's rounding errors are bounded row by row by a weighted sum of the ABSOLUTE products,
//     (|e~| + |e^|)_r  <=  E_r := sum_c w_c |K_rc| |z_c|   (input columns: |B_rj| |u_j|),
// with w_c fixed by the two arithmetics alone (mpmi_api.cu: bound_weights; each term is listed there):
//   * FP32 chain of D+M FMAs, columns in descending order: term c is rounded (c+1) times, 2^-24 each;
//   * 3xTF32: the dropped z_lo K_lo product (2^-21) and the TF32 rounding of z_lo (2^-21) and K_lo (2^-22);
//   * the tensor core's fp32 accumulation, <= 2 ulp (truncation) per MMA on the running sum, counted for the
//     full-magnitude Z_hi K_hi products from column c's k-block on (state block b: b+1 of them, the blocks run
//     in descending order); the small products before them add 2^-31 each.
//   Both orders put the physical dims (internal columns 0..n-1) last: for a model close to the identity on the physical
//   block the dominant product of a physical row is the diagonal one, and it is then re-rounded <= n (once) instead of
//   D+M (KB+1) times -- on C4 that alone cuts tau, and with it the second pass, to a third.
//   (tests/test_parity_full_gpu.py::test_single_step_error_within_bound measures one step of every kernel against
//   exactly these E_r.)
// |z_c| of an arbitrary candidate is bounded over the whole input box by the envelope of the affine map
//     z_j = K^j z_0 + (S_j B) u,  S_j = sum_{i<j} K^i:   |z_jc| <= |zeta_jc| + sum_i |(S_j B)_ci| (u_hi - u_lo)_i / 2,
// zeta_j = the rollout of the box centre.  K^j, S_j B and every tick-independent sum are tabulated in FP64 by
// mpmi_create; per tick two small kernels evaluate
//     bound_err_kernel   CTA j:  zeta_j = K^j Psi(x_t) + (S_j B) u_mid,   E[j][r] = sum_c w_c |K_rc| |zeta_jc| + Econst[j][r]
//     bound_tau_kernel   CTA k:  tau[k][i] = 1.01 * sum_{p<k} sum_c |(C K^p)_ic| E[k-1-p][c]
// (H CTAs each; they run beside the binning kernels in the tick graph).  A candidate whose tensor-core state never comes
// within tau_i(k) of a safe-set boundary has, step by step, the same isSafe result in FP32 arithmetic; one that does is
// handed to the FP32 kernel.  The factor 1.01 covers the fp32 evaluation of the bound itself and second-order terms
// (the envelope is taken around the exact trajectory, the rounding errors act on the computed ones: relative 1e-5).
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

constexpr int kTauPad = 4;            // tau row = [tau_0 .. tau_{NP-1} | thr(r_min^2), thr(r_max^2), 0, 0]

template <int D>
__global__ void __launch_bounds__(D < 64 ? 64 : D) bound_err_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    constexpr int T = D < 64 ? 64 : D;
    __shared__ float sz[D], sabs[D];
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    for (int f = threadIdx.x; f < D; f += T) sz[f] = lift_feature(cfg, f, x0p);
    __syncthreads();
    const int j = blockIdx.x, r = threadIdx.x;
    if (r < D) {
        const float *kp = cfg.bnd_kpow + (size_t)j * D * D;        // kpowT[j][c][r] = (K^j)[r][c]
        float s0 = cfg.bnd_mid[j * D + r], s1 = 0.f;
#pragma unroll 4
        for (int c = 0; c < D; c += 2) {
            s0 = __fmaf_rn(__ldg(kp + c * D + r), sz[c], s0);
            s1 = __fmaf_rn(__ldg(kp + (c + 1) * D + r), sz[c + 1], s1);
        }
        sabs[r] = fabsf(s0 + s1);
    }
    __syncthreads();
    if (r < D) {
        float e0 = cfg.bnd_econst[j * D + r], e1 = 0.f;
#pragma unroll 4
        for (int c = 0; c < D; c += 2) {
            e0 = __fmaf_rn(cfg.bnd_w[c] * fabsf(__ldg(cfg.KTa + c * D + r)), sabs[c], e0);
            e1 = __fmaf_rn(cfg.bnd_w[c + 1] * fabsf(__ldg(cfg.KTa + (c + 1) * D + r)), sabs[c + 1], e1);
        }
        cfg.bnd_e[j * D + r] = e0 + e1;
    }
}

constexpr int kBoundTauThreads = 512;         // 16 warps share the p < k terms of one tau row
template <int D, int NP>
__global__ void __launch_bounds__(kBoundTauThreads) bound_tau_kernel(const __grid_constant__ DevCfg cfg) {
    __shared__ float red[kBoundTauThreads / 32][NP];
    const int k = blockIdx.x + 1;                                   // bound for the predicted state x_k, k = 1..H
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float acc[NP];
#pragma unroll
    for (int i = 0; i < NP; i++) acc[i] = 0.f;
    // p = 0: C K^0 = [I_n 0]
    if (warp == 0 && lane < NP && lane < cfg.n) {
#pragma unroll
        for (int i = 0; i < NP; i++) if (i == lane) acc[i] = cfg.bnd_e[(k - 1) * D + lane];
    }
    for (int p = 1 + warp; p < k; p += kBoundTauThreads / 32) {    // rows of C K^p: cfg.aff_m[p - 1]
        const float *m = cfg.aff_m + (size_t)(p - 1) * NP * D;
        const float *e = cfg.bnd_e + (size_t)(k - 1 - p) * D;
#pragma unroll
        for (int c = lane; c < D; c += 32) {                        // (D / 32 independent column slices: all loads in flight)
            const float ec = e[c];
#pragma unroll
            for (int i = 0; i < NP; i++) acc[i] = __fmaf_rn(fabsf(__ldg(m + i * D + c)), ec, acc[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < NP; i++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], o);
        if (lane == 0) red[warp][i] = acc[i];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        float *row = cfg.bnd_tau + (size_t)k * (NP + kTauPad);
        float t[NP];
#pragma unroll
        for (int i = 0; i < NP; i++) {
            float s = 0.f;
#pragma unroll
            for (int w = 0; w < kBoundTauThreads / 32; w++) s += red[w][i];
            t[i] = i < cfg.n ? 1.01f * s + 1e-30f : 0.f;
            row[i] = t[i];
        }
        // annulus on internal dims 0, 1: |r~ - r^| <= hypot(tau_0, tau_1) =: tr, and a flag can differ only if r~ lies within tr
        // of r_min (r_max): |r~^2 - r_min^2| <= tr (2 r_min + tr).  Both kernels round r^2 = dx^2 + dy^2 in fp32 (relative 2^-23
        // at most, of values up to (r_max + tr)^2): added on both sides.
        float thr_lo = 0.f, thr_hi = 0.f;
        if (cfg.annulus && NP >= 2) {
            const float tr = 1.0001f * sqrtf(t[0] * t[0] + t[1] * t[1]);
            const float rmin = sqrtf(cfg.rmin2), rmax = sqrtf(fmaxf(cfg.rmax2, 0.f));
            const float rnd = 4.f * 1.2e-7f * (rmax + tr) * (rmax + tr);
            thr_lo = 1.0001f * tr * (2.f * rmin + tr) + rnd;
            thr_hi = 1.0001f * tr * (2.f * rmax + tr) + rnd;
        }
        row[NP] = thr_lo; row[NP + 1] = thr_hi; row[NP + 2] = 0.f; row[NP + 3] = 0.f;
    }
}

}  // namespace mpmi
