// rollout_relift.cuh -- rollout kernel for the re-lift model (MPMI_MODEL_RELIFT):
//     x_{k+1} = C (K Psi(x_k) + B u) [+ sigma eps_k],
// the literal "f(x, u)" on states of PAPER.md:132 (G18): the physical state is lifted again
// before every step, so only the n physical rows of K and B are ever needed and a step costs
// d feature evaluations + n (d + m) FMAs per candidate instead of d (d + m).
//
// One thread = one candidate; its physical state x (n <= NP floats, internal order) lives in
// registers.  Per step the thread publishes x (and sin x_j / cos x_j for the dims the lift uses) in a
// private shared-memory column, then walks the d features: a MONO feature is the product of four
// table-driven factors (slot indices staged in shared memory), an RFF feature is scale cos(W_r x + b_r);
// each feature value feeds the NP accumulators through a warp-uniform LDS.128 of the transposed
// physical rows Kp[f][0..NP).  Safe test, first-violation step, key, selection and dumps are those of
// the other kernels (a4-a7, a9); the optional prediction noise is the one of rollout_reg.cuh.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

constexpr int kRlBlock = 128;

template <int NP, int MODE>
__global__ void __launch_bounds__(kRlBlock, 4)
rollout_relift_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    static_assert(NP == 4 || NP == 8 || NP == 16, "padded physical dim");
    constexpr int NB = kMaxN;                                   // safe_check works on 16 internal dims
    __shared__ __align__(16) float sKp[(MPMI_MAX_D + kMaxM) * NP]; // Kp[c][r] = K[r][c] (c < d), B[r][c-d]; rows r < n, else 0
    __shared__ float sval[(1 + 3 * NP) * kRlBlock];             // slot s of thread t at sval[s * kRlBlock + t]
    __shared__ unsigned sslot[MPMI_MAX_D];                      // MONO: up to four 6-bit slot indices per feature + their count

    const int tid = threadIdx.x;
    const int n = cfg.n, m = cfg.m, d = cfg.d, D = cfg.D;
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const int H = (MODE == MODE_TICK) ? cfg.H : a.H;
    const long long ncand = (MODE == MODE_TICK) ? cfg.shard_count : a.ncand;
    const bool shared_x0 = (MODE == MODE_TICK) || a.x0_count == 1;
    const bool mono = cfg.lift_kind == MPMI_LIFT_MONO;

    // ---- stage the physical rows of the model and the lift table -----------------------------------
    for (int e = tid; e < (d + m) * NP; e += kRlBlock) {
        const int c = e / NP, r = e % NP;
        sKp[e] = r < n ? cfg.KTa[(c < d ? c : D + (c - d)) * D + r] : 0.f;
    }
    unsigned trig_mask = 0;                                     // bit j: sin x_j needed, bit 16 + j: cos x_j needed
    if (mono) {
        for (int f = tid; f < d; f += kRlBlock) {
            // the non-unit factors in order (a factor 1.0 multiplies exactly, so skipping it is bit-identical), their
            // count in bits 24..26: most features are single states or products of two, not of four
            unsigned packed = 0, cnt = 0;
            for (int q = 0; q < 4; q++) {
                const unsigned code = cfg.terms[4 * f + q];
                if (code == 0xFFu) continue;
                packed |= (1u + (code >> 6) * n + (code & 0x3Fu)) << (6 * cnt);
                cnt++;
            }
            sslot[f] = packed | (cnt << 24);
        }
        for (int f = 0; f < d; f++)                             // uniform, once per CTA
            for (int q = 0; q < 4; q++) {
                const unsigned code = cfg.terms[4 * f + q];
                if (code != 0xFFu && (code >> 6) == 1) trig_mask |= 1u << (code & 0x3Fu);
                if (code != 0xFFu && (code >> 6) == 2) trig_mask |= 1u << (16 + (code & 0x3Fu));
            }
    }
    float u_h[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    bool inputs_ok = true;
    if (MODE == MODE_TICK) {
        inputs_ok = finite_inputs(cfg, x0p, uup);
        clamp_user(cfg, uup, u_h);
    }
    __syncthreads();

    // ---- a1: this thread's candidate ------------------------------------------------------------------
    long long li = (long long)blockIdx.x * kRlBlock + tid;
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
    float x[NP];                                                // physical state, INTERNAL order
    {
        const long long row = (!shared_x0 && li < ncand) ? li : 0;
#pragma unroll
        for (int j = 0; j < NP; j++) x[j] = j < n ? (shared_x0 ? x0p[cfg.perm[j]] : a.x0[row * n + cfg.perm[j]]) : 0.f;
    }
    const long long gi = (MODE == MODE_TICK ? cfg.shard_begin : 0) + li;
    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const bool dump = (MODE == MODE_BATCH) && a.dump_kind != MPMI_DUMP_NONE;
    const bool dump_lifted = dump && a.dump_kind == MPMI_DUMP_LIFTED;
    const int J = dump ? (dump_lifted ? d : n) : 0;
    const float qnan = __int_as_float(0x7fc00000);
    float *sv = sval + tid;

    // publish x (original order) and the trig values the lift needs in this thread's column
    auto publish = [&]() {
        sv[0] = 1.0f;
#pragma unroll
        for (int j = 0; j < NP; j++) {
            if (j < n) {
                const int p = cfg.perm[j];
                sv[(1 + p) * kRlBlock] = x[j];
                if (trig_mask & (1u << p)) sv[(1 + n + p) * kRlBlock] = sinf(x[j]);
                if (trig_mask & (1u << (16 + p))) sv[(1 + 2 * n + p) * kRlBlock] = cosf(x[j]);
            }
        }
    };
    // feature f (internal index) of the published state; same factor order as lift_feature
    auto feature = [&](int f) -> float {
        if (mono) {
            const unsigned t = sslot[f], cnt = t >> 24;                   // warp-uniform: no divergence
            if (cnt == 0) return 1.0f;
            float p = sv[(t & 0x3Fu) * kRlBlock];
            if (cnt > 1) p = __fmul_rn(p, sv[((t >> 6) & 0x3Fu) * kRlBlock]);
            if (cnt > 2) p = __fmul_rn(p, sv[((t >> 12) & 0x3Fu) * kRlBlock]);
            if (cnt > 3) p = __fmul_rn(p, sv[((t >> 18) & 0x3Fu) * kRlBlock]);
            return p;
        }
        if (f < n) return sv[(1 + cfg.perm[f]) * kRlBlock];
        const int r = f - n;
        float s = __ldg(cfg.b + r);
        for (int j = 0; j < n; j++) s = __fmaf_rn(__ldg(cfg.W + r * n + j), sv[(1 + j) * kRlBlock], s);
        return __fmul_rn(cfg.rff_scale, cosf(s));
    };

    int k = 0;
    for (; k < H; k++) {
        if (!__any_sync(0xffffffffu, alive)) break;
        // ---- a2 + a3: x' = C (K Psi(x) + B u)
        publish();
        float acc[NP];
#pragma unroll
        for (int r = 0; r < NP; r++) acc[r] = 0.f;
#pragma unroll 2
        for (int f = 0; f < d; f++) {
            const float phi = feature(f);
#pragma unroll
            for (int r = 0; r < NP; r += 4) {
                const float4 kv = *reinterpret_cast<const float4 *>(sKp + f * NP + r);
                acc[r] = __fmaf_rn(kv.x, phi, acc[r]);         acc[r + 1] = __fmaf_rn(kv.y, phi, acc[r + 1]);
                acc[r + 2] = __fmaf_rn(kv.z, phi, acc[r + 2]); acc[r + 3] = __fmaf_rn(kv.w, phi, acc[r + 3]);
            }
        }
#pragma unroll
        for (int j = 0; j < kMaxM; j++) {
            if (j < m) {
#pragma unroll
                for (int r = 0; r < NP; r++) acc[r] = __fmaf_rn(sKp[(d + j) * NP + r], u[j], acc[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < NP; r++) x[r] = acc[r];
        if (cfg.noise_sigma != 0.f) {                           // Alg. 2 l.5: + z_i, as in rollout_reg.cuh
            float g[NP];
#pragma unroll
            for (int q = 0; 4 * q < NP; q++) {
                float g4[4] = {0.f, 0.f, 0.f, 0.f};
                if (4 * q < n) noise4(cfg, gi, k, q, tick, g4);
#pragma unroll
                for (int e = 0; e < 4; e++) g[4 * q + e] = g4[e];
            }
#pragma unroll
            for (int j = 0; j < NP; j++) {
                if (j < n) {
                    x[j] = __fmaf_rn(cfg.noise_sigma, g[cfg.perm[j] < NP ? cfg.perm[j] : 0], x[j]);
                }
            }
        }
        // ---- a4: isSafe(x_p), first violation
        float xs[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) xs[j] = j < NP ? x[j < NP ? j : 0] : 0.f;
        const bool was_alive = alive;
        alive = was_alive && safe_check<NB>(cfg, xs, nbox);
        steps += alive ? 1 : 0;
        // ---- a9: dump x_{k+1} (PHYS) or the carried lifted state Psi(x_{k+1}) (LIFTED), candidate fastest
        if (dump && li < ncand) {
            float *base = a.traj + (long long)k * J * ncand + li;
            if (!dump_lifted) {
#pragma unroll
                for (int j = 0; j < NP; j++)
                    if (j < n) base[(long long)cfg.perm[j] * ncand] = was_alive ? x[j] : qnan;
            } else {
                publish();
                for (int f = 0; f < d; f++) {
                    const int row = f < n ? (int)cfg.perm[f] : f;
                    base[(long long)row * ncand] = was_alive ? feature(f) : qnan;
                }
            }
        }
    }
    if (dump && li < ncand)                                     // states after the warp stopped: NaN
        for (; k < H; k++)
            for (int row = 0; row < J; row++) a.traj[((long long)k * J + row) * ncand + li] = qnan;

    if (MODE == MODE_BATCH) {
        if (li < ncand) {
            a.steps[li] = steps;
            if (a.safe) a.safe[li] = steps == H ? 1 : 0;
        }
        return;
    }
    // ---- a5-a7: key, argmin, finalise
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
    block_select_and_finalise<kRlBlock / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq);
}

}  // namespace mpmi
