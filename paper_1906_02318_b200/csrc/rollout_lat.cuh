// rollout_lat.cuh -- latency-oriented tick kernel for small candidate sets (N ~ 1e4, padded D <= 32).
//
// At the paper's scale (N = 10,000 / 10,120 candidates) one candidate per thread leaves
// most of the 148 SMs idle and the tick time is one warp's instruction stream (C3: 85k instructions).
// Here L = D/R consecutive lanes (R = 2 or 4) share ONE candidate: lane q owns rows [Rq, Rq+R) of
// z' = K z + B u and keeps those rows of the augmented model in REGISTERS for the whole horizon
// (R*(D+M) floats), so the horizon loop touches no memory at all: per step (R/2)*(D+M) FFMA2 (two
// rows per instruction, the state value broadcast), then the L lanes all-gather the new state with D
// warp shuffles.  Every lane then holds the full state and tests the safe set itself.
// Each row sum is split into an even-c and an odd-c chain (twice the ILP, half the dependent latency),
// so its rounding order differs from rollout_reg_kernel by one reassociation (well inside T1).
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

constexpr int kLatBlock = 64;
template <int D, int M, int R>
__global__ void __launch_bounds__(kLatBlock, (D == 32 && R == 4) ? 4 : 8)
rollout_lat_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    constexpr int L = D / R;                      // lanes per candidate: 2 ... 16
    static_assert(R == 2 || R == 4, "rows per lane");
    constexpr int NB = D < kMaxN ? D : kMaxN;
    __shared__ float sz0[D];

    const int tid = threadIdx.x, lane = tid & 31, q = lane & (L - 1);
    // mpmi_profile_timeline: thread 0 of every CTA stamps the stages (ns, %globaltimer); a.timeline == null costs one uniform branch each
    unsigned long long *tl = a.timeline ? a.timeline + 8ull * blockIdx.x : nullptr;
#define MPMI_STAMP(i) do { if (tl && tid == 0) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); tl[i] = t_; } } while (0)
    MPMI_STAMP(0);                                // kernel entry
    // this lane's rows of the augmented transposed model, as row pairs
    float2 kreg[D + M][R / 2];
    {
        const float2 *kt = reinterpret_cast<const float2 *>(cfg.KTa + q * R);
#pragma unroll
        for (int c = 0; c < D + M; c++)
#pragma unroll
            for (int p = 0; p < R / 2; p++) kreg[c][p] = __ldg(kt + (c * D) / 2 + p);
    }
    MPMI_STAMP(1);                                // model rows requested (the loads are still in flight)
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const int H = cfg.H;
    const long long ncand = cfg.shard_count;

    float u_h[kMaxM];
    const bool inputs_ok = finite_inputs(cfg, x0p, uup);
    clamp_user(cfg, uup, u_h);
    for (int f = tid; f < D; f += kLatBlock) sz0[f] = lift_feature(cfg, f, x0p);
    __syncthreads();
    MPMI_STAMP(2);                                // lift done, CTA synchronised

    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const bool no_annulus = cfg.annulus == 0;
    // only constrained dims are tested (as in every other kernel and in the oracle): an unconstrained dim passes whatever
    // it holds, Inf and NaN included -- its (-inf, +inf) limits alone would reject those.  One AND per dim: the state's bit
    // pattern is masked to +0.0 where the dim is unconstrained, and 0 lies inside (-inf, +inf).
    unsigned zm[NB];
#pragma unroll
    for (int j = 0; j < NB; j++) zm[j] = ((cfg.bmask >> j) & 1u) ? 0xFFFFFFFFu : 0u;
    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;

    // A CTA rolls batches blockIdx, blockIdx + gridDim, ... of kLatBlock / L candidates.  The grid is one batch per CTA unless
    // that exceeds what is resident at once (d = 32 with 4 rows per lane: 200 registers, i.e. two warps per sub-partition's 16 K
    // registers, 4 CTAs per SM; 10,000 candidates are 1,251 batches): then the grid is the resident set, and a CTA's later batches
    // re-use its model rows and its lift instead of paying the prologue again in another wave (mpmi_api.cu: lat_cap).  Measured:
    // C4 model at 2^14 candidates 131 -> 121 us, C3 46.7 -> 45.2 us.  (Three warps per sub-partition need <= 168 registers: spills,
    // 58 us at 176.)
    const long long nbatch = (ncand + kLatBlock / L - 1) / (kLatBlock / L);
  for (long long blk = blockIdx.x; blk < nbatch; blk += gridDim.x) {
    // ---- a1 + a2 ----------------------------------------------------------------------------------
    const long long li = blk * (kLatBlock / L) + tid / L;
    bool alive = li < ncand && inputs_ok;
    int steps = 0;
    float z[D + M];
    {
        float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
        if (li < ncand) sample_u(cfg, cfg.shard_begin + li, tick, u_h, u);
#pragma unroll
        for (int j = 0; j < M; j++) z[D + j] = u[j];
#pragma unroll
        for (int c = 0; c < D; c++) z[c] = sz0[c];
    }
    if (blk == blockIdx.x) MPMI_STAMP(3);         // candidate sampled (Philox / grid), state initialised (first batch)

    // ---- a3 + a4: no memory traffic inside this loop -----------------------------------------------
    for (int k = 0; k < H; k++) {
        if ((k & 3) == 0 && !__any_sync(0xffffffffu, alive)) break;      // warp exit, tested every 4th step
        float2 acc[R / 2], odd[R / 2];
#pragma unroll
        for (int p = 0; p < R / 2; p++) {
            acc[p] = make_float2(__fmul_rn(kreg[0][p].x, z[0]), __fmul_rn(kreg[0][p].y, z[0]));
            odd[p] = make_float2(__fmul_rn(kreg[1][p].x, z[1]), __fmul_rn(kreg[1][p].y, z[1]));
        }
#pragma unroll
        for (int c = 2; c < D + M; c++)
#pragma unroll
            for (int p = 0; p < R / 2; p++) fma2_bcast_z((c & 1) ? odd[p] : acc[p], kreg[c][p], z[c]);
#pragma unroll
        for (int p = 0; p < R / 2; p++) acc[p] = make_float2(__fadd_rn(acc[p].x, odd[p].x), __fadd_rn(acc[p].y, odd[p].y));
        // all-gather of the new state inside the L-lane group
#pragma unroll
        for (int qq = 0; qq < L; qq++)
#pragma unroll
            for (int r = 0; r < R; r++)
                z[qq * R + r] = __shfl_sync(0xffffffffu, (r & 1) ? acc[r / 2].y : acc[r / 2].x, qq, L);

        // a4, branch-free for the common shapes: dims 0..3 against their limits (always true where there is
        // none), the annulus folded in arithmetically; only more than 4 boxed dims take a branch
        bool ok = true;
#pragma unroll
        for (int j = 0; j < 4 && j < NB; j++) {
            const float zt = __uint_as_float(__float_as_uint(z[j]) & zm[j]);
            ok = ok & (zt > cfg.blo[j]) & (zt < cfg.bhi[j]);
        }
        {
            const float dx = __fsub_rn(z[0], cfg.cx), dy = __fsub_rn(z[1], cfg.cy);
            const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
            ok = ok & (((r2 >= cfg.rmin2) & (r2 <= cfg.rmax2)) | no_annulus);
        }
        if (nbox > 4) {
#pragma unroll
            for (int j = 4; j < NB; j++) {
                const float zt = __uint_as_float(__float_as_uint(z[j]) & zm[j]);
                ok = ok & (zt > cfg.blo[j]) & (zt < cfg.bhi[j]);
            }
        }
        alive = alive & ok;
        steps += alive ? 1 : 0;
    }

    if (blk == blockIdx.x) MPMI_STAMP(4);         // horizon loop left (warp 0 of the CTA, first batch)
    // ---- a5 ------------------------------------------------------------------------------------------
    if (a.steps && q == 0 && li < ncand) a.steps[li] = steps;    // mpmi_step_trace
    if (q == 0 && li < ncand && inputs_ok) {
        const bool safe = steps == H;
        float d2 = 0.f;
#pragma unroll
        for (int j = 0; j < M; j++) {
            const float df = __fsub_rn(z[D + j], u_h[j]);
            d2 = __fmaf_rn(df, df, d2);
        }
        const unsigned long long kk = make_key(safe, d2, H, steps, cfg.shard_begin + li);
        key = kk < key ? kk : key;
        n_safe += safe ? 1u : 0u;
        n_exec += (unsigned)(steps + 1 < H ? steps + 1 : H);
    }
  }
    // ---- a6 + a7 -------------------------------------------------------------------------------------
    block_select_and_finalise<kLatBlock / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq);
    MPMI_STAMP(5);                                // keys reduced, ticket taken (last CTA: result written)
#undef MPMI_STAMP
}

}  // namespace mpmi
