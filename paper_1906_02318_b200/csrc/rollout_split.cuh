// rollout_split.cuh -- row-split FP32 kernel for padded lifted dim D = 32: the SECOND PASS of the verified tensor-core tick
// (kernel_args.cuh: recheck) when it holds few candidates.
//
// rollout_reg_kernel gives one thread a whole candidate pair: D (D + M) = 1088 dependent-issue FFMA2 per step, ~2,200 clk of a
// sub-partition's FMA pipe.  That is the right shape when the grid fills the machine several times over, but the second pass sees
// a few per cent of the candidates -- about one such warp per sub-partition -- and then lasts as long as ONE warp needs for the
// whole horizon (measured on C4: 250 us for 3.8 % of 2^20 candidates, however the blocks are dealt out).  Here RS = 2, 4, 8 or 16
// consecutive lanes share a candidate pair: lane q owns rows [q D/RS, (q+1) D/RS) of z' = K z + B u for
// both candidates of the pair (FFMA2, model value broadcast to both halves, from shared memory: the lanes of a warp need different
// rows, so the constant-bank operand of rollout_reg_kernel does not apply), then the RS lanes all-gather the new state with warp
// shuffles and every lane tests the safe set itself.  The per-step chain of a warp shrinks RS-fold and RS times as
// many warps share the latency; the shuffles and the four-address LDS.128 cost throughput (as a whole tick it is SLOWER than
// rollout_reg_kernel at every N: 2^16 candidates 322 / 542 us at RS = 2 / 4 against 271 us), so it serves the second pass only:
// measured verified tick at 2^16 / 2^17 / 2^18 / 2^19 candidates 397 / 478 / 597 / 852 us with rollout_reg_kernel as second pass,
// 241 / 321 / 452 / 760 us with RS = 4; at 2^20 (40,000 deferred: throughput-bound again) 1.32 ms against 1.30 ms with RS = 2.
// (An all-gather through shared memory -- RL / 2 STS.128 + D / 2 LDS.128 per lane instead of 2 D shuffles -- was measured
// and is slightly slower: second pass 0.197 -> 0.212 ms at 2^20 candidates, 0.104 -> 0.108 ms at 2^18.)
// With 8 lanes per pair (4 rows per lane) the chain halves again: best up to ~300,000 candidates (tick at 40,000 / 2^16 / 2^17 / 2^18
// candidates 164 / 176 / 255 / 369 us against 180 / 192 / 266 / 376 us with 4 lanes).
// 16 lanes (one row pair per lane) still gain below ~80,000 candidates (40,000: 157 against 164 us, 2^16: 173 against 176 us; 100,000:
// 223 against 221 us): the all-gather's 64 shuffles per step do not shrink with the rows.
// (Round-2 late: FFMA2 over two ROWS of one candidate instead of one row of two candidates removed ~1.5 register moves per FFMA2
// -- the pass was bound by issue slots: second pass at 2^20 candidates 0.198 -> 0.166 ms, verified tick at 2^16 .. 2^20 now
// 208 / 263 / 376 / 596 / 964 us.)
// Every row is the same FMA chain as in rollout_reg_kernel (columns descending, first product a plain multiply), so states,
// flags and keys are bit-identical to it: which lane computes a row does not change its bits.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

constexpr int kSplitBlock = 128;

// One-warp CTAs walk the deferral lists (longest-lived first) in blocks of 64 / RS candidates, their own block first, then
// first come, first served (a.recheck_count[kRecheckBuckets]); the last CTA finalises the tick.
template <int D, int M, int RS, bool NOISE = false>
__global__ void __launch_bounds__(kSplitBlock, 3)
rollout_split_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    static_assert(D == 32 && (RS == 2 || RS == 4 || RS == 8 || RS == 16), "row-split kernel: D = 32; 2, 4, 8 or 16 lanes per candidate pair");
    constexpr int RL = D / RS;                   // rows per lane
    constexpr int NB = kMaxN;
    __shared__ __align__(16) float sK[(D + M) * D];
    __shared__ float sz0[D];
    const int tid = threadIdx.x, bdim = blockDim.x, lane = tid & 31, q = lane & (RS - 1);
    for (int i = tid; i < (D + M) * D / 4; i += bdim)
        reinterpret_cast<float4 *>(sK)[i] = reinterpret_cast<const float4 *>(cfg.KTa)[i];
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(sK) + (unsigned)(q * RL * 4);
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const int H = cfg.H;
    const long long ncand = cfg.shard_count;
    float u_h[kMaxM];
    const bool inputs_ok = finite_inputs(cfg, x0p, uup);
    clamp_user(cfg, uup, u_h);
    for (int f = tid; f < D; f += bdim) sz0[f] = lift_feature(cfg, f, x0p);
    __syncthreads();

    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;
    int rc_count[kRecheckBuckets], rc_total = 0;
#pragma unroll
    for (int b = 0; b < kRecheckBuckets; b++) { rc_count[b] = (int)a.recheck_count[b]; rc_total += rc_count[b]; }
    const int cpb = 2 * (bdim / RS);             // candidates per block
    for (long long blk = blockIdx.x; blk * cpb < rc_total;) {
        // ---- a1 + a2: the candidate pair of this lane group (both halves of the float2 registers)
        long long li[2];
        bool alive[2];
        int steps[2] = {0, 0};
        float2 z[D + M];
#pragma unroll
        for (int s = 0; s < 2; s++) {
            li[s] = blk * cpb + 2 * (tid / RS) + s;
            {                                                                         // slot p of the concatenated lists
                int p = (int)li[s];
                long long hit = ncand;
#pragma unroll
                for (int b = 0; b < kRecheckBuckets; b++) {
                    if (p >= 0 && p < rc_count[b]) hit = (long long)a.recheck[(long long)b * ncand + p];
                    p -= rc_count[b];
                }
                li[s] = hit;
            }
            alive[s] = li[s] < ncand && inputs_ok;
            float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
            if (li[s] < ncand) sample_u(cfg, cfg.shard_begin + li[s], tick, u_h, u);
#pragma unroll
            for (int j = 0; j < M; j++) { if (s) z[D + j].y = u[j]; else z[D + j].x = u[j]; }
        }
#pragma unroll
        for (int c = 0; c < D; c++) z[c] = make_float2(sz0[c], sz0[c]);

        // ---- a3 + a4: horizon loop
        for (int k = 0; k < H; k++) {
            if (!__any_sync(0xffffffffu, alive[0] || alive[1])) break;
            // FFMA2 over two ROWS of one candidate (model pair straight from the LDS.128, state value broadcast): with the model
            // value as the broadcast operand every FFMA2 needed its own {k, k} register pair -- ~1.5 moves per FFMA2, and the
            // pass was bound by issue slots (two such warps per sub-partition), not by the FMA pipe.  The state value's pair
            // is built once per column and candidate.  Same fma(k, z, acc) sequence per row as before: same bits.
            float2 acc0[RL / 2], acc1[RL / 2];                   // candidate 0 / 1 of the pair, rows (2i, 2i + 1) of this lane
#pragma unroll
            for (int cc = 0; cc < D + M; cc++) {                 // columns descending, as in rollout_reg_kernel
                const int c = D + M - 1 - cc;
                const float2 zc = z[c];
                if (RL == 2) {                               // 16 lanes per pair: one row pair per lane
                    float2 k01;
                    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(k01.x), "=f"(k01.y) : "r"(sbase + (unsigned)(c * D * 4)));
                    if (cc == 0) { mul2_bcast_z(acc0[0], k01, zc.x); mul2_bcast_z(acc1[0], k01, zc.y); }
                    else         { fma2_bcast_z(acc0[0], k01, zc.x); fma2_bcast_z(acc1[0], k01, zc.y); }
                }
#pragma unroll
                for (int r = 0; r + 3 < RL; r += 4) {
                    const float4 kv = lds128(sbase + (c * D + r) * 4);
                    const float2 k01 = make_float2(kv.x, kv.y), k23 = make_float2(kv.z, kv.w);
                    if (cc == 0) {
                        mul2_bcast_z(acc0[r / 2], k01, zc.x); mul2_bcast_z(acc0[r / 2 + 1], k23, zc.x);
                        mul2_bcast_z(acc1[r / 2], k01, zc.y); mul2_bcast_z(acc1[r / 2 + 1], k23, zc.y);
                    } else {
                        fma2_bcast_z(acc0[r / 2], k01, zc.x); fma2_bcast_z(acc0[r / 2 + 1], k23, zc.x);
                        fma2_bcast_z(acc1[r / 2], k01, zc.y); fma2_bcast_z(acc1[r / 2 + 1], k23, zc.y);
                    }
                }
            }
            // all-gather of the new state inside the RS-lane group
#pragma unroll
            for (int qq = 0; qq < RS; qq++)
#pragma unroll
                for (int r = 0; r < RL; r++) {
                    z[qq * RL + r].x = __shfl_sync(0xffffffffu, (r & 1) ? acc0[r / 2].y : acc0[r / 2].x, qq, RS);
                    z[qq * RL + r].y = __shfl_sync(0xffffffffu, (r & 1) ? acc1[r / 2].y : acc1[r / 2].x, qq, RS);
                }
            if (NOISE) {
                // Algorithm 2 l.5: + z_i on the physical rows, before isSafe (every lane of the group draws the same eps)
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const long long gi = cfg.shard_begin + li[s];
                    float g[NB];
#pragma unroll
                    for (int qn = 0; 4 * qn < NB; qn++) {
                        float g4[4] = {0.f, 0.f, 0.f, 0.f};
                        if (4 * qn < cfg.n) noise4(cfg, gi, k, qn, tick, g4);
#pragma unroll
                        for (int e = 0; e < 4; e++) g[4 * qn + e] = g4[e];
                    }
#pragma unroll
                    for (int j = 0; j < NB; j++) {
                        if (j < cfg.n) {
                            const float e = g[cfg.perm[j]];
                            if (s) z[j].y = __fmaf_rn(cfg.noise_sigma, e, z[j].y);
                            else   z[j].x = __fmaf_rn(cfg.noise_sigma, e, z[j].x);
                        }
                    }
                }
            }
#pragma unroll
            for (int s = 0; s < 2; s++) {
                float x[NB];
#pragma unroll
                for (int j = 0; j < NB; j++) x[j] = s ? z[j].y : z[j].x;
                alive[s] = alive[s] && safe_check<NB>(cfg, x, nbox);
                steps[s] += alive[s] ? 1 : 0;
            }
        }

        // ---- a5: keys of the pair (lane 0 of the group)
#pragma unroll
        for (int s = 0; s < 2; s++) {
            if (q == 0 && li[s] < ncand) {
                if (a.steps) a.steps[li[s]] = steps[s];                              // mpmi_step_trace
                if (inputs_ok) {
                    const bool safe = steps[s] == H;
                    float d2 = 0.f;
#pragma unroll
                    for (int j = 0; j < M; j++) {
                        const float df = __fsub_rn(s ? z[D + j].y : z[D + j].x, u_h[j]);
                        d2 = __fmaf_rn(df, df, d2);
                    }
                    const unsigned long long kk = make_key(safe, d2, H, steps[s], cfg.shard_begin + li[s]);
                    key = kk < key ? kk : key;
                    n_safe += safe ? 1u : 0u;
                    n_exec += (unsigned)(steps[s] + 1 < H ? steps[s] + 1 : H);
                }
            }
        }
        unsigned nxt = 0;                        // (blockDim == 32: one warp, no block-level hand-off)
        if (tid == 0) nxt = atomicAdd(a.recheck_count + kRecheckBuckets, 1u);
        blk = (long long)gridDim.x + (long long)__shfl_sync(0xffffffffu, nxt, 0);
    }
    // ---- a6 + a7
    block_select_and_finalise<kSplitBlock / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq, nullptr, false,
                                                a.recheck_count, kRecheckBuckets, a.deferred_out);
}

}  // namespace mpmi
