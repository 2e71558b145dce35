// rollout_tile.cuh -- warp-tile rollout kernel for padded lifted dim D in {64, 128} (a1-a7, a9).
//
// A lifted state of 128 floats cannot be thread-private, so every WARP keeps a private tile of 32
// candidates in shared memory for the whole horizon: Zw[c][i] (c < D+M rows: lifted state, then the
// candidate's input u as M extra rows; i < 32) beside the CTA-wide augmented transposed model
// KTa[c][r] (D = 128, M = 3: 8 x 16.4 KB + 67 KB).  One step is the dense contraction
// Z'[r][i] = sum_c KTa[c][r] * Z[c][i], register-blocked like an SGEMM: every lane owns D/8 rows x
// 8 candidates as float2 accumulators and advances two candidates per FFMA2 with the model value
// broadcast to both halves -- D*(D+M) fp32 FMAs per candidate-step, the algorithmic count of
// z' = K z + B u.  After write-back lane i tests candidate i against the
// safe set; a warp leaves the horizon loop when none of its 32 candidates is alive
// and fetches its next batch of 32 from a global counter (persistent CTAs, one per SM), so that
// early exits (Algorithm 2 l.4) turn into time saved.  Only warp-level synchronisation is used
// inside the horizon loop.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

constexpr int kTileWC = 16;                      // candidates per warp batch (16 -> 16 warps per CTA)
constexpr int kTileWarps = kTileNC / kTileWC;
constexpr int kTileThreadsT = kTileWarps * 32;

#ifndef MPMI_TILE_WC_RECHECK
#define MPMI_TILE_WC_RECHECK 4
#endif
constexpr int kTileWCRecheck = MPMI_TILE_WC_RECHECK;   // second pass of the verified tensor-core tick: candidates per warp batch

template <int D, int M, int WCP = kTileWC>
constexpr int tile_smem_bytes() { return ((D + M) * D + kTileWarps * (D + M) * WCP) * 4; }

// WCP = candidates per warp batch.  16 for whole ticks (lane = 8 rows x 8 candidates).  The second pass of the verified
// tensor-core tick (kernel_args.cuh: recheck) sees a few per cent of the candidates -- fewer warp batches than the machine
// has warps -- and lasts as long as its full-horizon batches: there the batch is 4 candidates (lane = 4 rows x 4 candidates),
// which quarters that chain, and four warps per CTA fetch batches longest first (see the batch loop).  Same FMA chain per
// (row, candidate), hence the same bits, for every batch size.
template <int D, int M, int MODE, bool NOISE = false, int WCP = kTileWC>
__global__ void __launch_bounds__(kTileThreadsT, 1)
rollout_tile_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    constexpr int WC = WCP;
    constexpr int CL = WC < 8 ? WC : 8;           // candidates per lane (8; 4 for 4-candidate batches)
    constexpr int CG = WC / CL;                   // candidate groups per warp
    constexpr int RG = 32 / CG;                   // row groups per warp
    constexpr int TR = D / RG;                    // rows per lane
    constexpr int QR = TR / 4;                    // float4 groups of rows per lane
    constexpr int NZ = CL / 4;                    // float4 groups of candidates per lane
    static_assert(CL == 4 || CL == 8, "lane tile: 4 or 8 candidates");
    constexpr int kTileThreads = kTileThreadsT;
    static_assert(TR % 4 == 0, "lane tile");
    static_assert(D == 64 || D == 128, "tile kernel: D in {64, 128}");
    extern __shared__ __align__(16) float smem[];
    float *sK = smem;                             // (D+M) x D
    __shared__ float sz0[D];
    __shared__ unsigned s_batch[kTileWarps];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float *zw = smem + (D + M) * D + warp * (D + M) * WC;     // this warp's (D+M) x 32 tile
    for (int i = tid; i < (D + M) * D / 4; i += kTileThreads)
        reinterpret_cast<float4 *>(sK)[i] = reinterpret_cast<const float4 *>(cfg.KTa)[i];
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const int H = (MODE == MODE_TICK) ? cfg.H : a.H;
    const long long ncand = (MODE == MODE_TICK) ? cfg.shard_count : a.ncand;
    const bool shared_x0 = (MODE == MODE_TICK) || a.x0_count == 1;

    float u_h[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    bool inputs_ok = true;
    if (MODE == MODE_TICK) {
        inputs_ok = finite_inputs(cfg, x0p, uup);
        clamp_user(cfg, uup, u_h);
    }
    if (shared_x0) {
        for (int f = tid; f < D; f += kTileThreads) sz0[f] = lift_feature(cfg, f, x0p);
    }
    __syncthreads();

    constexpr int NB = kMaxN;
    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const int nphys = cfg.annulus ? (nbox > 2 ? nbox : 2) : nbox;      // internal dims the safe test reads
    const bool dump = (MODE == MODE_BATCH) && a.dump_kind != MPMI_DUMP_NONE;
    const int J = dump ? (a.dump_kind == MPMI_DUMP_PHYS ? cfg.n : cfg.d) : 0;
    const int rg = lane / CG, cg = lane % CG;
    const float *kp = sK + rg * 4;                // rows  q*(4 RG) + rg*4 + e,  q < QR
    const float *zp = zw + cg * 4;                // cands q*(4 CG) + cg*4 + e,  q < 2
    const int col = lane % WC;                    // the candidate this lane fills and tests (lanes >= WC mirror)
    // second pass of the verified tensor-core tick / batch (kernel_args.cuh): walk the deferral lists, longest-lived first
    const bool rc = a.recheck_mode != 0;
    int rc_count[kRecheckBuckets], rc_total = 0;
#pragma unroll
    for (int b = 0; b < kRecheckBuckets; b++) { rc_count[b] = rc ? (int)a.recheck_count[b] : 0; rc_total += rc_count[b]; }
    const long long nbatch = ((rc ? (long long)rc_total : ncand) + WC - 1) / WC;

    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;

    for (long long round = 0;; round++) {
        // ---- next batch of WC candidates for this warp (dynamic: warps that exit early take more).
        // Second pass: the lists are sorted longest-lived first and most deferred candidates are short-lived.  Only FOUR warps of
        // the CTA work, one per SM sub-partition (with the 16-fold unrolled column loop one warp keeps its sub-partition's FMA pipe
        // busy; more warps only stretch the full-horizon batches, which set the length of the pass), each starting with one of
        // the 4 * gridDim longest batches and fetching every further one first come, first served -- longest processing time first.
        // (Measured on C5, 4.8 % of the candidates.  8-candidate batches: all 16 warps first-come 1.3 ms; all dealt out statically
        // 0.52 ms; static head + first-come tail, sub-partition 0 left to its head batch, 13 warps 0.37 ms.  4-candidate batches,
        // which halve a full-horizon batch's chain: 13 warps 0.33 ms; 16 / 12 / 8 / 4 warps first-come 0.31 / 0.30 / 0.28 / 0.275 ms.)
        const int rc_warps = (a.recheck_mode >> 8) ? (a.recheck_mode >> 8) : 4;     // (MPMI_RC_WARPS: measurement)
        if (rc && warp >= rc_warps) break;
        const bool fixed = rc && round == 0;
        if (lane == 0) s_batch[warp] = fixed ? 0u : atomicAdd(a.work, 1u);
        __syncwarp();
        const long long batch = fixed ? (long long)blockIdx.x + (long long)gridDim.x * warp
                                      : (long long)s_batch[warp] + (rc ? (long long)rc_warps * gridDim.x : 0LL);
        __syncwarp();
        if (batch >= nbatch) break;

        // ---- a1 + a2: lane i fills column i of the warp tile
        // ordered walk: the ragged last batch holds the injected u_h (often the full horizon): first, not last
        const long long wbatch = (MODE == MODE_TICK && a.perm) ? (batch == 0 ? nbatch - 1 : batch - 1) : batch;
        long long li = wbatch * WC + col;
        if (MODE == MODE_TICK && a.perm && li < a.nsamp) li = a.perm[li];
        if (rc) {                                          // slot li of the concatenated lists -> candidate
            int p = (int)li;
            long long hit = ncand;
#pragma unroll
            for (int b = 0; b < kRecheckBuckets; b++) {
                if (p >= 0 && p < rc_count[b]) hit = (long long)a.recheck[(long long)b * ncand + p];
                p -= rc_count[b];                          // negative once the slot has been found
            }
            li = hit;
        }
        bool alive = li < ncand && inputs_ok;
        int steps = 0;
        {
            float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
            if (li < ncand) {
                if (MODE == MODE_BATCH && a.U) {
                    for (int j = 0; j < cfg.m; j++) u[j] = a.U[li * cfg.m + j];
                } else {
                    sample_u(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, tick, u_h, u);
                }
            }
#pragma unroll
            for (int j = 0; j < M; j++) zw[(D + j) * WC + col] = u[j];
            if (shared_x0) {
                for (int c = 0; c < D; c++) zw[c * WC + col] = sz0[c];
            } else {
                float x[kMaxN];
                const long long row = li < ncand ? li : 0;
                for (int j = 0; j < kMaxN; j++) x[j] = j < cfg.n ? a.x0[row * cfg.n + j] : 0.f;
                for (int c = 0; c < D; c++) zw[c * WC + col] = lift_feature(cfg, c, x);
            }
        }
        __syncwarp();

        // ---- a3 + a4: horizon loop
        int k = 0;
        for (; k < H; k++) {
            if (!__any_sync(0xffffffffu, alive)) break;

            float2 acc[TR][CL / 2];
#pragma unroll
            for (int r = 0; r < TR; r++)
#pragma unroll
                for (int q = 0; q < CL / 2; q++) acc[r][q] = make_float2(0.f, 0.f);

            // (second pass, WC = 8: few warps per sub-partition, so the shared-memory loads of the next columns must be in flight
            // under the FFMA2s of this one: deeper unrolling.  Measured on C5: unroll 2 / 8 / 16 / 32 -> 0.49 / 0.40 / 0.37 / 0.36 ms)
#pragma unroll (WC <= 8 ? 16 : 2)
            for (int cc = 0; cc < D + M; cc++) {                // descending column order: see rollout_reg.cuh
                const int c = D + M - 1 - cc;
                float kr[TR];
#pragma unroll
                for (int q = 0; q < QR; q++) {
                    const float4 v = *reinterpret_cast<const float4 *>(kp + c * D + q * (4 * RG));
                    kr[4 * q] = v.x; kr[4 * q + 1] = v.y; kr[4 * q + 2] = v.z; kr[4 * q + 3] = v.w;
                }
                float2 zc[CL / 2];
#pragma unroll
                for (int q = 0; q < NZ; q++) {
                    const float4 v = *reinterpret_cast<const float4 *>(zp + c * WC + q * (4 * CG));
                    zc[2 * q] = make_float2(v.x, v.y);
                    zc[2 * q + 1] = make_float2(v.z, v.w);
                }
#pragma unroll
                for (int r = 0; r < TR; r++)
#pragma unroll
                    for (int q = 0; q < CL / 2; q++) fma2_bcast(acc[r][q], kr[r], zc[q]);
            }
            __syncwarp();                                  // every lane has finished reading Zw
#pragma unroll
            for (int r = 0; r < TR; r++) {
                const int row = (r >> 2) * (4 * RG) + rg * 4 + (r & 3);
#pragma unroll
                for (int q = 0; q < NZ; q++)
                    *reinterpret_cast<float4 *>(zw + row * WC + q * (4 * CG) + cg * 4) =
                        make_float4(acc[r][2 * q].x, acc[r][2 * q].y, acc[r][2 * q + 1].x, acc[r][2 * q + 1].y);
            }
            __syncwarp();

            if (NOISE) {
                // Algorithm 2 l.5: + z_i: sigma * eps on the physical rows of candidate `col`, before isSafe
                if (lane < WC) {
                    const long long gi = (MODE == MODE_TICK ? cfg.shard_begin : 0) + li;
                    for (int q = 0; 4 * q < cfg.n; q++) {
                        float g[4];
                        noise4(cfg, gi, k, q, tick, g);
                        for (int j = 0; j < cfg.n; j++) {            // internal dim j = original dim perm[j]
                            const int p = cfg.perm[j];
                            if ((p >> 2) == q) {
                                const float e = (p & 3) == 0 ? g[0] : (p & 3) == 1 ? g[1] : (p & 3) == 2 ? g[2] : g[3];
                                zw[j * WC + col] = __fmaf_rn(cfg.noise_sigma, e, zw[j * WC + col]);
                            }
                        }
                    }
                }
                __syncwarp();
            }
            float x[NB];
#pragma unroll
            for (int j = 0; j < NB; j++) x[j] = j < nphys ? zw[j * WC + col] : 0.f;
            const bool was_alive = alive;
            const bool ok = safe_check<NB>(cfg, x, nbox);
            alive = was_alive && ok;
            steps += alive ? 1 : 0;
            if (dump && li < ncand && lane < WC) {
                for (int j = 0; j < D; j++) {
                    const int row = j < cfg.n ? (int)cfg.perm[j] : j;
                    if (row < J)
                        a.traj[((long long)k * J + row) * ncand + li] = was_alive ? zw[j * WC + col] : __int_as_float(0x7fc00000);
                }
            }
        }
        if (dump && li < ncand && lane < WC) {
            for (; k < H; k++)
                for (int row = 0; row < J; row++)
                    a.traj[((long long)k * J + row) * ncand + li] = __int_as_float(0x7fc00000);
        }

        if (MODE == MODE_BATCH) {
            if (li < ncand && lane < WC) {
                a.steps[li] = steps;
                if (a.safe) a.safe[li] = steps == H ? 1 : 0;
            }
        } else if (li < ncand && inputs_ok && lane < WC) {  // a5: this candidate's key
            if (a.steps) a.steps[li] = steps;               // mpmi_step_trace
            const bool safe = steps == H;
            float d2 = 0.f;
#pragma unroll
            for (int j = 0; j < M; j++) {
                const float df = __fsub_rn(zw[(D + j) * WC + col], u_h[j]);
                d2 = __fmaf_rn(df, df, d2);
            }
            const unsigned long long kk = make_key(safe, d2, H, steps, cfg.shard_begin + li);
            key = kk < key ? kk : key;
            n_safe += safe ? 1u : 0u;
            n_exec += (unsigned)(steps + 1 < H ? steps + 1 : H);
        }
        __syncwarp();
    }

    if (MODE == MODE_BATCH) {
        // the last CTA to finish re-arms the work counter for the next launch
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            if (atomicAdd(&a.st->ticket, 1u) == gridDim.x - 1) {
                *a.work = 0u; a.st->ticket = 0u;
                if (rc) for (int b = 0; b <= kRecheckBuckets; b++) a.recheck_count[b] = 0u;
                __threadfence();
            }
        }
        return;
    }
    // ---- a6 + a7
    block_select_and_finalise<kTileWarps>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq, a.work, false,
                                          rc ? a.recheck_count : nullptr, kRecheckBuckets, a.deferred_out);
}

}  // namespace mpmi
