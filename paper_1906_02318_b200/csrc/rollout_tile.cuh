// rollout_tile.cuh -- CTA-tile rollout kernel for padded lifted dim D in {64, 128} (a1-a7, a9).
//
// A lifted state of 128 floats cannot be thread-private, so one CTA keeps a tile of NC = 256
// candidates on chip for the whole horizon: Z[c][i] (c < D+M rows: lifted state, then the
// candidate's input u as M extra rows; i < NC candidates) and the augmented transposed model
// KTa[c][r] both live in shared memory (D = 128: 66 KB + 132 KB).  One step is the dense
// contraction Z'[r][i] = sum_c KTa[c][r] * Z[c][i], register-blocked like an SGEMM: every thread
// owns 8 rows x TC candidates as float2 accumulators and advances two candidates per FFMA2 with
// the model value broadcast to both halves -- D*(D+M) fp32 FMAs per candidate-step, the
// algorithmic count of z' = K z + B u.  After write-back thread i tests
// candidate i against the safe set and the CTA leaves the horizon loop when none of
// its candidates is alive.
#pragma once
#include "mpmi_device.cuh"
#include "rollout_reg.cuh"

namespace mpmi {

template <int D, int M>
constexpr int tile_smem_bytes() { return ((D + M) * D + (D + M) * kTileNC) * 4; }

template <int D, int M, int MODE>
__global__ void __launch_bounds__(kTileThreads, 1)
rollout_tile_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    constexpr int NC = kTileNC;
    constexpr int TYN = D / 8;                    // threads along rows
    constexpr int TXN = kTileThreads / TYN;       // threads along candidates
    constexpr int TC = NC / TXN;                  // candidates per thread (16 for D=128, 8 for D=64)
    constexpr int QC = TC / 4;                    // float4 groups of candidates per thread
    static_assert(TC % 4 == 0 && TYN * TXN == kTileThreads, "tile shape");
    extern __shared__ __align__(16) float smem[];
    float *sK = smem;                             // (D+M) x D
    float *sZ = smem + (D + M) * D;               // (D+M) x NC
    __shared__ float sz0[D];

    const int tid = threadIdx.x;
    const int ty = tid / TXN, tx = tid % TXN;
    for (int i = tid; i < (D + M) * D / 4; i += kTileThreads)
        reinterpret_cast<float4 *>(sK)[i] = reinterpret_cast<const float4 *>(cfg.KTa)[i];
    const unsigned long long tick = a.tick_ptr ? *a.tick_ptr : a.tick_val;
    const int H = (MODE == MODE_TICK) ? cfg.H : a.H;
    const long long ncand = (MODE == MODE_TICK) ? cfg.shard_count : a.ncand;
    const bool shared_x0 = (MODE == MODE_TICK) || a.x0_count == 1;

    float u_h[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    bool inputs_ok = true;
    if (MODE == MODE_TICK) {
        inputs_ok = finite_inputs(cfg, a.x0, a.u_user);
        clamp_user(cfg, a.u_user, u_h);
    }
    if (shared_x0) {
        for (int f = tid; f < D; f += kTileThreads) sz0[f] = lift_feature(cfg, f, a.x0);
    }
    __syncthreads();

    // ---- a1 + a2: thread i fills column i of the tile ----------------------------------------------
    long long li = (long long)blockIdx.x * NC + tid;            // kTileThreads == NC
    if (MODE == MODE_TICK && a.perm && li < a.nsamp) li = a.perm[li];   // spatially ordered walk
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
        for (int j = 0; j < M; j++) sZ[(D + j) * NC + tid] = u[j];
        if (shared_x0) {
            for (int c = 0; c < D; c++) sZ[c * NC + tid] = sz0[c];
        } else {
            float x[kMaxN];
            const long long row = li < ncand ? li : 0;
            for (int j = 0; j < kMaxN; j++) x[j] = j < cfg.n ? a.x0[row * cfg.n + j] : 0.f;
            for (int c = 0; c < D; c++) sZ[c * NC + tid] = lift_feature(cfg, c, x);
        }
    }
    __syncthreads();

    // ---- a3 + a4: horizon loop ------------------------------------------------------------------------
    constexpr int NB = kMaxN;
    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const bool dump = (MODE == MODE_BATCH) && a.dump_kind != MPMI_DUMP_NONE;
    const int J = dump ? (a.dump_kind == MPMI_DUMP_PHYS ? cfg.n : cfg.d) : 0;
    const float *kp = sK + ty * 4;
    const float *zp = sZ + tx * 4;
    int k = 0;
    for (; k < H; k++) {
        if (!__syncthreads_or(alive ? 1 : 0)) break;

        float2 acc[8][TC / 2];
#pragma unroll
        for (int r = 0; r < 8; r++)
#pragma unroll
            for (int q = 0; q < TC / 2; q++) acc[r][q] = make_float2(0.f, 0.f);

#pragma unroll 2
        for (int c = 0; c < D + M; c++) {
            const float4 k0 = *reinterpret_cast<const float4 *>(kp + c * D);
            const float4 k1 = *reinterpret_cast<const float4 *>(kp + c * D + D / 2);
            const float kr[8] = {k0.x, k0.y, k0.z, k0.w, k1.x, k1.y, k1.z, k1.w};
            float2 zc[TC / 2];
#pragma unroll
            for (int q = 0; q < QC; q++) {
                const float4 zv = *reinterpret_cast<const float4 *>(zp + c * NC + q * 4 * TXN);
                zc[2 * q] = make_float2(zv.x, zv.y);
                zc[2 * q + 1] = make_float2(zv.z, zv.w);
            }
#pragma unroll
            for (int r = 0; r < 8; r++)
#pragma unroll
                for (int q = 0; q < TC / 2; q++)
                    acc[r][q] = __ffma2_rn(make_float2(kr[r], kr[r]), zc[q], acc[r][q]);
        }
        __syncthreads();                                   // every thread has finished reading Z
#pragma unroll
        for (int r = 0; r < 8; r++) {
            const int row = (r < 4 ? 0 : D / 2) + ty * 4 + (r & 3);
#pragma unroll
            for (int q = 0; q < QC; q++)
                *reinterpret_cast<float4 *>(sZ + row * NC + q * 4 * TXN + tx * 4) =
                    make_float4(acc[r][2 * q].x, acc[r][2 * q].y, acc[r][2 * q + 1].x, acc[r][2 * q + 1].y);
        }
        __syncthreads();

        float x[NB];
#pragma unroll
        for (int j = 0; j < NB; j++) x[j] = sZ[j * NC + tid];
        const bool was_alive = alive;
        const bool ok = safe_check<NB>(cfg, x, nbox);
        alive = was_alive && ok;
        steps += alive ? 1 : 0;
        if (dump && li < ncand) {
            for (int j = 0; j < D; j++) {
                const int row = j < cfg.n ? (int)cfg.perm[j] : j;
                if (row < J)
                    a.traj[((long long)k * J + row) * ncand + li] = was_alive ? sZ[j * NC + tid] : __int_as_float(0x7fc00000);
            }
        }
    }
    if (dump && li < ncand) {
        for (; k < H; k++)
            for (int row = 0; row < J; row++)
                a.traj[((long long)k * J + row) * ncand + li] = __int_as_float(0x7fc00000);
    }

    if (MODE == MODE_BATCH) {
        if (li < ncand) {
            a.steps[li] = steps;
            if (a.safe) a.safe[li] = steps == H ? 1 : 0;
        }
        return;
    }

    // ---- a5-a7 ---------------------------------------------------------------------------------------
    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;
    if (li < ncand && inputs_ok) {
        const bool safe = steps == H;
        float d2 = 0.f;
#pragma unroll
        for (int j = 0; j < M; j++) {
            const float df = __fsub_rn(sZ[(D + j) * NC + tid], u_h[j]);
            d2 = __fmaf_rn(df, df, d2);
        }
        key = make_key(safe, d2, H, steps, cfg.shard_begin + li);
        n_safe = safe ? 1u : 0u;
        n_exec = (unsigned)(steps + 1 < H ? steps + 1 : H);
    }
    block_select_and_finalise<kTileThreads / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial);
}

}  // namespace mpmi
