// rollout_reg.cuh -- register-resident rollout kernel for padded lifted dim D <= 32 (a1-a7, a9).
//
// Each thread owns 2P candidates; candidate pair p is packed into the two halves of float2
// registers so that one FFMA2 (Blackwell packed fp32 FMA, fma.rn.f32x2) advances one row of two
// candidates: a[p][r] += K[r][c] * z[p][c], the K value broadcast to both halves.  The model, as the
// augmented transpose KTa[c][r] (c < D: K[r][c]; c >= D: B[r][c-D]), sits in __constant__ memory and
// enters FFMA2 as a uniform-register operand (kernel_args.cuh), so the horizon loop issues no
// load/store-unit instruction at all (shared memory + LDS.128 remains as the KC = false variant); the candidate's
// input u is appended to z as "state" D..D+M-1, so one step executes exactly D*(D+M) fp32 FMAs per
// candidate -- the algorithmic count of z' = K z + B u.
// The safe set is tested after every step; a warp leaves the horizon loop when none
// of its candidates is alive.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"

namespace mpmi {

// model slots in constant memory (one copy of this array per translation unit: no relocatable device code; the
// host fills the slot of a context in every translation unit whose kernels it launches, see inst_reg.cu)
static __constant__ float4 c_model[kModelSlots][kModelFloats / 4];

template <int D, int P>
constexpr int reg_min_blocks() { return (D * P >= 32) ? 3 : 4; }

// KC = true: model values from the constant bank (slot a.kslot of c_model), the choice for grids that fill the machine;
// KC = false: staged in shared memory and read with warp-uniform LDS.128 -- better when an SM holds only one or two
// warps, which cannot hide the constant-cache misses of a 4.3 KB model (measured crossover: ~2^19 candidates at D = 32).
// RC = true: second pass of the verified tensor-core tick (kernel_args.cuh): the CTAs walk the deferral lists (longest-lived
// first) in blocks of 2P * blockDim candidates.  The pass is launched as 4 one-warp CTAs per SM, one per sub-partition (a
// warp of FFMA2 saturates its sub-partition's FMA pipe on its own); CTA x starts with block x and fetches every further
// block from a counter (a.recheck_count[kRecheckBuckets]), so a warp whose candidates stop early takes more, and the
// long-lived blocks at the head of the lists end up on different sub-partitions.  The last CTA finalises the tick.
template <int D, int M, int P, int MODE, bool NOISE = false, bool KC = true, bool RC = false>
__global__ void __launch_bounds__(kRegBlock, reg_min_blocks<D, P>())
rollout_reg_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    static_assert(!RC || MODE == MODE_TICK, "the second pass is a tick kernel");
    constexpr int S = 2 * P;                 // candidates per thread
    constexpr int NB = D < kMaxN ? D : kMaxN;
    __shared__ __align__(16) float sK[KC ? 4 : (D + M) * D];
    if (!KC) {
        for (int i = threadIdx.x; i < (D + M) * D / 4; i += blockDim.x)
            reinterpret_cast<float4 *>(sK)[i] = reinterpret_cast<const float4 *>(cfg.KTa)[i];
    }
    const unsigned sbase = (unsigned)__cvta_generic_to_shared(sK);
    __shared__ float sz0[D];
    __shared__ float sstage[MODE == MODE_BATCH ? D * kRegBlock : 1];

    const int tid = threadIdx.x, bdim = blockDim.x;
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
        for (int f = tid; f < D; f += bdim) sz0[f] = lift_feature(cfg, f, x0p);
    }
    __syncthreads();

    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;
    int rc_count[kRecheckBuckets], rc_total = 0;
#pragma unroll
    for (int b = 0; b < kRecheckBuckets; b++) { rc_count[b] = RC ? (int)a.recheck_count[b] : 0; rc_total += rc_count[b]; }
  for (long long blk = blockIdx.x; !RC || blk * (2 * P * (long long)blockDim.x) < rc_total;) {
    // ---- a1 + a2: candidates of this thread ------------------------------------------------------
    float2 z[P][D + M];
    long long li[S];
    bool alive[S];
    int steps[S];
#pragma unroll
    for (int s = 0; s < S; s++) {
        // the two halves of a register pair are ADJACENT candidates (2*tid, 2*tid+1): dumps store float2
        li[s] = blk * (S * bdim) + (s >> 1) * (2 * bdim) + 2 * tid + (s & 1);
        if (MODE == MODE_TICK && !RC && a.perm && li[s] < a.nsamp) li[s] = a.perm[li[s]];   // spatially ordered walk
        if (RC) {                                                                     // second pass of the verified tensor-core tick
            int p = (int)li[s];                                                       // slot p of the concatenated lists
            long long hit = ncand;
#pragma unroll
            for (int b = 0; b < kRecheckBuckets; b++) {
                if (p >= 0 && p < rc_count[b]) hit = (long long)a.recheck[(long long)b * ncand + p];
                p -= rc_count[b];                                                     // negative once the slot has been found
            }
            li[s] = hit;
        }
        const bool valid = li[s] < ncand && inputs_ok;
        alive[s] = valid;
        steps[s] = 0;
        float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
        if (li[s] < ncand) {
            if (MODE == MODE_BATCH && a.U) {
#pragma unroll
                for (int j = 0; j < M; j++) u[j] = a.U[li[s] * cfg.m + (j < cfg.m ? j : 0)] * (j < cfg.m ? 1.f : 0.f);
            } else {
                sample_u(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li[s], tick, u_h, u);
            }
        }
#pragma unroll
        for (int j = 0; j < M; j++) {
            if (s & 1) z[s >> 1][D + j].y = u[j]; else z[s >> 1][D + j].x = u[j];
        }
        if (shared_x0) {
#pragma unroll
            for (int c = 0; c < D; c++) {
                if (s & 1) z[s >> 1][c].y = sz0[c]; else z[s >> 1][c].x = sz0[c];
            }
        } else {
            // per-candidate x0 (benchmark entry only): lift through a private shared-memory column so
            // that the lift code is not replicated D times
            float x[kMaxN];
            const long long row = li[s] < ncand ? li[s] : 0;
            for (int j = 0; j < kMaxN; j++) x[j] = j < cfg.n ? a.x0[row * cfg.n + j] : 0.f;
#pragma unroll 1
            for (int c = 0; c < D; c++) sstage[c * kRegBlock + tid] = lift_feature(cfg, c, x);
#pragma unroll
            for (int c = 0; c < D; c++) {
                const float v = sstage[c * kRegBlock + tid];
                if (s & 1) z[s >> 1][c].y = v; else z[s >> 1][c].x = v;
            }
        }
    }

    // ---- a3 + a4: horizon loop --------------------------------------------------------------------
    const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
    const bool dump = (MODE == MODE_BATCH) && a.dump_kind != MPMI_DUMP_NONE;
    const int J = dump ? (a.dump_kind == MPMI_DUMP_PHYS ? cfg.n : cfg.d) : 0;
    const bool vec2 = dump && (ncand % 2 == 0) && ((reinterpret_cast<unsigned long long>(a.traj) & 7ull) == 0);
    const bool dump_fast = vec2 && ((blk + 1) * (S * bdim) <= ncand) && ((long long)J * ncand < (1ll << 31));
    const bool dump_full = J == D;           // lifted dump of an unpadded model: every row is stored
    unsigned dump_row[NB];                   // original row of internal row j (only the first n are permuted)
#pragma unroll
    for (int j = 0; j < NB; j++) dump_row[j] = (dump && j < cfg.n) ? (unsigned)cfg.perm[j] : (unsigned)j;
    int k = 0;
    for (; k < H; k++) {
        bool any = false;
#pragma unroll
        for (int s = 0; s < S; s++) any = any || alive[s];
        if (!__any_sync(0xffffffffu, any)) break;

        float2 acc[P][D];
#pragma unroll
        // Columns run in DESCENDING order, the physical dims (internal columns 0..n-1) last: a product's rounding error is
        // re-rounded by every FMA after it, and for a model close to the identity on the physical block (small time step) the
        // dominant product of a physical row is its diagonal one -- it now passes through <= n roundings instead of D + M
        // (the per-column weights of csrc/bound.cuh follow this order).
        for (int cc = 0; cc < D + M; cc++) {
            const int c = D + M - 1 - cc;
#pragma unroll
            for (int r = 0; r < D; r += 4) {
                const float4 kv = KC ? c_model[a.kslot][(c * D + r) / 4]
                                     : lds128(sbase + (c * D + r) * 4);
#pragma unroll
                for (int p = 0; p < P; p++) {
                    const float2 zc = z[p][c];
                    if (cc == 0) {
                        mul2_bcast(acc[p][r + 0], kv.x, zc); mul2_bcast(acc[p][r + 1], kv.y, zc);
                        mul2_bcast(acc[p][r + 2], kv.z, zc); mul2_bcast(acc[p][r + 3], kv.w, zc);
                    } else {
                        fma2_bcast(acc[p][r + 0], kv.x, zc); fma2_bcast(acc[p][r + 1], kv.y, zc);
                        fma2_bcast(acc[p][r + 2], kv.z, zc); fma2_bcast(acc[p][r + 3], kv.w, zc);
                    }
                }
            }
        }
#pragma unroll
        for (int p = 0; p < P; p++)
#pragma unroll
            for (int r = 0; r < D; r++) z[p][r] = acc[p][r];

        if (NOISE) {
            // Algorithm 2 l.5: x_p <- f(x_p, xi(i)) + z_i: sigma * eps on the physical rows, before isSafe
#pragma unroll
            for (int s = 0; s < S; s++) {
                const long long gi = (MODE == MODE_TICK ? cfg.shard_begin : 0) + li[s];
                float g[NB];                                   // eps of the ORIGINAL dims
#pragma unroll
                for (int q = 0; 4 * q < NB; q++) {
                    float g4[4] = {0.f, 0.f, 0.f, 0.f};
                    if (4 * q < cfg.n) noise4(cfg, gi, k, q, tick, g4);
#pragma unroll
                    for (int e = 0; e < 4; e++) if (4 * q + e < NB) g[4 * q + e] = g4[e];
                }
#pragma unroll
                for (int j = 0; j < NB; j++) {
                    if (j < cfg.n) {                           // internal dim j = original dim perm[j] (warp-uniform index)
                        const float e = g[cfg.perm[j]];
                        if (s & 1) z[s >> 1][j].y = __fmaf_rn(cfg.noise_sigma, e, z[s >> 1][j].y);
                        else       z[s >> 1][j].x = __fmaf_rn(cfg.noise_sigma, e, z[s >> 1][j].x);
                    }
                }
            }
        }
        bool was_alive[S];
#pragma unroll
        for (int s = 0; s < S; s++) {
            float x[NB];
#pragma unroll
            for (int j = 0; j < NB; j++) x[j] = (s & 1) ? z[s >> 1][j].y : z[s >> 1][j].x;
            was_alive[s] = alive[s];
            const bool ok = safe_check<NB>(cfg, x, nbox);
            alive[s] = was_alive[s] && ok;
            steps[s] += alive[s] ? 1 : 0;
        }
        if (dump && dump_fast) {
            // a9 fast path (whole CTA in range, aligned, one step of the dump < 2^31 floats): no per-store
            // branches; address = per-pair pointer + warp-uniform row offset (one IMAD.WIDE per store).
            // Row j is stored iff j < J (the internal order permutes only the first n rows among themselves).
            const float qnan = __int_as_float(0x7fc00000);
            const unsigned long long step_base = reinterpret_cast<unsigned long long>(a.traj + (long long)k * J * ncand);
            const unsigned nc32 = (unsigned)ncand;
#pragma unroll
            for (int p = 0; p < P; p++) {
                const unsigned long long qp = step_base + 4ull * (unsigned)li[2 * p];
                const bool a0 = was_alive[2 * p], a1 = was_alive[2 * p + 1];
                if (dump_full) {
#pragma unroll
                    for (int j = 0; j < D; j++) {
                        float2 v = z[p][j];
                        v.x = a0 ? v.x : qnan;
                        v.y = a1 ? v.y : qnan;
                        stg64_off(qp, (j < NB ? dump_row[j] : (unsigned)j) * nc32, v);
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < D; j++) {
                        float2 v = z[p][j];
                        v.x = a0 ? v.x : qnan;
                        v.y = a1 ? v.y : qnan;
                        stg64_off_if(qp, (j < NB ? dump_row[j] : (unsigned)j) * nc32, v, j < J);
                    }
                }
            }
        } else if (dump) {
            // a9: traj[(k*J + j)*Ncand + i], candidate fastest.  A pair is two adjacent candidates, so one
            // 8-byte store per (pair, row): a warp writes 256 contiguous bytes per instruction.
            const float qnan = __int_as_float(0x7fc00000);
            float *step_base = a.traj + (long long)k * J * ncand;
#pragma unroll
            for (int p = 0; p < P; p++) {
                const long long l0 = li[2 * p];
                const bool v0 = l0 < ncand, v1 = l0 + 1 < ncand;
#pragma unroll
                for (int j = 0; j < D; j++) {
                    const int row = j < cfg.n ? (int)cfg.perm[j < kMaxN ? j : 0] : j;
                    if (row < J && v0) {
                        float2 v = z[p][j];
                        v.x = was_alive[2 * p] ? v.x : qnan;
                        v.y = was_alive[2 * p + 1] ? v.y : qnan;
                        float *q = step_base + (long long)row * ncand + l0;
                        if (vec2 && v1) *reinterpret_cast<float2 *>(q) = v;
                        else { q[0] = v.x; if (v1) q[1] = v.y; }
                    }
                }
            }
        }
    }
    if (dump) {                              // states after the warp stopped: NaN
        for (; k < H; k++)
#pragma unroll
            for (int s = 0; s < S; s++)
                if (li[s] < ncand)
                    for (int row = 0; row < J; row++)
                        a.traj[((long long)k * J + row) * ncand + li[s]] = __int_as_float(0x7fc00000);
    }

    if (MODE == MODE_BATCH) {
#pragma unroll
        for (int s = 0; s < S; s++) {
            if (li[s] < ncand) {
                a.steps[li[s]] = steps[s];
                if (a.safe) a.safe[li[s]] = steps[s] == H ? 1 : 0;
            }
        }
        return;
    }

    // ---- a5-a7: key, argmin, finalise -------------------------------------------------------------
#pragma unroll
    for (int s = 0; s < S; s++) {
        if (a.steps && li[s] < ncand) a.steps[li[s]] = steps[s];   // mpmi_step_trace: per-candidate steps of THIS tick kernel
        if (li[s] < ncand && inputs_ok) {
            const bool safe = steps[s] == H;
            float d2 = 0.f;
#pragma unroll
            for (int j = 0; j < M; j++) {
                const float uj = (s & 1) ? z[s >> 1][D + j].y : z[s >> 1][D + j].x;
                const float df = __fsub_rn(uj, u_h[j]);
                d2 = __fmaf_rn(df, df, d2);
            }
            const unsigned long long kk = make_key(safe, d2, H, steps[s], cfg.shard_begin + li[s]);
            key = kk < key ? kk : key;
            n_safe += safe ? 1u : 0u;
            n_exec += (unsigned)(steps[s] + 1 < H ? steps[s] + 1 : H);
        }
    }
    if (!RC) break;
    // next block of the lists: first come, first served (blockDim == 32: one warp, no block-level hand-off needed)
    unsigned nxt = 0;
    if (tid == 0) nxt = atomicAdd(a.recheck_count + kRecheckBuckets, 1u);
    blk = (long long)gridDim.x + (long long)__shfl_sync(0xffffffffu, nxt, 0);
  }
    block_select_and_finalise<kRegBlock / 32>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq, nullptr, false,
                                              RC ? a.recheck_count : nullptr, kRecheckBuckets, a.deferred_out);
}

}  // namespace mpmi
