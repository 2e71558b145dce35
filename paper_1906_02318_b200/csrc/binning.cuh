// binning.cuh -- spatial ordering of the Philox candidates before the rollout.
//
// Algorithm 2 stops a candidate at its first unsafe state.  On a SIMT machine that
// only saves time when the candidates of one warp / CTA stop together.  Trajectories are affine in u,
// so candidates that are close in the input box share their fate; Philox hands them out in random
// order.  These two kernels counting-sort the candidate INDICES of one tick by the cell of the input
// box they fall in (cell = the top bits of the Philox words, row-major over the input dimensions):
//   bin_hist_kernel    histogram of cells (one RED per candidate) + exclusive scan by the last CTA
//   bin_scatter_kernel perm[cursor[cell]++] = local candidate index
//   bin_predict_kernel (life-time order, below) replaces bin_hist_kernel: keys + histogram + scan
// The rollout kernel then walks perm, so a warp owns candidates of the same cell.  The candidate SET,
// every key and hence the result are unchanged (keys carry the original index).
// Life-time order (persistent tile kernels, d > 32): in a 3-D input box cubic cells leave a tile of 128 candidates
// running 0.65 N*H tile-steps for 0.46 N*H candidate-steps; there the cell is instead the first-violation step
// PREDICTED by the affine-in-u form x_k = a_k + G_k u (rollout_affine.cuh, n*m FMAs per step), longest first, so
// that the candidates of a tile stop together.  The prediction only schedules: the dense rollout decides.
#pragma once
#include "mpmi_device.cuh"

namespace mpmi {

struct BinArgs {
    unsigned long long tick_val;
    long long nsamp;          // sampled candidates of this shard (the injected u_h is not binned)
    int bits[kMaxM];          // cell bits per input dimension
    int ncells;
    int *hist;                // ncells, zero on entry, zero on exit
    int *cursor;              // ncells, written by the scan
    int *perm;                // nsamp
    unsigned *ticket;
    int *keys;                // life-time order: predicted steps of the local candidates (cell = H - steps), or null
    int H;
};

__device__ __forceinline__ int cell_of(const DevCfg &cfg, const BinArgs &b, long long gi, unsigned long long tick) {
    if (b.keys) {                                            // predicted life time, longest first
        const int st = b.keys[gi - cfg.shard_begin];
        return b.H - (st < 0 ? 0 : st > b.H ? b.H : st);
    }
    unsigned w[4];
    philox4x32_10((unsigned)gi, (unsigned)((unsigned long long)gi >> 32), (unsigned)tick, (unsigned)(tick >> 32),
                  cfg.seed_lo, cfg.seed_hi, w);
    int cell = 0;
#pragma unroll
    for (int j = 0; j < kMaxM; j++)
        if (j < cfg.m && b.bits[j] > 0) cell = (cell << b.bits[j]) | (int)(w[j] >> (32 - b.bits[j]));
    return cell;
}

// exclusive scan of hist -> cursor by the last CTA to arrive (256 threads); hist is cleared for the next tick
__device__ __forceinline__ void bin_scan_last_cta(const BinArgs &b) {
    __shared__ bool last;
    __shared__ int warp_tot[8];
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(b.ticket, 1u) == gridDim.x - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    // exclusive scan of hist -> cursor by this (last) CTA; hist is cleared for the next tick
    int carry = 0;
    for (int base = 0; base < b.ncells; base += 256 * 4) {
        int v[4], s = 0;
        const int c0 = base + threadIdx.x * 4;
#pragma unroll
        for (int q = 0; q < 4; q++) {
            v[q] = c0 + q < b.ncells ? __ldcg(&b.hist[c0 + q]) : 0;
            if (c0 + q < b.ncells) b.hist[c0 + q] = 0;
            s += v[q];
        }
        int incl = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if ((threadIdx.x & 31) >= o) incl += t;
        }
        if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = incl;
        __syncthreads();
        int woff = 0, tot = 0;
#pragma unroll
        for (int wi = 0; wi < 8; wi++) {
            if (wi < (int)(threadIdx.x >> 5)) woff += warp_tot[wi];
            tot += warp_tot[wi];
        }
        int run = carry + woff + incl - s;
#pragma unroll
        for (int q = 0; q < 4; q++) {
            if (c0 + q < b.ncells) b.cursor[c0 + q] = run;
            run += v[q];
        }
        carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) *b.ticket = 0u;
}

__global__ void __launch_bounds__(256) bin_hist_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    const unsigned long long tick = b.tick_val;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < b.nsamp; i += (long long)gridDim.x * blockDim.x) {
        const int cell = cell_of(cfg, b, cfg.shard_begin + i, tick);
        if (b.keys) {
            // few cells, and one of them (life = H) may hold most candidates: one RED per warp and cell
            const unsigned peers = __match_any_sync(__activemask(), cell);
            if ((threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&b.hist[cell], __popc(peers));
        } else {
            atomicAdd(&b.hist[cell], 1);
        }
    }
    bin_scan_last_cta(b);
}

// Life-time keys and their histogram in one pass: thread = candidate, x_k = a_k + G_k u from the [k][1 + m][NP] table
// in shared memory (a_k: affine_base_kernel of this tick, G_k: mpmi_create), first violation -> keys[i]; then the same
// last-CTA scan as bin_hist_kernel.  The warp leaves the horizon loop once all its candidates are predicted dead.
template <int NP, int M>
__global__ void __launch_bounds__(256) bin_predict_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    static_assert(NP == 4 || NP == 8 || NP == 16, "padded physical dim");
    extern __shared__ __align__(16) float sag[];
    constexpr int stride = (1 + M) * NP;
    const int H = b.H;
    for (int e = threadIdx.x; e < H * stride; e += 256) {
        const int k = e / stride, c = (e % stride) / NP, j = e % NP;
        sag[e] = c == 0 ? cfg.aff_a[k * NP + j] : cfg.aff_g[(k * M + (c - 1)) * NP + j];
    }
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    const float none[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    float u[kMaxM];
    sample_u(cfg, cfg.shard_begin + (i < b.nsamp ? i : 0), b.tick_val, none, u);
    // branch-free safe test: dims without a box limit hold (-inf, +inf) in cfg, no annulus becomes [0, +inf].  (An infinite
    // state in an unlimited dim is predicted unsafe here, the rollout kernels call it safe: the prediction only orders the walk.)
    const float r2lo = cfg.annulus ? cfg.rmin2 : 0.f, r2hi = cfg.annulus ? cfg.rmax2 : __int_as_float(0x7f800000);
    __syncthreads();
    bool alive = i < b.nsamp;
    int steps = 0;
#pragma unroll 2
    for (int k = 0; k < H; k++) {
        if (!__any_sync(0xffffffffu, alive)) break;
        const float4 *row = reinterpret_cast<const float4 *>(sag + k * stride);
        float x[NP];
#pragma unroll
        for (int j = 0; j < NP / 4; j++) {
            float4 v = row[j];
#pragma unroll
            for (int q = 0; q < M; q++) {
                const float4 g = row[(1 + q) * (NP / 4) + j];
                v.x = __fmaf_rn(g.x, u[q], v.x); v.y = __fmaf_rn(g.y, u[q], v.y);
                v.z = __fmaf_rn(g.z, u[q], v.z); v.w = __fmaf_rn(g.w, u[q], v.w);
            }
            x[4 * j] = v.x; x[4 * j + 1] = v.y; x[4 * j + 2] = v.z; x[4 * j + 3] = v.w;
        }
        const float dx = __fsub_rn(x[0], cfg.cx), dy = __fsub_rn(x[1], cfg.cy);
        const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
        bool ok = alive && (r2 >= r2lo) && (r2 <= r2hi);
#pragma unroll
        for (int j = 0; j < NP; j++) ok = ok && (x[j] > cfg.blo[j]) && (x[j] < cfg.bhi[j]);
        alive = ok;
        steps += alive ? 1 : 0;
    }
    if (i < b.nsamp) {
        b.keys[i] = steps;
        const int cell = H - steps;
        const unsigned peers = __match_any_sync(__activemask(), cell);
        if ((threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&b.hist[cell], __popc(peers));
    }
    bin_scan_last_cta(b);
}

__global__ void __launch_bounds__(256) bin_scatter_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    const unsigned long long tick = b.tick_val;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < b.nsamp; i += (long long)gridDim.x * blockDim.x) {
        const int cell = cell_of(cfg, b, cfg.shard_begin + i, tick);
        int pos = 0;
        if (b.keys) {
            const unsigned peers = __match_any_sync(__activemask(), cell);
            const int lead = __ffs(peers) - 1, lane = threadIdx.x & 31;
            if (lane == lead) pos = atomicAdd(&b.cursor[cell], __popc(peers));
            pos = __shfl_sync(peers, pos, lead) + __popc(peers & ((1u << lane) - 1u));
        } else {
            pos = atomicAdd(&b.cursor[cell], 1);
        }
        b.perm[pos] = (int)i;
    }
}

}  // namespace mpmi
