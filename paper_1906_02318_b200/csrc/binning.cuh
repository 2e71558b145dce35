// binning.cuh -- spatial ordering of the Philox candidates before the rollout.
//
// Algorithm 2 stops a candidate at its first unsafe state.  On a SIMT machine that
// only saves time when the candidates of one warp / CTA stop together.  Trajectories are affine in u,
// so candidates that are close in the input box share their fate; Philox hands them out in random
// order.  These two kernels counting-sort the candidate INDICES of one tick by the cell of the input
// box they fall in (cell = the top bits of the Philox words, row-major over the input dimensions):
//   bin_hist_kernel    histogram of cells (one RED per candidate) + exclusive scan by the last CTA
//   bin_scatter_kernel perm[cursor[cell]++] = local candidate index
// The rollout kernel then walks perm, so a warp owns candidates of the same cell.  The candidate SET,
// every key and hence the result are unchanged (keys carry the original index).
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
};

__device__ __forceinline__ int cell_of(const DevCfg &cfg, const BinArgs &b, long long gi, unsigned long long tick) {
    unsigned w[4];
    philox4x32_10((unsigned)gi, (unsigned)((unsigned long long)gi >> 32), (unsigned)tick, (unsigned)(tick >> 32),
                  cfg.seed_lo, cfg.seed_hi, w);
    int cell = 0;
#pragma unroll
    for (int j = 0; j < kMaxM; j++)
        if (j < cfg.m && b.bits[j] > 0) cell = (cell << b.bits[j]) | (int)(w[j] >> (32 - b.bits[j]));
    return cell;
}

__global__ void __launch_bounds__(256) bin_hist_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    const unsigned long long tick = b.tick_val;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < b.nsamp; i += (long long)gridDim.x * blockDim.x)
        atomicAdd(&b.hist[cell_of(cfg, b, cfg.shard_begin + i, tick)], 1);
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

__global__ void __launch_bounds__(256) bin_scatter_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    const unsigned long long tick = b.tick_val;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < b.nsamp; i += (long long)gridDim.x * blockDim.x) {
        const int pos = atomicAdd(&b.cursor[cell_of(cfg, b, cfg.shard_begin + i, tick)], 1);
        b.perm[pos] = (int)i;
    }
}

}  // namespace mpmi
