// binning.cuh -- spatial ordering of the Philox candidates before the rollout.
//
// Algorithm 2 stops a candidate at its first unsafe state.  On a SIMT machine that
// only saves time when the candidates of one warp / CTA stop together.  Trajectories are affine in u,
// so candidates that are close in the input box share their fate; Philox hands them out in random
// order.  These two kernels counting-sort the candidate INDICES of one tick by the cell of the input
// box they fall in (cell = the top bits of the Philox words, row-major over the input dimensions):
//   bin_hist_kernel    histogram of cells (one RED per candidate) + exclusive scan by the last CTA
//   bin_scatter_kernel perm[cursor[cell]++] = local candidate index
//   bin_predict_kernel (life-time order, below) replaces bin_hist_kernel: keys + histogram + scan;
//   bin_scatter_keys_kernel is its scatter
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
    // exclusive scan of hist -> cursor by this (last) CTA; hist is cleared for the next tick.  64 consecutive cells per thread
    // and pass as 16 int4 loads, all in flight at once: 16,384 cells are one L2 round trip (with 4 cells per thread the 16
    // dependent passes were a serial tail of bin_hist_kernel on C4).  hist and cursor are allocated padded to a multiple of 64
    // cells (mpmi_api.cu), the padding of hist stays zero.
    constexpr int kScanCpt = 64;
    int carry = 0;
    for (int base = 0; base < b.ncells; base += 256 * kScanCpt) {
        int4 v[kScanCpt / 4];
        int s = 0;
        const int c0 = base + threadIdx.x * kScanCpt;
#pragma unroll
        for (int q = 0; q < kScanCpt / 4; q++)
            v[q] = c0 + 4 * q < b.ncells ? __ldcg(reinterpret_cast<const int4 *>(b.hist + c0) + q) : make_int4(0, 0, 0, 0);
#pragma unroll
        for (int q = 0; q < kScanCpt / 4; q++) {
            if (c0 + 4 * q < b.ncells) reinterpret_cast<int4 *>(b.hist + c0)[q] = make_int4(0, 0, 0, 0);
            s += v[q].x + v[q].y + v[q].z + v[q].w;
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
        for (int q = 0; q < kScanCpt / 4; q++) {
            int4 o4;
            o4.x = run; run += v[q].x;
            o4.y = run; run += v[q].y;
            o4.z = run; run += v[q].z;
            o4.w = run; run += v[q].w;
            if (c0 + 4 * q < b.ncells) reinterpret_cast<int4 *>(b.cursor + c0)[q] = o4;
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

// Life-time keys and their histogram in one pass: x_k = a_k + G_k u from the [k][1 + m][NP] table in shared memory (a_k:
// affine_base_kernel of this tick, G_k: mpmi_create), first violation -> keys[i]; then the same last-CTA scan as
// bin_hist_kernel.  A thread predicts kPredCand candidates: the table rows are warp-uniform LDS.128, each of which delivers
// 512 B to the warp, and with one candidate per thread those loads alone were the kernel (78 us for C5's 262,144 candidates:
// 8 LDS.128 per candidate-step = 32 clk of an SM's shared-memory bandwidth).  The life-time histogram is first built per CTA in
// shared memory: the cell "survives the horizon" holds ~40 % of the candidates, and one global RED per warp on that one
// address is serialised in L2.  Dynamic shared memory: the table, then H + 1 counters.
constexpr int kPredCand = 4;
template <int NP, int M>
__global__ void __launch_bounds__(256) bin_predict_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    static_assert(NP == 4 || NP == 8 || NP == 16, "padded physical dim");
    extern __shared__ __align__(16) float sag[];
    constexpr int stride = (1 + M) * NP;
    constexpr int C = kPredCand;
    const int H = b.H;
    int *s_hist = reinterpret_cast<int *>(sag + H * stride);
    for (int e = threadIdx.x; e < H * stride; e += 256) {
        const int k = e / stride, c = (e % stride) / NP, j = e % NP;
        sag[e] = c == 0 ? cfg.aff_a[k * NP + j] : cfg.aff_g[(k * M + (c - 1)) * NP + j];
    }
    for (int e = threadIdx.x; e <= H; e += 256) s_hist[e] = 0;
    const long long i0 = (long long)blockIdx.x * (256 * C) + threadIdx.x;
    const float none[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    float u[C][kMaxM];
    bool alive[C];
    int steps[C];
#pragma unroll
    for (int c = 0; c < C; c++) {
        const long long i = i0 + c * 256;
        sample_u(cfg, cfg.shard_begin + (i < b.nsamp ? i : 0), b.tick_val, none, u[c]);
        alive[c] = i < b.nsamp;
        steps[c] = 0;
    }
    // branch-free safe test: dims without a box limit hold (-inf, +inf) in cfg, no annulus becomes [0, +inf].  (An infinite
    // state in an unlimited dim is predicted unsafe here, the rollout kernels call it safe: the prediction only orders the walk.)
    const float r2lo = cfg.annulus ? cfg.rmin2 : 0.f, r2hi = cfg.annulus ? cfg.rmax2 : __int_as_float(0x7f800000);
    __syncthreads();
    for (int k = 0; k < H; k++) {
        bool any = false;
#pragma unroll
        for (int c = 0; c < C; c++) any = any || alive[c];
        if (!__any_sync(0xffffffffu, any)) break;
        const float4 *row = reinterpret_cast<const float4 *>(sag + k * stride);
        bool ok[C];
#pragma unroll
        for (int c = 0; c < C; c++) ok[c] = alive[c];
#pragma unroll
        for (int j = 0; j < NP / 4; j++) {                 // four physical dims at a time: the box test is separable
            const float4 a4 = row[j];
            float4 g4[M];
#pragma unroll
            for (int q = 0; q < M; q++) g4[q] = row[(1 + q) * (NP / 4) + j];
#pragma unroll
            for (int c = 0; c < C; c++) {
                float4 v = a4;
#pragma unroll
                for (int q = 0; q < M; q++) {
                    v.x = __fmaf_rn(g4[q].x, u[c][q], v.x); v.y = __fmaf_rn(g4[q].y, u[c][q], v.y);
                    v.z = __fmaf_rn(g4[q].z, u[c][q], v.z); v.w = __fmaf_rn(g4[q].w, u[c][q], v.w);
                }
                if (j == 0) {
                    const float dx = __fsub_rn(v.x, cfg.cx), dy = __fsub_rn(v.y, cfg.cy);
                    const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
                    ok[c] = ok[c] && (r2 >= r2lo) && (r2 <= r2hi);
                }
                ok[c] = ok[c] && (v.x > cfg.blo[4 * j]) && (v.x < cfg.bhi[4 * j]) && (v.y > cfg.blo[4 * j + 1]) && (v.y < cfg.bhi[4 * j + 1]) &&
                        (v.z > cfg.blo[4 * j + 2]) && (v.z < cfg.bhi[4 * j + 2]) && (v.w > cfg.blo[4 * j + 3]) && (v.w < cfg.bhi[4 * j + 3]);
            }
        }
#pragma unroll
        for (int c = 0; c < C; c++) { alive[c] = ok[c]; steps[c] += ok[c] ? 1 : 0; }
    }
#pragma unroll
    for (int c = 0; c < C; c++) {
        const long long i = i0 + c * 256;
        if (i < b.nsamp) {
            b.keys[i] = steps[c];
            const int cell = H - steps[c];
            const unsigned peers = __match_any_sync(__activemask(), cell);
            if ((threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&s_hist[cell], __popc(peers));
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e <= H; e += 256) {
        const int v = s_hist[e];
        if (v) atomicAdd(&b.hist[e], v);
    }
    bin_scan_last_cta(b);
}

// cells from the Philox words (uniform over the cells: no contention; four candidates per thread and pass with their
// fetch-and-adds in flight together were measured slower: 20.2 against 18.3 us for 2^20 candidates)
__global__ void __launch_bounds__(256) bin_scatter_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    const unsigned long long tick = b.tick_val;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < b.nsamp; i += (long long)gridDim.x * blockDim.x) {
        const int cell = cell_of(cfg, b, cfg.shard_begin + i, tick);
        b.perm[atomicAdd(&b.cursor[cell], 1)] = (int)i;
    }
}

// life-time order: few cells, one of them holding ~40 % of the candidates.  A CTA ranks its 1,024 candidates per cell in shared
// memory and takes ONE global fetch-and-add per cell it holds (with one per warp and cell the hot cell's 8,192 same-address
// atomics were the kernel: 18 us for 262,144 candidates).  Dynamic shared memory: 2 * ncells ints.
__global__ void __launch_bounds__(256) bin_scatter_keys_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ BinArgs b) {
    constexpr int C = 4;
    extern __shared__ int s_bin[];
    int *s_cnt = s_bin, *s_base = s_bin + b.ncells;
    const int lane = threadIdx.x & 31;
    for (long long chunk = blockIdx.x; chunk * (256 * C) < b.nsamp; chunk += gridDim.x) {
        for (int e = threadIdx.x; e < b.ncells; e += 256) s_cnt[e] = 0;
        __syncthreads();
        int cell[C], rank[C];
#pragma unroll
        for (int c = 0; c < C; c++) {
            const long long i = chunk * (256 * C) + c * 256 + threadIdx.x;
            cell[c] = 0; rank[c] = 0;
            if (i < b.nsamp) {
                const int st = b.keys[i];
                cell[c] = b.H - (st < 0 ? 0 : st > b.H ? b.H : st);
                const unsigned peers = __match_any_sync(__activemask(), cell[c]);
                const int lead = __ffs(peers) - 1;
                int pos = 0;
                if (lane == lead) pos = atomicAdd(&s_cnt[cell[c]], __popc(peers));
                rank[c] = __shfl_sync(peers, pos, lead) + __popc(peers & ((1u << lane) - 1u));
            }
        }
        __syncthreads();
        for (int e = threadIdx.x; e < b.ncells; e += 256) {
            const int v = s_cnt[e];
            if (v) s_base[e] = atomicAdd(&b.cursor[e], v);
        }
        __syncthreads();
#pragma unroll
        for (int c = 0; c < C; c++) {
            const long long i = chunk * (256 * C) + c * 256 + threadIdx.x;
            if (i < b.nsamp) b.perm[s_base[cell[c]] + rank[c]] = (int)i;
        }
        __syncthreads();
    }
}

}  // namespace mpmi
