// rollout_tc.cuh -- tensor-core rollout kernel for padded lifted dim D = 128 (a1-a7, a9), sm_100a.
//
// At d = 128 one rollout step of a tile of 128 candidates IS a dense contraction
// Z'[128 x 128] = [Z | U][128 x 136] * [K | B | 0]^T ("a single matrix-matrix
// multiplication").  Plain TF32 fails the 1e-4 trajectory tolerance, so every step
// is computed as the 3xTF32 split product
//     Z' = Z_hi * K_hi + Z_hi * K_lo + Z_lo * K_hi,      x_hi = x with the low 13 mantissa bits
// cleared, x_lo = x - x_hi (exact in fp32); the dropped x_lo * k_lo term is 2^-22 relative.
// tcgen05.mma reads TF32 operands by IGNORING the low 13 bits of the fp32 word (measured), so the
// fp32 accumulator tile itself serves as the A operand Z_hi of the next step:
//
//   TMEM (512 columns x 128 lanes, lane = candidate):  D0 | D1 (ping-pong fp32 state / accumulator)
//        | A_lo (128 cols) | U = [u_hi (4) | u_lo (4)]
//   shared memory: K_hi and K_lo as K-major no-swizzle B operands ([K | B B], 128 x 136 fp32 each; the second copy of B
//   is zero in the lo image, so the input costs two MMAs per step: U K_lo = u_hi B_lo, U K_hi = (u_hi + u_lo) B_hi).
//
// Warp roles: warps 0..7 are "state" warps -- warp e owns TMEM lanes 32*(e%4).. and columns
// 64*(e/4)..: after every step they read the new state with tcgen05.ld (thread = one candidate,
// so the safe test is thread-local), write Z_lo back with tcgen05.st and hand the
// tile back through an mbarrier; warp 8 (one elected lane) issues the MMAs.  Z_hi * K_lo of step
// s+1 needs only the accumulator of step s, so it runs WHILE the state warps test and split step
// s; Z_lo * K_hi waits for them, Z_hi * K_hi goes last: the tensor core accumulates with
// truncation toward zero (measured), so the small products are added while the accumulator is
// still ~2^-11 |z| and only 17 accumulations run at full magnitude (trajectory error 1.3e-5
// against 6.6e-5 with the large product first; FP32 SIMT: 1.5e-6; tolerance 1e-4).
// Tiles of 128 candidates are fetched from a global counter (persistent CTAs, one per SM); a
// tile stops when none of its candidates is alive.  Consecutive MMAs that read the accumulator of
// earlier MMAs as their A operand are NOT ordered by the pipeline (measured: stale reads), hence
// the commit + mbarrier wait between steps.
#pragma once
#include "mpmi_device.cuh"
#include "kernel_args.cuh"
#include "tcgen05.cuh"

namespace mpmi {

constexpr int kTcTile = 128;                      // candidates per tile = TMEM lanes
constexpr int kTcLBO = 128;                       // bytes between 16-byte K chunks (core matrices contiguous along K)
#ifndef MPMI_TC_KSPLIT
#define MPMI_TC_KSPLIT 17            // d = 128: all 17 k-blocks of Z_hi * K_lo go out before the hand-back wait (measured with the
#endif                               // convergent issue loop: 10 / 15 / 17 -> first pass 1.51 / 1.41 / 1.37 ms on C5)
#ifndef MPMI_TC_STATE_WARPS
#define MPMI_TC_STATE_WARPS 8
#endif
#ifndef MPMI_TC32_STATE_WARPS
#define MPMI_TC32_STATE_WARPS 4      // (8, i.e. 16 columns per thread at 56 registers, was measured slower: first pass 0.76 -> 0.82 ms)
#endif
// Geometry for padded lifted dim D = 128 (one CTA per SM, all 512 TMEM columns) and D = 32 (the same kernel with
// N = 32 MMAs: a tile needs 3 D + 24 = 120 TMEM columns and 12 KB of operand images, so FOUR CTAs share an SM and
// their step phases interleave -- measured: one CTA issues an M128 N32 K8 MMA every ~49 clk, four reach the 16 clk floor).
template <int D>
struct TcGeom {
    static_assert(D == 128 || D == 32, "tensor-core rollout: D = 128 or 32");
    static constexpr int kD = D;
    static constexpr int kKB = D / 8;                              // k-blocks of the state
    static constexpr int kKD = D + 16;                             // contraction length: D state + 8 input columns ([u_hi | u_lo], m <= 4)
                                                                   // + 8 noise columns (n <= 8; used by the NOISE instantiation only)
    static constexpr int kStateWarps = D == 128 ? MPMI_TC_STATE_WARPS : MPMI_TC32_STATE_WARPS;   // 4 lane quadrants x column groups
    static constexpr int kCols = D / (kStateWarps / 4);            // state columns per state-warp thread
    static constexpr int kThreads = (kStateWarps + 1) * 32;
    static constexpr int kSBO = (kKD / 4) * 128;                   // bytes between 8-row groups
    static constexpr int kImg = (D / 8) * kSBO;                    // bytes of one B-operand image (69,632 at D = 128)
    static constexpr int kSmemBytes = 2 * kImg;
    static constexpr int kTmemCols = D == 128 ? 512 : 128;
    static constexpr int kCtasPerSm = 512 / kTmemCols;
    static constexpr int kSplit = D == 128 ? MPMI_TC_KSPLIT : kKB + 1;   // group-1 k-blocks issued before the hand-back wait
    static constexpr uint32_t kColD0 = 0, kColD1 = D, kColAlo = 2 * D, kColU = 3 * D, kColNhi = 3 * D + 8, kColNlo = 3 * D + 16;
};
// the kernel body keeps the short names
#define MPMI_TC_GEOM(D)                                                                                                     \
    using G = TcGeom<D>;                                                                                                    \
    constexpr int kTcD = G::kD, kTcKB = G::kKB, kTcKD = G::kKD, kTcStateWarps = G::kStateWarps, kTcCols = G::kCols,           \
                  kTcThreads = G::kThreads, kTcSBO = G::kSBO, kTcImg = G::kImg;                                              \
    constexpr uint32_t kTcColD0 = G::kColD0, kTcColD1 = G::kColD1, kTcColAlo = G::kColAlo, kTcColU = G::kColU,                \
                       kTcColNhi = G::kColNhi, kTcColNlo = G::kColNlo;                                                       \
    (void)kTcKB; (void)kTcKD; (void)kTcCols; (void)kTcThreads; (void)kTcSBO; (void)kTcImg; (void)kTcColD0; (void)kTcColD1;    \
    (void)kTcColAlo; (void)kTcColU; (void)kTcColNhi; (void)kTcColNlo; (void)kTcStateWarps; (void)kTcD

__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
// x_lo = x - x_hi (exact) has up to 13 significant bits and the tensor core keeps 11 by TRUNCATION, a bias
// toward zero of ~2^-22 |x| per operand that adds up coherently over the horizon.  Adding half a TF32 ulp
// to the bit pattern first turns the hardware's truncation into round-half-away (one integer add).
__device__ __forceinline__ uint32_t tf32_lo(float x) { return __float_as_uint(x - tf32_hi(x)) + 0x1000u; }
// the same for two values at once: the exact subtraction as one packed FADD2 (sub.rn.f32x2) -- per step and thread the split
// is the bulk of the state warps' instructions (LOP3 + FADD + IADD per value), and four CTAs per SM share each scheduler
__device__ __forceinline__ void tf32_lo2(uint32_t x0, uint32_t x1, uint32_t &l0, uint32_t &l1) {
    const uint32_t h0 = x0 & 0xFFFFE000u, h1 = x1 & 0xFFFFE000u;
    unsigned long long xx, hh, ll;
    asm("mov.b64 %0, {%1,%2};" : "=l"(xx) : "r"(x0), "r"(x1));
    asm("mov.b64 %0, {%1,%2};" : "=l"(hh) : "r"(h0), "r"(h1));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(ll) : "l"(xx), "l"(hh));
    asm("mov.b64 {%0,%1}, %2;" : "=r"(l0), "=r"(l1) : "l"(ll));
    l0 += 0x1000u; l1 += 0x1000u;
}
// round-to-nearest TF32 (ties away) and the matching low part x - x_hi (exact in fp32, either sign), itself rounded as above
__device__ __forceinline__ float tf32_rn(float x) { return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u); }
__device__ __forceinline__ uint32_t tf32_lo_of(float x, float x_hi) { return __float_as_uint(x - x_hi) + 0x1000u; }

// Same decision as safe_check (mpmi_device.cuh) -- box strict, annulus closed, NaN / Inf unsafe -- but without
// the 2*nbox-long chain of dependent predicate ANDs (~13 cycles per link), which sits on the per-step critical
// path here: lo < x < hi  <=>  min(x - lo, hi - x) > 0 (the sign of an fp32 difference is exact); the minimum
// over all tested dims is a NaN-propagating tree (min.NaN), and NaN fails the final comparison.
template <int NB, int J0, int J1>
__device__ __forceinline__ float box_slack(const DevCfg &cfg, const float (&x)[NB]) {
    if constexpr (J1 - J0 == 1) {
        return min_nan(__fsub_rn(x[J0], cfg.blo[J0]), __fsub_rn(cfg.bhi[J0], x[J0]));
    } else {
        constexpr int JM = (J0 + J1) / 2;
        return min_nan(box_slack<NB, J0, JM>(cfg, x), box_slack<NB, JM, J1>(cfg, x));
    }
}
template <int NB>
__device__ __forceinline__ bool safe_check_par(const DevCfg &cfg, const float (&x)[NB], int nbox) {
    static_assert(NB == 16, "tensor-core kernel: 16 physical-state columns");
    float m = __int_as_float(0x7f800000);
    if (nbox > 0) {
        m = box_slack<NB, 0, 2>(cfg, x);
        if (nbox > 2) {
            m = min_nan(m, box_slack<NB, 2, 4>(cfg, x));
            if (nbox > 4) {
                m = min_nan(m, box_slack<NB, 4, 8>(cfg, x));
                if (nbox > 8) m = min_nan(m, box_slack<NB, 8, 16>(cfg, x));
            }
        }
    }
    bool ok = m > 0.f;
    if (cfg.annulus) {
        const float dx = __fsub_rn(x[0], cfg.cx), dy = __fsub_rn(x[1], cfg.cy);
        const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
        ok = ok && (r2 >= cfg.rmin2) && (r2 <= cfg.rmax2);
    }
    return ok;
}

// Verified tick: did this state come within tau_i(k) of the safe-set boundary (on either side)?  tau_i(k) (bound.cuh) bounds
// |x~_k - x^_k|_i between this kernel's state and the FP32 kernel's for the same candidate, so a candidate that never does has,
// step by step, the same isSafe result in both; one that does is rolled again by the FP32 kernel (kernel_args.cuh: recheck).
// trow = this step's row of the tau table: [tau_0 .. tau_{np-1} | thr(r_min^2), thr(r_max^2)].  NaN counts as near.
template <int NB, int J0, int J1>
__device__ __forceinline__ float box_near(const DevCfg &cfg, const float (&x)[NB], const float *trow, float sc) {
    if constexpr (J1 - J0 == 1) {
        const float q = fminf(fabsf(__fsub_rn(x[J0], cfg.blo[J0])), fabsf(__fsub_rn(cfg.bhi[J0], x[J0])));
        return __fmaf_rn(-sc, __ldg(trow + J0), q);                    // distance to the nearer limit, minus tau
    } else {
        constexpr int JM = (J0 + J1) / 2;
        return min_nan(box_near<NB, J0, JM>(cfg, x, trow, sc), box_near<NB, JM, J1>(cfg, x, trow, sc));
    }
}
template <int NB>
__device__ __forceinline__ bool near_boundary(const DevCfg &cfg, const float (&x)[NB], int nbox, const float *trow, int np, float sc) {
    bool nr = false;
    if (nbox > 0) {
        float m = box_near<NB, 0, 2>(cfg, x, trow, sc);
        if (nbox > 2) {
            m = min_nan(m, box_near<NB, 2, 4>(cfg, x, trow, sc));
            if (nbox > 4) {
                m = min_nan(m, box_near<NB, 4, 8>(cfg, x, trow, sc));
                if (nbox > 8) m = min_nan(m, box_near<NB, 8, 16>(cfg, x, trow, sc));
            }
        }
        nr = !(m >= 0.f);
    }
    if (cfg.annulus) {
        const float dx = __fsub_rn(x[0], cfg.cx), dy = __fsub_rn(x[1], cfg.cy);
        const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
        const float qa = __fmaf_rn(-sc, __ldg(trow + np), fabsf(__fsub_rn(r2, cfg.rmin2)));
        const float qb = __fmaf_rn(-sc, __ldg(trow + np + 1), fabsf(__fsub_rn(cfg.rmax2, r2)));
        nr = nr || !(min_nan(qa, qb) >= 0.f);
    }
    return nr;
}

template <int D>
struct TcShared {
    unsigned long long bar_full, bar_alo, bar_tile;
    uint32_t tmem_base;
    unsigned tile[2];
    unsigned stop_tile;
    unsigned warp_alive[4];
    float z0[D];
#ifdef MPMI_TC_DEBUG
    long long dbg_wake;
#endif
};

// sigma * eps of Algorithm 2 l.5 for the tensor-core kernel: the state lives in the accumulator, so the
// noise enters the contraction as 8 extra A columns [sigma eps_hi | sigma eps_lo] against the selector rows of the K_hi
// image (1.0 at (r = j, c = D + 8 + j): exact in TF32, its lo part is 0): z'_j += sigma eps_j through two more MMAs per step.
// Split in two so that the expensive half -- two Philox calls and three Box-Muller pairs per candidate and step, more than twice the
// rest of a state warp's step -- runs AFTER the hand-back, while the tensor core works on this tile, and only the two stores stay
// on the step's critical path.
template <int D>
__device__ __forceinline__ void tc_noise_compute(const DevCfg &cfg, long long gi, int k, unsigned long long tick, float (&v)[8]) {
    float g[8];                                                  // eps of the ORIGINAL dims 0..7
#pragma unroll
    for (int q = 0; q < 2; q++) {
        float g4[4] = {0.f, 0.f, 0.f, 0.f};
        if (4 * q < cfg.n) noise4(cfg, gi, k, q, tick, g4);
#pragma unroll
        for (int e = 0; e < 4; e++) g[4 * q + e] = g4[e];
    }
#pragma unroll
    for (int j = 0; j < 8; j++)                                  // internal dim j = original dim perm[j]
        v[j] = j < cfg.n ? __fmul_rn(cfg.noise_sigma, g[cfg.perm[j] & 7]) : 0.f;
}
template <int D>
__device__ __forceinline__ void tc_noise_put(const float (&v)[8], uint32_t tlane) {
    MPMI_TC_GEOM(D);
    uint32_t nh[8], nl[8];
#pragma unroll
    for (int j = 0; j < 8; j++) { nh[j] = __float_as_uint(v[j]); nl[j] = tf32_lo(v[j]); }
    tc::tmem_st8(tlane + kTcColNhi, nh);
    tc::tmem_st8(tlane + kTcColNlo, nl);
}

template <int D, int MODE, bool NOISE = false>
__global__ void __launch_bounds__(TcGeom<D>::kThreads, TcGeom<D>::kCtasPerSm)
rollout_tc_kernel(const __grid_constant__ DevCfg cfg, const __grid_constant__ KArgs a) {
    using namespace tc;
    MPMI_TC_GEOM(D);
    extern __shared__ __align__(1024) unsigned char smem_img[];      // K_hi image | K_lo image
    __shared__ TcShared<D> sh;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned long long tick = a.tick_val;
    const float *x0p = a.inline_inputs ? a.x0_val : a.x0;
    const float *uup = a.inline_inputs ? a.u_val : a.u_user;
    const int H = (MODE == MODE_TICK) ? cfg.H : a.H;
    const long long ncand = (MODE == MODE_TICK) ? cfg.shard_count : a.ncand;
    const bool shared_x0 = (MODE == MODE_TICK) || a.x0_count == 1;
    const unsigned ntile = (unsigned)((ncand + kTcTile - 1) / kTcTile);

    // ---- one-off: B-operand images [K | B | 0] split into hi / lo, TMEM, barriers, shared lift
    for (int e = tid; e < kTcD * kTcKD; e += kTcThreads) {
        const int r = e % kTcD, c = e / kTcD;                        // K[r][c] = KTa[c][r]; rows D.. are B's columns
        // columns D..D+7 meet the A block [u_hi (4) | u_lo (4)]: B twice in the hi image (u_hi B_hi + u_lo B_hi), B_lo once
        // in the lo image (u_hi B_lo) -- two MMAs per step for the input instead of three
        const int cb = c - kTcD;                                     // (at D = 128: columns 128..135 and 136..143)
        const bool bcol = cb >= 0 && cb < 8 && (cb & 3) < cfg.m;
        const float v = c < kTcD ? cfg.KTa[c * kTcD + r] : bcol ? cfg.KTa[(kTcD + (cb & 3)) * kTcD + r]
                      : (c >= kTcD + 8 && r == c - (kTcD + 8)) ? 1.f : 0.f;                       // [K | B B | noise selector]
        const int off = (r >> 3) * kTcSBO + (c >> 2) * kTcLBO + (r & 7) * 16 + (c & 3) * 4;
        // K_hi = v ROUNDED to nearest TF32 (the model image is built here, so it need not be the truncation the hardware applies
        // to the state): |K_lo| <= 2^-11 |K| instead of 2^-10, which halves the dropped z_lo K_lo product (csrc/bound.cuh)
        const float vh = tf32_rn(v);
        *reinterpret_cast<float *>(smem_img + off) = vh;
        *reinterpret_cast<uint32_t *>(smem_img + kTcImg + off) = (cb >= 4 && cb < 8) ? 0u : tf32_lo_of(v, vh);
    }
    float u_h[kMaxM] = {0.f, 0.f, 0.f, 0.f};
    bool inputs_ok = true;
    if (MODE == MODE_TICK) {
        inputs_ok = finite_inputs(cfg, x0p, uup);
        clamp_user(cfg, uup, u_h);
    }
    if (shared_x0)
        for (int f = tid; f < kTcD; f += kTcThreads) sh.z0[f] = lift_feature(cfg, f, x0p);
    if (warp == kTcStateWarps) tmem_alloc<G::kTmemCols>(smem_u32(&sh.tmem_base));
    if (tid == 0) {
        mbar_init(smem_u32(&sh.bar_full), 1);
        mbar_init(smem_u32(&sh.bar_alo), kTcStateWarps * 32);
        mbar_init(smem_u32(&sh.bar_tile), 1);
        sh.stop_tile = 0xFFFFFFFFu;
        fence_barrier_init();
    }
    fence_proxy_async_smem();
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tb = sh.tmem_base;
    const uint32_t bar_full = smem_u32(&sh.bar_full), bar_alo = smem_u32(&sh.bar_alo), bar_tile = smem_u32(&sh.bar_tile);

    unsigned long long key = kKeyNone;
    unsigned n_safe = 0, n_exec = 0;

    if (warp == kTcStateWarps) {
        // ================= MMA issuer ====================================================================
        // The whole warp runs this loop CONVERGENTLY and one elected lane issues the MMAs (elect.sync): every tcgen05.mma
        // operand (TMEM addresses, shared-memory descriptors) is then a warp-uniform value that ptxas can keep in uniform
        // registers.  With the loop inside `if (lane == 0)` (round 1) every operand lived in a vector register of a divergent
        // region and each MMA was wrapped in an ELECT / R2UR.BROADCAST sequence, ~49 clk per MMA.
        {
            const uint32_t tbu = __reduce_max_sync(0xffffffffu, tb);          // uniform by construction
            const uint32_t idesc = idesc_tf32(kTcTile, kTcD);
            const uint64_t dhi = smem_desc_kmajor(smem_u32(smem_img), kTcLBO, kTcSBO);
            const uint64_t dlo = smem_desc_kmajor(smem_u32(smem_img + kTcImg), kTcLBO, kTcSBO);
            constexpr uint64_t kstep = (2 * kTcLBO) >> 4;                 // descriptor address units per k-block
            unsigned p_full = 0, p_alo = 0;
#ifdef MPMI_TC_DEBUG
            long long tw_full = 0, ti_1 = 0, tw_alo = 0, ti_23 = 0, nsteps = 0, tq = 0;
#define TCT(acc) do { long long t_ = clock64(); acc += t_ - tq; tq = t_; } while (0)
#else
#define TCT(acc) do {} while (0)
#endif
            auto tile_alive = [&]() { return (sh.warp_alive[0] | sh.warp_alive[1] | sh.warp_alive[2] | sh.warp_alive[3]) != 0u; };
            for (unsigned it = 0;; it++) {
                unsigned tile = 0;
                if (lane == 0) tile = atomicAdd(a.work, 1u);
                tile = __shfl_sync(0xffffffffu, tile, 0);
                if (lane == 0) { sh.tile[it & 1] = tile; mbar_arrive(bar_tile); }
                __syncwarp();
                if (tile >= ntile) break;
                for (int s = 0; s < H; s++) {
                    const uint32_t dcur = tbu + ((s & 1) ? kTcColD1 : kTcColD0), dnxt = tbu + ((s & 1) ? kTcColD0 : kTcColD1);
#ifdef MPMI_TC_DEBUG
                    tq = clock64(); nsteps++;
#endif
                    // z_s complete in TMEM: written by the previous step's MMAs (s > 0) or by the prologue (s = 0)
                    if (s > 0) { mbar_wait(bar_full, p_full); p_full ^= 1; }
                    else { mbar_wait(bar_alo, p_alo); p_alo ^= 1; }
                    fence_after_sync();
                    TCT(tw_full);
#ifdef MPMI_TC_DEBUG
                    if (s > 0 && lane == 0) *reinterpret_cast<volatile long long *>(&sh.dbg_wake) = clock64();
#endif
                    // The small products go first: the tensor core accumulates with truncation toward zero
                    // (measured), so terms added while the accumulator is still ~2^-11 |z| lose nothing that
                    // matters, and only the accumulations of Z_hi * K_hi run at full magnitude.
                    if (s == 0 && !tile_alive()) {                         // nothing valid in this tile
                        if (lane == 0) { sh.stop_tile = tile; mbar_arrive(bar_full); }
                        __syncwarp();
                        break;
                    }
                    constexpr int kSplit = G::kSplit;                      // k-blocks of group 1 issued before the hand-back wait
                    if (elect_one()) {
#pragma unroll
                        for (int kk = 0; kk < kSplit; kk++)                // Z_hi * K_lo  (Z_hi = the fp32 state itself)
                            mma_tf32_ts(dnxt, kk < kTcKB ? dcur + 8 * kk : tbu + kTcColU, dlo + kk * kstep, idesc, kk > 0);
                    }
                    __syncwarp();
                    TCT(ti_1);
                    if (s > 0) {                                           // state warps: z_s tested, Z_lo written
                        mbar_wait(bar_alo, p_alo); p_alo ^= 1;             // (its latency hides behind the queued MMAs)
                        fence_after_sync();
                        if (!tile_alive()) {                               // stop: the queued MMAs drain, then the commit wakes the state warps
                            if (elect_one()) { sh.stop_tile = tile; mma_commit(bar_full); }
                            __syncwarp();
                            break;
                        }
                    }
                    TCT(tw_alo);
                    if (elect_one()) {
#pragma unroll
                        for (int kk = kSplit; kk < kTcKB + 1; kk++)        // (last k-block: u_hi * B_lo)
                            mma_tf32_ts(dnxt, kk < kTcKB ? dcur + 8 * kk : tbu + kTcColU, dlo + kk * kstep, idesc, true);
#pragma unroll
                        for (int kk = 0; kk < kTcKB; kk++)                 // Z_lo * K_hi
                            mma_tf32_ts(dnxt, tbu + kTcColAlo + 8 * kk, dhi + kk * kstep, idesc, true);
                        if (NOISE) mma_tf32_ts(dnxt, tbu + kTcColNlo, dhi + (kTcKB + 1) * kstep, idesc, true);     // (sigma eps)_lo through the selector
                        // Z_hi * K_hi, the only products at full magnitude, in DESCENDING k-block order: input block ((u_hi + u_lo) * B_hi),
                        // (sigma eps)_hi, then the state blocks KB-1 .. 0.  Every accumulation truncates the running sum (<= 2 ulp), so the
                        // block of the physical dims (columns 0..7), the dominant one of a physical row when K is close to the identity
                        // there, goes last and is truncated once (csrc/bound.cuh weighs block b with b + 1 accumulations).
                        mma_tf32_ts(dnxt, tbu + kTcColU, dhi + kTcKB * kstep, idesc, true);
                        if (NOISE) mma_tf32_ts(dnxt, tbu + kTcColNhi, dhi + (kTcKB + 1) * kstep, idesc, true);
#pragma unroll
                        for (int kk = kTcKB - 1; kk >= 0; kk--)
                            mma_tf32_ts(dnxt, dcur + 8 * kk, dhi + kk * kstep, idesc, true);
                        mma_commit(bar_full);
                    }
                    __syncwarp();
                    TCT(ti_23);
                }
                mbar_wait(bar_full, p_full); p_full ^= 1;                 // last commit (or the stop signal) of this tile
            }
#ifdef MPMI_TC_DEBUG
            if (blockIdx.x == 0 && lane == 0 && nsteps > 0)
                printf("tc timing (clk/step): wait_full %lld issue1 %lld wait_alo %lld issue23 %lld  steps %lld\n",
                       tw_full / nsteps, ti_1 / nsteps, tw_alo / nsteps, ti_23 / nsteps, nsteps);
#endif
        }
        __syncwarp();
    } else {
        // ================= state warps: thread = (candidate row, column half) ===========================
        const int q = warp & 3, hc = warp >> 2;                          // TMEM lane quadrant, column group
        const int row = q * 32 + lane;
        const uint32_t tlane = tb + ((uint32_t)(q * 32) << 16);
        const int c0 = hc * kTcCols;
        constexpr int NB = kMaxN;
        const int nbox = __popc(cfg.bmask) ? 32 - __clz(cfg.bmask) : 0;
        const bool dump = (MODE == MODE_BATCH) && a.dump_kind != MPMI_DUMP_NONE;
        const int J = dump ? (a.dump_kind == MPMI_DUMP_PHYS ? cfg.n : cfg.d) : 0;
        const float qnan = __int_as_float(0x7fc00000);
        // verified tick / batch: a.recheck != null -- candidates that come within tau_i(k) of the boundary go to the FP32 kernel
        const bool verify = a.recheck != nullptr;
        const int tau_stride = cfg.aff_np + 4;                       // bound.cuh: kTauPad
        const float tau_sc = a.recheck_tau_scale;
        unsigned p_full = 0, p_tile = 0;
#ifdef MPMI_TC_DEBUG
        long long sw_wait = 0, sw_ld = 0, sw_math = 0, sw_st = 0, sw_n = 0, sw_skew = 0, sq = clock64();
#define SWT(acc) do { long long t_ = clock64(); acc += t_ - sq; sq = t_; } while (0)
#else
#define SWT(acc) do {} while (0)
#endif
        for (unsigned it = 0;; it++) {
            mbar_wait(bar_tile, p_tile); p_tile ^= 1;
            const unsigned tile = sh.tile[it & 1];
            if (tile >= ntile) break;

            // ---- a1 + a2: this thread's candidate, its half of z_0 and (column half 0) its input
            // ordered walk (longest first): the ragged last tile holds the injected u_h, which may well run the
            // whole horizon -- it goes first instead of alone at the very end
            const unsigned wtile = (MODE == MODE_TICK && a.perm) ? (tile == 0 ? ntile - 1 : tile - 1) : tile;
            long long li = (long long)wtile * kTcTile + row;
            if (MODE == MODE_TICK && a.perm && li < a.nsamp) li = a.perm[li];
            const bool valid = li < ncand && inputs_ok;
            bool alive = valid;
            bool near = false;
            int steps = 0;
            float u[kMaxM] = {0.f, 0.f, 0.f, 0.f};
            if (li < ncand) {
                if (MODE == MODE_BATCH && a.U) {
                    for (int j = 0; j < cfg.m; j++) u[j] = a.U[li * cfg.m + j];
                } else {
                    sample_u(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, tick, u_h, u);
                }
            }
            __syncwarp();                                                // tcgen05.st / ld below are .sync.aligned
            float nz[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};      // NOISE: sigma * eps of the next MMA step (internal dims 0..7)
            {
                float x[kMaxN];
                if (!shared_x0) {
                    const long long r0 = li < ncand ? li : 0;
                    for (int j = 0; j < kMaxN; j++) x[j] = j < cfg.n ? a.x0[r0 * cfg.n + j] : 0.f;
                }
#pragma unroll 1
                for (int cc = 0; cc < kTcCols; cc += 16) {
                    uint32_t v[16], lo[16];
#pragma unroll
                    for (int j = 0; j < 16; j++) {
                        const float z = shared_x0 ? sh.z0[c0 + cc + j] : lift_feature(cfg, c0 + cc + j, x);
                        v[j] = __float_as_uint(z);
                        lo[j] = tf32_lo(z);
                    }
                    tmem_st16(tlane + kTcColD0 + c0 + cc, v);
                    tmem_st16(tlane + kTcColAlo + c0 + cc, lo);
                }
                if (hc == 0) {
                    static_assert(kMaxM <= 4, "input block: [u_hi (4) | u_lo (4)]");
                    uint32_t uv[8];
#pragma unroll
                    for (int j = 0; j < 4; j++) {
                        const float uj = j < kMaxM ? u[j < kMaxM ? j : 0] : 0.f;
                        uv[j] = __float_as_uint(uj);
                        uv[4 + j] = tf32_lo(uj);
                    }
                    tmem_st8(tlane + kTcColU, uv);
                    const bool any = __any_sync(0xffffffffu, alive);
                    if (lane == 0) sh.warp_alive[q] = any ? 1u : 0u;
                }
                if (NOISE && hc == kTcStateWarps / 4 - 1)          // the last column group draws the noise of step 0
                {
                    tc_noise_compute<D>(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, 0, tick, nz);
                    tc_noise_put<D>(nz, tlane);
                }
            }
            wait_st();
            fence_before_sync();
            mbar_arrive(bar_alo);
            if (NOISE && hc == kTcStateWarps / 4 - 1 && H > 1)           // noise of MMA step 1, while step 0 runs
                tc_noise_compute<D>(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, 1, tick, nz);

            // ---- a3 + a4: after MMA step s-1 the accumulator holds z_s; test it, split it, hand it back
            int s = 1;
            for (; s <= H; s++) {
                SWT(sw_math);
                mbar_wait(bar_full, p_full); p_full ^= 1;
                fence_after_sync();
                SWT(sw_wait);
#ifdef MPMI_TC_DEBUG
                sw_n++;
                if (s > 1) sw_skew += clock64() - *reinterpret_cast<volatile long long *>(&sh.dbg_wake);
#endif
                if (*reinterpret_cast<volatile unsigned *>(&sh.stop_tile) == tile) break;
                const uint32_t dcol = (s & 1) ? kTcColD1 : kTcColD0;
                const bool was_alive = alive;
                __syncwarp();
                // this thread's kTcCols columns of z_s: all loads in flight, one wait
                uint32_t r[kTcCols];
#pragma unroll
                for (int cc = 0; cc < kTcCols; cc += 16) tmem_ld16(tlane + dcol + c0 + cc, *reinterpret_cast<uint32_t(*)[16]>(&r[cc]));
                uint32_t rp[16];                                         // the physical state sits in columns 0..15
                if (dump && hc != 0) tmem_ld16(tlane + dcol, rp);
                wait_ld();
                SWT(sw_ld);
                if (hc == 0 || dump) {
                    float x[NB];
#pragma unroll
                    for (int j = 0; j < NB; j++) x[j] = __uint_as_float(hc == 0 ? r[j] : rp[j]);
                    alive = safe_check_par<NB>(cfg, x, nbox) && was_alive;
                    steps += alive ? 1 : 0;
                }
                if (hc == 0) {
                    const bool any = __any_sync(0xffffffffu, alive);
                    if (lane == 0) sh.warp_alive[q] = any ? 1u : 0u;
                }
                if (s < H) {
#pragma unroll
                    for (int cc = 0; cc < kTcCols; cc += 8) {
                        uint32_t lo[8];
#pragma unroll
                        for (int j = 0; j < 8; j += 2) tf32_lo2(r[cc + j], r[cc + j + 1], lo[j], lo[j + 1]);
                        tmem_st8(tlane + kTcColAlo + c0 + cc, lo);
                    }
                    if (NOISE && hc == kTcStateWarps / 4 - 1)      // noise of MMA step s (it produces z_{s+1})
                        tc_noise_put<D>(nz, tlane);                  // (computed after the previous hand-back)
                }
                if (dump && li < ncand) {                                // a9: traj[(k*J + row)*Ncand + i], k = s-1
#pragma unroll
                    for (int j = 0; j < kTcCols; j++) {
                        const int ji = c0 + j;
                        const int orow = ji < cfg.n ? (int)cfg.perm[ji < kMaxN ? ji : 0] : ji;
                        if (orow < J)
                            a.traj[((long long)(s - 1) * J + orow) * ncand + li] = was_alive ? __uint_as_float(r[j]) : qnan;
                    }
                }
                if (s < H) {
                    SWT(sw_math);
                    wait_st();
                    fence_before_sync();
                    mbar_arrive(bar_alo);
                    SWT(sw_st);
                }
                if (NOISE && hc == kTcStateWarps / 4 - 1 && s + 1 < H)   // noise of MMA step s + 1, while step s runs
                    tc_noise_compute<D>(cfg, (MODE == MODE_TICK ? cfg.shard_begin : 0) + li, s + 1, tick, nz);
                if (verify && hc == 0) {                                 // off the step's critical path: after the hand-back
                    float x[NB];
#pragma unroll
                    for (int j = 0; j < NB; j++) x[j] = __uint_as_float(r[j]);
                    near = near || (was_alive && near_boundary<NB>(cfg, x, nbox, cfg.bnd_tau + (size_t)s * tau_stride, cfg.aff_np, tau_sc));
                }
            }
            if (dump && li < ncand) {                                    // states after the tile stopped: NaN
                for (int k = s - 1; k < H; k++)
                    for (int j = 0; j < kTcCols; j++) {
                        const int ji = c0 + j;
                        const int orow = ji < cfg.n ? (int)cfg.perm[ji < kMaxN ? ji : 0] : ji;
                        if (orow < J) a.traj[((long long)k * J + orow) * ncand + li] = qnan;
                    }
            }
            if (hc == 0) {
                if (MODE == MODE_BATCH) {
                    if (li < ncand) {
                        a.steps[li] = steps;
                        if (a.safe) a.safe[li] = steps == H ? 1 : 0;
                    }
                }
                bool push = false;
                if (verify) {                                            // near the boundary: the FP32 kernel decides (warp-aggregated append)
                    push = li < ncand && inputs_ok && near;
                    // kRecheckBuckets lists by the first pass's step count, longest first: the second pass then walks candidates
                    // of similar life time together (its warps stop together, its long CTAs start first)
                    const int bucket = kRecheckBuckets - 1 - min(kRecheckBuckets - 1, steps * kRecheckBuckets / H);
#pragma unroll
                    for (int b = 0; b < kRecheckBuckets; b++) {
                        const unsigned mk = __ballot_sync(0xffffffffu, push && bucket == b);
                        if (mk) {
                            const int leader = __ffs(mk) - 1;
                            unsigned base = 0;
                            if (lane == leader) base = atomicAdd(a.recheck_count + b, (unsigned)__popc(mk));
                            base = __shfl_sync(0xffffffffu, base, leader);
                            if (push && bucket == b) a.recheck[(long long)b * ncand + base + __popc(mk & ((1u << lane) - 1u))] = (int)li;
                        }
                    }
                }
                if (MODE == MODE_TICK && a.steps && valid) a.steps[li] = steps;   // mpmi_step_trace (a deferred candidate: overwritten by the second pass)
                if (MODE == MODE_TICK && valid && !push) {               // a5: this candidate's key
                    const bool safe = steps == H;
                    float d2 = 0.f;
#pragma unroll
                    for (int j = 0; j < kMaxM; j++) {
                        const float df = __fsub_rn(u[j], u_h[j]);
                        d2 = __fmaf_rn(df, df, d2);
                    }
                    const unsigned long long kk = make_key(safe, d2, H, steps, cfg.shard_begin + li);
                    key = kk < key ? kk : key;
                    n_safe += safe ? 1u : 0u;
                    n_exec += (unsigned)(steps + 1 < H ? steps + 1 : H);
                }
            }
        }
#ifdef MPMI_TC_DEBUG
        if (blockIdx.x == 0 && lane == 0 && (warp == 0 || warp == 4) && sw_n > 0)
            printf("state warp %d (clk/step): wait %lld ld %lld math+st-issue %lld wait_st+arrive %lld  wake after the MMA thread %lld  steps %lld\n",
                   warp, sw_wait / sw_n, sw_ld / sw_n, sw_math / sw_n, sw_st / sw_n, sw_skew / sw_n, sw_n);
#endif
    }

    // ---- teardown: all MMAs of this CTA have completed (the state warps waited for the last commit)
    fence_before_sync();
    __syncthreads();
    if (warp == kTcStateWarps) tc::tmem_dealloc<G::kTmemCols>(tb);
    if (MODE == MODE_BATCH) {
        if (tid == 0) {                          // the last CTA to finish re-arms the work counter for the next launch
            __threadfence();
            if (atomicAdd(&a.st->ticket, 1u) == gridDim.x - 1) { *a.work = 0u; a.st->ticket = 0u; __threadfence(); }
        }
        return;
    }
    // ---- a6 + a7
    block_select_and_finalise<kTcStateWarps + 1>(cfg, key, n_safe, n_exec, tick, u_h, a.st, a.out, a.partial, a.seq, a.work,
                                                  a.recheck != nullptr);
}

}  // namespace mpmi
