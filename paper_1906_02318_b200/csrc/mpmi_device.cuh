// mpmi_device.cuh -- device-side building blocks of the MPMI-SC tick (Algorithm 2):
// sampler (a1), lift (a2), safe test (a4), selection key (a5), reductions (a6), finalise (a7).
// sm_100a only.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/mpmi.h"

namespace mpmi {

constexpr int kMaxM = MPMI_MAX_M;
constexpr int kMaxN = MPMI_MAX_N;

// Everything the kernels need, passed by value as a __grid_constant__ kernel parameter so that
// bounds, box limits and sampler constants are direct constant-bank operands.
struct DevCfg {
    int n, m, d, D;                 // D = padded lifted dim (zero rows / columns)
    int N, H, include_user;
    long long ncand_global;         // N + include_user
    long long shard_begin, shard_count;
    int sampler;
    int grid_counts[kMaxM];
    unsigned seed_lo, seed_hi;
    float u_lo[kMaxM], u_hi[kMaxM];
    int lift_kind;
    float rff_scale;
    unsigned bmask;                 // bit j set: internal physical dim j has a box constraint
    float blo[kMaxN], bhi[kMaxN];   // per INTERNAL dimension limits, inflation folded in (+-inf if none)
    int annulus;                    // annulus on INTERNAL dims 0,1
    float cx, cy, rmin2, rmax2;     // inflation folded in, squared
    unsigned char perm[kMaxN];      // internal physical dim j = original dim perm[j] (annulus / box dims first)
    const float *KTa;               // device: augmented transposed model, layout per variant
    const float *Kpad;              // device: D*D row-major padded K (tile variant)
    const float *Bpad;              // device: D*4 row-major padded B
    const uint8_t *terms;           // device: D*4 lift factor codes (MONO)
    const float *W, *b;             // device: RFF tables
    float noise_sigma;              // std of the additive prediction noise (Alg. 2 l.5); 0 = none
    int model;                      // MPMI_MODEL_*
    // affine-in-u fast path (rollout_affine.cuh): x_k = a_k + G_k u
    float *aff_a;                   // device: H x aff_np, written per tick by affine_base_kernel
    const float *aff_g;             // device: H x m x aff_np, from mpmi_create (FP64 -> fp32)
    const float *aff_m;             // device: H x aff_np x D, rows of C K^k (FP64 -> fp32)
    int aff_np;                     // padded physical dim: 4, 8 or 16
    // verified tensor-core tick (bound.cuh): tables of mpmi_create (FP64 -> fp32) and the two per-tick results
    const float *bnd_kpow;          // device: H x D x D, kpowT[j][c][r] = (K^j)[r][c], internal order
    const float *bnd_mid;           // device: H x D, (S_j B) u_mid
    const float *bnd_econst;        // device: H x D, tick-independent part of the per-step error bound E
    const float *bnd_w;             // device: D + M column weights w_c of E
    float *bnd_e;                   // device: H x D, E[j][r] of this tick (bound_err_kernel)
    float *bnd_tau;                 // device: (H + 1) x (aff_np + 4), tau_i(k) of this tick (bound_tau_kernel)
};

// Cross-block selection state; reset by the block that finalises the tick.
struct TickState {
    unsigned long long best_key;
    unsigned long long n_exec;
    unsigned int n_safe;
    unsigned int ticket;
    unsigned int work;          // next candidate batch of the persistent tile kernel
    unsigned int pad;
};

constexpr unsigned long long kKeyNone = 0x7FFFFFFFFFFFFFFFull;
constexpr int kKeyIndexBits = 30;

// ---- a1: Philox4x32-10 (Salmon et al. SC'11), counter-based; DESIGN G4 ------------------------
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3,
                                              unsigned k0, unsigned k1, unsigned (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const unsigned hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const unsigned n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// candidate input u_i for GLOBAL index gi.  gi == N is the injected u_h.
__device__ __forceinline__ void sample_u(const DevCfg &cfg, long long gi, unsigned long long tick,
                                         const float (&u_h)[kMaxM], float (&u)[kMaxM]) {
#pragma unroll
    for (int j = 0; j < kMaxM; j++) u[j] = 0.0f;
    if (gi >= cfg.N) {
#pragma unroll
        for (int j = 0; j < kMaxM; j++) u[j] = u_h[j];
        return;
    }
    if (cfg.sampler == MPMI_SAMPLER_PHILOX) {
        unsigned w[4];
        philox4x32_10((unsigned)gi, (unsigned)((unsigned long long)gi >> 32), (unsigned)tick,
                      (unsigned)(tick >> 32), cfg.seed_lo, cfg.seed_hi, w);
#pragma unroll
        for (int j = 0; j < kMaxM; j++) {
            if (j < cfg.m) {
                const float r = __uint2float_rn(w[j] >> 8) * 0x1p-24f;       // exact
                u[j] = __fmaf_rn(r, __fsub_rn(cfg.u_hi[j], cfg.u_lo[j]), cfg.u_lo[j]);
            }
        }
    } else {
        long long rem = gi;                                                    // row-major, dim 0 slowest
#pragma unroll
        for (int j = kMaxM - 1; j >= 0; j--) {
            if (j < cfg.m) {
                const int cnt = cfg.grid_counts[j];
                const int k = (int)(rem % cnt);
                rem /= cnt;
                const float lo = cfg.u_lo[j], hi = cfg.u_hi[j];
                float v;
                if (cnt == 1)          v = __fmul_rn(0.5f, __fadd_rn(lo, hi));
                else if (k == cnt - 1) v = hi;
                else                   v = __fmaf_rn(__fdiv_rn((float)k, (float)(cnt - 1)), __fsub_rn(hi, lo), lo);
                u[j] = v;
            }
        }
    }
}

// Algorithm 2 l.5 noise z_i (DESIGN G17): four standard normals for the original physical
// dims 4q..4q+3 of candidate gi at step k, Box-Muller on the Philox words (w0, w1) and (w2, w3).
__device__ __forceinline__ void noise4(const DevCfg &cfg, long long gi, int k, int q, unsigned long long tick, float (&g)[4]) {
    unsigned w[4];
    philox4x32_10((unsigned)gi, ((unsigned)q << 16) | (unsigned)k, (unsigned)tick, (unsigned)(tick >> 32),
                  cfg.seed_lo, cfg.seed_hi ^ 0x6E6F6973u, w);
#pragma unroll
    for (int h = 0; h < 2; h++) {
        g[2 * h] = 0.f; g[2 * h + 1] = 0.f;
        if (4 * q + 2 * h >= cfg.n) continue;                                              // dims beyond n: no transform (uniform)
        const float u1 = __fmaf_rn(__uint2float_rn(w[2 * h] >> 8), 0x1p-24f, 0x1p-24f);   // ((w >> 8) + 1) 2^-24, exact
        const float u2 = __uint2float_rn(w[2 * h + 1] >> 8) * 0x1p-23f;                    // 2 u2: angle in units of pi
        const float r = sqrtf(-2.0f * logf(u1));
        float sn, cs;
        sincospif(u2, &sn, &cs);
        g[2 * h] = r * cs;
        g[2 * h + 1] = r * sn;
    }
}

__device__ __forceinline__ void clamp_user(const DevCfg &cfg, const float *u_user, float (&u_h)[kMaxM]) {
#pragma unroll
    for (int j = 0; j < kMaxM; j++) {
        float v = 0.0f;
        if (j < cfg.m) {
            v = u_user[j];
            v = v < cfg.u_lo[j] ? cfg.u_lo[j] : v;
            v = v > cfg.u_hi[j] ? cfg.u_hi[j] : v;
        }
        u_h[j] = v;
    }
}

// ---- a2: lift, one feature.  Accurate sinf/cosf (no fast-math). ------------
__device__ __forceinline__ float lift_factor(unsigned code, const float *x) {
    if (code == 0xFFu) return 1.0f;
    const float v = x[code & 0x3Fu];
    const unsigned kind = code >> 6;
    return kind == 0 ? v : (kind == 1 ? sinf(v) : cosf(v));
}
__device__ __forceinline__ float lift_feature(const DevCfg &cfg, int f, const float *x) {
    // f is the INTERNAL feature index; x is the state in the caller's order
    if (f >= cfg.d) return 0.0f;                       // zero padding
    if (f < cfg.n) return x[cfg.perm[f]];
    if (cfg.lift_kind == MPMI_LIFT_MONO) {
        const uint8_t *t = cfg.terms + 4 * f;
        float p = lift_factor(t[0], x);
        p = __fmul_rn(p, lift_factor(t[1], x));
        p = __fmul_rn(p, lift_factor(t[2], x));
        p = __fmul_rn(p, lift_factor(t[3], x));
        return p;
    }
    const int r = f - cfg.n;
    float s = cfg.b[r];
    for (int j = 0; j < cfg.n; j++) s = __fmaf_rn(cfg.W[r * cfg.n + j], x[j], s);
    return __fmul_rn(cfg.rff_scale, cosf(s));
}

// ---- a5: selection key.  bit 63 = 0, bit 62 = unsafe, bits 61..30 = primary, bits 29..0 = index.
// safe:   primary = bits of the fp32 squared distance (monotone for >= 0);
// unsafe: primary = H - steps  (most safe steps first).  Lexicographic order == integer order.
__device__ __forceinline__ unsigned long long make_key(bool safe, float dist2, int H, int steps, long long gi) {
    const unsigned primary = safe ? __float_as_uint(dist2) : (unsigned)(H - steps);
    return ((unsigned long long)(safe ? 0 : 1) << 62) | ((unsigned long long)primary << kKeyIndexBits) |
           (unsigned long long)gi;
}

__device__ __forceinline__ unsigned long long shfl_xor_u64(unsigned long long v, int lane_mask) {
    unsigned lo = (unsigned)v, hi = (unsigned)(v >> 32);
    lo = __shfl_xor_sync(0xffffffffu, lo, lane_mask);
    hi = __shfl_xor_sync(0xffffffffu, hi, lane_mask);
    return ((unsigned long long)hi << 32) | lo;
}
__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const unsigned long long w = shfl_xor_u64(v, o);
        v = w < v ? w : v;
    }
    return v;
}
__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += shfl_xor_u64(v, o);
    return v;
}
__device__ __forceinline__ unsigned warp_sum_u32(unsigned v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- a6 (block part) + a7: block min -> one 64-bit atomicMin per block; the last block to arrive
// decodes the key, regenerates the winning input from its index and writes the result.
// If `partial` is non-null the block writes the shard's mpmi_partial instead (multi-GPU path).
__device__ __forceinline__ void decode_result(const DevCfg &cfg, unsigned long long key, unsigned long long n_exec,
                                              unsigned n_safe, unsigned long long tick,
                                              const float (&u_h)[kMaxM], mpmi_result *out, unsigned seq = 0) {
    mpmi_result r;
    const long long gi = (long long)(key & ((1ull << kKeyIndexBits) - 1));
    const bool safe = ((key >> 62) & 1ull) == 0;
    const unsigned primary = (unsigned)(key >> kKeyIndexBits);
    float u[kMaxM];
    sample_u(cfg, gi, tick, u_h, u);
    float d2 = 0.0f;
#pragma unroll
    for (int j = 0; j < kMaxM; j++) {
        r.u[j] = u[j];
        const float df = __fsub_rn(u[j], u_h[j]);
        d2 = __fmaf_rn(df, df, d2);
    }
    r.index = (int)gi;
    r.safe = safe ? 1 : 0;
    r.steps = safe ? cfg.H : cfg.H - (int)primary;
    r.n_safe = (int)n_safe;
    r.dist = sqrtf(d2);
    r.reserved = 0;
    r.n_exec = (long long)n_exec;
    r.key = key;
    if (key == kKeyNone) { r.index = -1; r.safe = 0; r.steps = 0; r.dist = 0.0f; }
    *out = r;
    if (seq) {                       // out is host-mapped: publish the sequence number after the payload
        __threadfence_system();
        *reinterpret_cast<volatile int *>(&out->reserved) = (int)seq;
    }
}

template <int kWarps>
__device__ __forceinline__ void block_select_and_finalise(const DevCfg &cfg, unsigned long long key,
                                                          unsigned n_safe, unsigned long long n_exec,
                                                          unsigned long long tick, const float (&u_h)[kMaxM],
                                                          TickState *st, mpmi_result *out, mpmi_partial *partial,
                                                          unsigned seq = 0, unsigned *work = nullptr, bool defer = false,
                                                          unsigned *lists = nullptr, int nlists = 0, int *deferred_out = nullptr) {
    __shared__ unsigned long long s_key[kWarps];
    __shared__ unsigned s_safe[kWarps];
    __shared__ unsigned long long s_exec[kWarps];
    __shared__ bool s_last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    key = warp_min_u64(key);
    n_safe = warp_sum_u32(n_safe);
    n_exec = warp_sum_u64(n_exec);
    if (lane == 0) { s_key[warp] = key; s_safe[warp] = n_safe; s_exec[warp] = n_exec; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long k = s_key[0];
        unsigned ns = s_safe[0];
        unsigned long long ne = s_exec[0];
#pragma unroll
        for (int w = 1; w < kWarps; w++) {
            if (w * 32 < (int)blockDim.x) { k = s_key[w] < k ? s_key[w] : k; ns += s_safe[w]; ne += s_exec[w]; }
        }
        if (k != kKeyNone) atomicMin(&st->best_key, k);
        if (ns) atomicAdd(&st->n_safe, ns);
        if (ne) atomicAdd(&st->n_exec, ne);
        __threadfence();
        const unsigned t = atomicAdd(&st->ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last && defer) {          // a later kernel of this tick merges its candidates and finalises: only re-arm the counters
            st->ticket = 0u;
            if (work) *work = 0u;
            __threadfence();
        } else if (s_last) {
            __threadfence();
            const unsigned long long bk = atomicMin(&st->best_key, kKeyNone);     // atomic read
            const unsigned long long tot_exec = atomicAdd(&st->n_exec, 0ull);
            const unsigned tot_safe = atomicAdd(&st->n_safe, 0u);
            if (lists) {                 // second pass of a verified tick: empty the deferral lists, report how many it rolled
                unsigned tot = 0;
                for (int i = 0; i < nlists; i++) { tot += lists[i]; lists[i] = 0u; }
                lists[nlists] = 0u;      // (the block counter of the second pass, kept behind the list counters)
                st->pad = tot;
                if (deferred_out) *reinterpret_cast<volatile int *>(deferred_out) = (int)tot;     // (mapped: before the sequence number)
            }
            if (partial) {
                partial->key = bk; partial->n_safe = tot_safe; partial->n_exec = (long long)tot_exec;
            } else {
                decode_result(cfg, bk, tot_exec, tot_safe, tick, u_h, out, seq);
            }
            st->best_key = kKeyNone; st->n_exec = 0ull; st->n_safe = 0u; st->ticket = 0u;   // ready for next tick
            if (work) *work = 0u;
            __threadfence();
        }
    }
}

__device__ __forceinline__ bool finite_inputs(const DevCfg &cfg, const float *x0, const float *u_user) {
    bool ok = true;
    for (int j = 0; j < cfg.n; j++) ok = ok && isfinite(x0[j]);
    for (int j = 0; j < cfg.m; j++) ok = ok && isfinite(u_user[j]);
    return ok;
}

// acc += k * z on a candidate pair: one FFMA2 (fma.rn.f32x2) with the model value broadcast to both
// halves.  Written as in-place PTX ("+l") so that ptxas keeps the accumulator where it is; the
// intrinsic form made it rotate accumulators through MOVs in partially unrolled loops.
__device__ __forceinline__ void fma2_bcast(float2 &acc, float k, const float2 &z) {
    unsigned long long kk, zz, aa;
    asm("mov.b64 %0, {%1,%1};" : "=l"(kk) : "f"(k));
    asm("mov.b64 %0, {%1,%2};" : "=l"(zz) : "f"(z.x), "f"(z.y));
    asm("mov.b64 %0, {%1,%2};" : "=l"(aa) : "f"(acc.x), "f"(acc.y));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(aa) : "l"(kk), "l"(zz));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(acc.x), "=f"(acc.y) : "l"(aa));
}
// acc += kpair * z on a ROW pair of one candidate: the state value is the broadcast operand
__device__ __forceinline__ void fma2_bcast_z(float2 &acc, const float2 &k, float z) {
    unsigned long long kk, zz, aa;
    asm("mov.b64 %0, {%1,%2};" : "=l"(kk) : "f"(k.x), "f"(k.y));
    asm("mov.b64 %0, {%1,%1};" : "=l"(zz) : "f"(z));
    asm("mov.b64 %0, {%1,%2};" : "=l"(aa) : "f"(acc.x), "f"(acc.y));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(aa) : "l"(kk), "l"(zz));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(acc.x), "=f"(acc.y) : "l"(aa));
}
// acc = kpair * z (first column of a step, row-pair form)
__device__ __forceinline__ void mul2_bcast_z(float2 &acc, const float2 &k, float z) {
    unsigned long long kk, zz, aa;
    asm("mov.b64 %0, {%1,%2};" : "=l"(kk) : "f"(k.x), "f"(k.y));
    asm("mov.b64 %0, {%1,%1};" : "=l"(zz) : "f"(z));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(aa) : "l"(kk), "l"(zz));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(acc.x), "=f"(acc.y) : "l"(aa));
}
// acc = k * z (first column of a step)
__device__ __forceinline__ void mul2_bcast(float2 &acc, float k, const float2 &z) {
    unsigned long long kk, zz, aa;
    asm("mov.b64 %0, {%1,%1};" : "=l"(kk) : "f"(k));
    asm("mov.b64 %0, {%1,%2};" : "=l"(zz) : "f"(z.x), "f"(z.y));
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(aa) : "l"(kk), "l"(zz));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(acc.x), "=f"(acc.y) : "l"(aa));
}

// ---- a4: isSafe(x) -----------------------------------------------------
// box limits on internal dims 0..nbox-1 (strict), annulus on internal dims 0,1 (closed); NaN -> unsafe
template <int NB>
__device__ __forceinline__ bool safe_check(const DevCfg &cfg, const float (&x)[NB], int nbox) {
    bool ok = true;
    if (nbox > 0) {
#pragma unroll
        for (int j = 0; j < 2 && j < NB; j++) ok = ok && (x[j] > cfg.blo[j]) && (x[j] < cfg.bhi[j]);
        if (nbox > 2) {
#pragma unroll
            for (int j = 2; j < 4 && j < NB; j++) ok = ok && (x[j] > cfg.blo[j]) && (x[j] < cfg.bhi[j]);
            if (nbox > 4) {
#pragma unroll
                for (int j = 4; j < 8 && j < NB; j++) ok = ok && (x[j] > cfg.blo[j]) && (x[j] < cfg.bhi[j]);
                if (nbox > 8) {
#pragma unroll
                    for (int j = 8; j < 16 && j < NB; j++) ok = ok && (x[j] > cfg.blo[j]) && (x[j] < cfg.bhi[j]);
                }
            }
        }
    }
    if (cfg.annulus) {
        const float dx = __fsub_rn(x[0], cfg.cx), dy = __fsub_rn(x[1], cfg.cy);
        const float r2 = __fmaf_rn(dx, dx, __fmul_rn(dy, dy));
        ok = ok && (r2 >= cfg.rmin2) && (r2 <= cfg.rmax2);
    }
    return ok;
}

// NaN-propagating minimum (min.NaN.f32): the safe test as one tree instead of a chain of predicate ANDs
__device__ __forceinline__ float min_nan(float a, float b) {
    float d;
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
    return d;
}

__device__ __forceinline__ float4 lds128(unsigned addr) {
    // volatile: keeps the compiler from hoisting the (loop-invariant) model loads out of the
    // horizon loop, which would spill ~D*D registers
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

// 8-byte global store at base + 4*off (off in floats, warp-uniform): written as PTX so that the
// address stays one IMAD.WIDE instead of being re-associated into 64-bit element arithmetic
__device__ __forceinline__ void stg64_off(unsigned long long base, unsigned off, const float2 &v) {
    asm volatile("{\n\t.reg .u64 a;\n\tmad.wide.u32 a, %0, 4, %1;\n\tst.global.v2.f32 [a], {%2,%3};\n\t}"
                 :: "r"(off), "l"(base), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void stg64_off_if(unsigned long long base, unsigned off, const float2 &v, bool pred) {
    asm volatile("{\n\t.reg .u64 a;\n\t.reg .pred p;\n\tsetp.ne.u32 p, %4, 0;\n\tmad.wide.u32 a, %0, 4, %1;\n\t"
                 "@p st.global.v2.f32 [a], {%2,%3};\n\t}"
                 :: "r"(off), "l"(base), "f"(v.x), "f"(v.y), "r"((unsigned)pred) : "memory");
}

}  // namespace mpmi
