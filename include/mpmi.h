/*
 * mpmi.h -- C ABI of the B200-native MPMI-SC tick (Model Predictive Minimal Intervention Shared
 * Control; Broad, Murphey, Argall, arXiv 1906.02318, Algorithm 2).
 *
 * One control tick (readings G1-G13 in DESIGN.md section 3):
 *   1. sample N candidate inputs u_i over the input box: Philox4x32-10
 *      uniform or an endpoint-inclusive equally spaced grid; optionally inject the (clamped) user
 *      input u_h as candidate index N;
 *   2. lift the current state once, z_0 = Psi(x_t);
 *   3. roll every candidate H steps through z' = K z + B u_i, the same input held over the horizon
 *      (PAPER.md:120, 147-150, 304);
 *   4. after each step test the physical state x = z[0:n] against the safe set and stop at the first
 *      violation;
 *   5. return the safe candidate closest to u_h, key (||u_i-u_h||_2, i);
 *      if none is safe, the candidate with the most safe steps, then the lowest index.
 * All five steps run in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - Every function returns MPMI_OK (0) or a negative mpmi_status.  Nothing throws or aborts.
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device memory on the
 *     context's device.  mpmi_create copies everything it is given; the caller keeps ownership of
 *     all arrays passed to any function and may free host arrays as soon as the call returns.
 *     The library never frees or retains caller device pointers.
 *   - cuda_stream is a cudaStream_t cast to void* (NULL = the legacy default stream).
 *   - One context = one device = one tick in flight; a context is not thread-safe.
 *   - Arithmetic type of the path: IEEE fp32 (fused multiply-add), candidates and keys bit-exact
 *     integers / fp32 as defined below.
 */
#ifndef MPMI_H
#define MPMI_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MPMI_MAX_M       4     /* input dimension (one Philox call yields 4 words)     */
#define MPMI_MAX_N       16    /* physical state dimension                             */
#define MPMI_MAX_D       128   /* lifted dimension                                     */
#define MPMI_MAX_BOUNDS  32    /* box constraints accepted by mpmi_create              */
#define MPMI_MAX_CAND    ((1 << 30) - 2)

typedef enum {
    MPMI_OK = 0,
    MPMI_ERR_INVALID = -1,      /* null pointer, bad size, N != prod(grid), non-finite value ... */
    MPMI_ERR_UNSUPPORTED = -2,  /* d > MPMI_MAX_D, m > MPMI_MAX_M, n > MPMI_MAX_N, no sm_100 GPU */
    MPMI_ERR_CUDA = -3,         /* CUDA runtime error; text in mpmi_last_error                   */
    MPMI_ERR_NOMEM = -4
} mpmi_status;

enum { MPMI_SAMPLER_PHILOX = 0, MPMI_SAMPLER_GRID = 1 };
enum { MPMI_LIFT_MONO = 0, MPMI_LIFT_RFF = 1 };
enum { MPMI_DUMP_NONE = 0, MPMI_DUMP_PHYS = 1, MPMI_DUMP_LIFTED = 2 };
enum { MPMI_MODEL_LINEAR = 0,   /* z' = K z + B u, lifted once, x = z[0:n] (north_star)        */
       MPMI_MODEL_RELIFT = 1 }; /* x' = C (K Psi(x) + B u): the physical state is re-lifted before every
                                   step, the literal f(x, u) on states of PAPER.md:132 (G18)     */
/* mpmi_config.variant: speed knobs.  Flags and winner do not depend on them, with one documented exception: the latency
 * kernel associates each row sum as two chains (csrc/rollout_lat.cuh), so a candidate within rounding of a boundary can
 * differ between it and the other FP32 kernels (well inside tolerance T1). */
enum { MPMI_VARIANT_NARROW = 1,         /* 2 candidates per thread (latency)                  */
       MPMI_VARIANT_WIDE = 2,           /* 64/D candidates per thread (throughput)            */
       MPMI_VARIANT_NO_BINNING = 4,     /* never order the Philox candidates spatially        */
       MPMI_VARIANT_FORCE_BINNING = 8,  /* order them even for small N                        */
       MPMI_VARIANT_LATENCY = 16,       /* several lanes per candidate (d <= 32), any N       */
       MPMI_VARIANT_LAT_R2 = 32,        /* latency kernel: 2 rows per lane                    */
       MPMI_VARIANT_LAT_R4 = 64,        /* latency kernel: 4 rows per lane                    */
       MPMI_VARIANT_NO_TENSOR = 128,    /* d = 128: FP32 SIMT tile kernel instead of the 3xTF32
                                           tcgen05 kernel (results agree within the tolerances) */
       MPMI_VARIANT_AFFINE = 256,     /* noise-free linear model: x_k = a_k + G_k u (G_k tabulated at
                                           create, a_k per tick): n*m instead of d*(d+m) FMAs per
                                           sample-step; ignored with noise or the re-lift model   */
       MPMI_VARIANT_NO_PREDICT = 512,   /* d > 32: walk the candidates in input-box-cell order instead of
                                           the order of their predicted life time                 */
       MPMI_VARIANT_SMEM_MODEL = 2048,  /* d <= 32: model staged in shared memory (LDS.128) even where the constant
                                           bank would be chosen -- the variant a context falls back to when all
                                           constant-memory slots of its device are taken                      */
       MPMI_VARIANT_TC_UNVERIFIED = 4096, /* tensor-core kernels WITHOUT the verification below: the bare 3xTF32
                                           rollout (benchmark / test knob -- its flags are only as good as T1) */
       MPMI_VARIANT_TENSOR32 = 1024 };  /* padded d = 32: take the tensor-core tick for small candidate sets too */
/* The tensor-core tick (default at padded d = 128, and at padded d = 32 above 256 candidates per SM, ~38,000; linear model) is VERIFIED:
 * the 3xTF32 tcgen05 kernel rolls all candidates; every candidate whose state came within tau_i(k) of a safe-set
 * boundary is rolled again by the FP32 kernel (register kernel at d = 32, warp-tile kernel at d = 128), which merges
 * its keys and finalises, so that flags and winner are those of the FP32 tick.  tau_i(k) is a per-tick, per-step,
 * per-dimension bound on the difference between the two arithmetics, derived from the model (csrc/bound.cuh,
 * DESIGN.md section 6a).  The environment variable MPMI_TC_TAU_SCALE (0 <= v <= 16, read by mpmi_create) scales
 * tau: it measures how conservative the bound is and is not a tuning knob. */

/* Lift z = Psi(x).  The first n features MUST be the state itself.
 * MONO: feature f = product of up to 4 factors, codes terms[4f..4f+3]:
 *         0xFF = 1,  0x00+j = x_j,  0x40+j = sin(x_j),  0x80+j = cos(x_j)   (j < n).
 * RFF:  feature f<n = x_f;  feature n+r = scale * cos(W[r,:] . x + b[r]),  W is (d-n) x n row-major. */
typedef struct {
    int32_t        kind;      /* MPMI_LIFT_*                          */
    const uint8_t *terms;     /* host, d*4 (MONO)                     */
    const float   *W;         /* host, (d-n)*n (RFF)                  */
    const float   *b;         /* host, d-n (RFF)                      */
    float          scale;     /* RFF                                  */
} mpmi_lift_spec;

/* Safe set: AND of
 *   box constraints   lo[q] + inflate <  x[idx[q]]  <  hi[q] - inflate   (strict; +-INFINITY allowed)
 *   optional annulus  rmin + inflate <= hypot(x[ix]-cx, x[iy]-cy) <= rmax - inflate   (closed)
 * Only constrained dims (box idx, annulus ix / iy) are tested: NaN or Inf there is unsafe, an unconstrained
 * physical dim is never looked at (same rule in every kernel and in the oracle).
 * inflate is the hand-tuned inflation radius of PAPER.md:221. */
typedef struct {
    int32_t        nbounds;
    const int32_t *idx;       /* host, nbounds, each < n              */
    const float   *lo;        /* host, nbounds                        */
    const float   *hi;        /* host, nbounds                        */
    int32_t        annulus;   /* 0 / 1                                */
    int32_t        ix, iy;
    float          cx, cy, rmin, rmax;
    float          inflate;
} mpmi_safe_spec;

typedef struct {
    int32_t  n, m, d;         /* physical state, input, lifted dims   */
    int32_t  N;               /* sampled candidates per tick (10,000 / 10,120)       */
    int32_t  H;               /* horizon T in steps (30 / 25)                        */
    const float *K;           /* host, d*d row-major                  */
    const float *B;           /* host, d*m row-major                  */
    const float *u_lo, *u_hi; /* host, m each: the input box                   */
    int32_t  sampler;         /* MPMI_SAMPLER_*                       */
    const int32_t *grid_counts;/* host, m, product == N (GRID only); row-major, dim 0 slowest      */
    uint64_t seed;            /* Philox key                           */
    int32_t  include_user;    /* 1: clamp(u_user) is candidate index N (N+1 rollouts per tick)     */
    mpmi_lift_spec lift;
    mpmi_safe_spec safe;
    int32_t  device;          /* CUDA device ordinal, -1 = current device                          */
    /* Candidate sharding across GPUs: this context owns the global candidate
     * indices [shard_begin, shard_begin + shard_count) of the N (+1) candidates; 0,0 = all of them. */
    int64_t  shard_begin, shard_count;
    int32_t  variant;         /* 0 = automatic; else OR of MPMI_VARIANT_* (benchmark / test knobs)  */
    /* Additive Gaussian white noise of Algorithm 2 l.5, "x_p <- f(x_p, xi(i)) + z_i":
     * sigma * eps, eps ~ N(0, I_n), is added to the n physical rows of every predicted state before
     * isSafe and stays in the state that is carried on; one independent draw per (tick, candidate, step,
     * dim) from the Philox4x32-10 stream key = (seed_lo, seed_hi ^ 0x6E6F6973), counter = (i, (q << 16) | k,
     * tick_lo, tick_hi), q = dim / 4, Box-Muller on (w0, w1) and (w2, w3) (G17).  0 = none. */
    float    noise_sigma;
    int32_t  model;           /* MPMI_MODEL_* : how f(x, u) is evaluated                            */
    int32_t  reserved;
} mpmi_config;

/* Result of one tick.  Same layout on host and device. */
typedef struct {
    float    u[4];            /* selected input u_r (bit-identical to candidate `index`)            */
    int32_t  index;           /* winner, in [0, N]; N = the injected user input                     */
    int32_t  safe;            /* 1: safe over the whole horizon; 0: fallback (no candidate was safe)*/
    int32_t  steps;           /* safe predicted states before the first violation, in [0, H]        */
    int32_t  n_safe;          /* number of safe candidates (control-style metric)     */
    float    dist;            /* ||u_r - u_h||_2 (control-skill metric)               */
    int32_t  reserved;
    int64_t  n_exec;          /* executed sample-steps: sum_i min(steps_i + 1, H)                   */
    uint64_t key;             /* packed selection key of the winner       */
} mpmi_result;

/* Partial result of one shard: what a rank contributes to the 24-byte exchange of section 8. */
typedef struct {
    uint64_t key;             /* min key over the shard (bit 63 always 0, so int64 order == order)  */
    int64_t  n_safe;
    int64_t  n_exec;
} mpmi_partial;

typedef struct {
    int32_t  d_pad;           /* internal padded lifted dim (zero rows / columns: exact)            */
    int32_t  variant;         /* 1 = register-resident FFMA2 (d<=32), 2 = warp-tile FFMA2 (d<=128),
                                 3 = latency kernel, 4 lanes per candidate (d<=32, small N),
                                 4 = verified 3xTF32 tcgen05 tensor-core tick (d_pad = 128; d_pad = 32 above 256 candidates per SM),
                                 5 = re-lift kernel (MPMI_MODEL_RELIFT), 6 = affine-in-u kernel       */
    int32_t  cand_per_block, threads_per_block, blocks, smem_bytes, regs_per_thread;
    int32_t  sm_count, launches_per_tick, uses_graph;
    int32_t  binning_cells;   /* 0 = candidates walked in index order; else cells of the spatial pre-sort */
    int32_t  reserved;        /* verified tensor-core tick: candidates the last finished mpmi_step tick handed to the FP32 pass; else 0 */
    int64_t  ncand_local;     /* candidates this context rolls out per tick                         */
} mpmi_info;

typedef struct mpmi_ctx mpmi_ctx;   /* opaque, owned by the library */

/* Validate cfg, copy it, upload K / B / tables, choose the kernel, build the tick graph.
 * Errors: INVALID (null, n/m/d/N/H <= 0, N != prod(grid_counts), u_lo > u_hi, non-finite K/B/box,
 * lift's first n features not the identity, bound idx >= n, shard outside [0, N+include_user]),
 * UNSUPPORTED (limits above, device is not compute capability 10.x), CUDA, NOMEM. */
int mpmi_create(const mpmi_config *cfg, mpmi_ctx **out);
void mpmi_destroy(mpmi_ctx *ctx);

/* One tick, MPMI-SC(t, x_t, u_h) -> u_r.  x0: host, n floats.  u_user: host,
 * m floats; values outside the box are clamped (bounded joystick).  tick selects the
 * Philox sample set (fresh samples each tick; the grid ignores it).
 * mpmi_step enqueues the tick on cuda_stream and returns; mpmi_step_result waits for it and copies
 * the result to out (host).  mpmi_step_sync = both.  Non-finite x0 / u_user -> INVALID. */
int mpmi_step(mpmi_ctx *ctx, const float *x0, const float *u_user, uint64_t tick, void *cuda_stream);
int mpmi_step_result(mpmi_ctx *ctx, mpmi_result *out);
int mpmi_step_sync(mpmi_ctx *ctx, const float *x0, const float *u_user, uint64_t tick,
                   void *cuda_stream, mpmi_result *out);

/* Same tick with everything resident on the device: d_x0 (n floats), d_u_user (m floats) are read
 * and d_out (one mpmi_result) is written by the kernels on cuda_stream; asynchronous.  Non-finite
 * inputs give a result with index = -1. */
int mpmi_step_device(mpmi_ctx *ctx, const float *d_x0, const float *d_u_user, uint64_t tick,
                     void *cuda_stream, mpmi_result *d_out);

/* Diagnostic twin of mpmi_step_device: the SAME kernels in the SAME launch configuration (binning, tensor-core first
 * pass + FP32 second pass, ...), which additionally store the step count of every local candidate as the tick kernels
 * decided it: d_steps (device, ncand_local int32; entry = global candidate index - shard_begin; the injected user
 * input is the last entry of the shard that owns index N) = safe predicted states before the first violation
 * (H <=> safe).  This is what the full-size parity tests compare with the oracle candidate by
 * candidate; the extra 4-byte store per candidate is the only difference to mpmi_step_device.  Asynchronous. */
int mpmi_step_trace(mpmi_ctx *ctx, const float *d_x0, const float *d_u_user, uint64_t tick,
                    void *cuda_stream, mpmi_result *d_out, int32_t *d_steps);

/* Measurement aid for bench.py's roofline: while enabled, the plain-launch entries (mpmi_step_device, mpmi_step_trace,
 * mpmi_shard_step) record CUDA events on cuda_stream before the tick kernel, after it and after the second pass of a
 * verified tensor-core tick (three event records per tick, no synchronisation).  mpmi_profile_read waits for the
 * recorded ticks and returns, oldest first, the device time of the tick kernel and of the second pass (0 if there is
 * none) of the last `*count` <= min(capacity, 64) ticks, in milliseconds (host arrays). */
int mpmi_profile_enable(mpmi_ctx *ctx, int32_t enable);
/* Stage timeline of a paper-scale tick (latency kernel, info.variant == 3; else UNSUPPORTED): while d_stamps (device,
 * 8 * info.blocks uint64) is set, the plain-launch entries make thread 0 of every CTA store %globaltimer (ns) at
 * [0] kernel entry, [1] model rows requested, [2] lift done, [3] candidate sampled, [4] horizon loop left,
 * [5] keys reduced and ticket taken; NULL switches it off. */
int mpmi_profile_timeline(mpmi_ctx *ctx, uint64_t *d_stamps);
int mpmi_profile_read(mpmi_ctx *ctx, int32_t capacity, int32_t *count, float *ms_tick_kernel, float *ms_second_pass);

/* Sharded tick (section 8(e)): roll out this context's shard and write its mpmi_partial to
 * d_partial (device).  After the caller has gathered the G partials of all ranks into d_partials
 * (device, G entries), mpmi_shard_finalize reduces them (min key, summed counters), regenerates
 * the winning input from its index and writes the full result to d_out (device).  Asynchronous. */
int mpmi_shard_step(mpmi_ctx *ctx, const float *d_x0, const float *d_u_user, uint64_t tick,
                    void *cuda_stream, mpmi_partial *d_partial);
int mpmi_shard_finalize(mpmi_ctx *ctx, const mpmi_partial *d_partials, int32_t G,
                        const float *d_u_user, uint64_t tick, void *cuda_stream, mpmi_result *d_out);

/* Rollouts without selection, for benchmarking and parity (trajectory cloud of Fig. 1).
 *   d_U     device, Ncand*m row-major, or NULL = internal sampler (indices 0..Ncand-1, `tick`)
 *   d_X0    device, x0_count*n row-major; x0_count is 1 (shared) or Ncand (per candidate)
 *   H       horizon for this call (<= 65535)
 *   d_traj  device or NULL; dump_kind PHYS: H*n*Ncand floats, LIFTED: H*d*Ncand floats, laid out
 *           traj[(k*J + j)*Ncand + i] = component j of z_{k+1} of candidate i (candidate fastest);
 *           entries after a candidate's first violating state are NaN; with MPMI_MODEL_RELIFT a LIFTED
 *           dump holds the carried state Psi(x_{k+1}); with noise the dumped state includes it
 *   d_steps device, Ncand int32: safe predicted states before the first violation (H <=> safe)
 *   d_safe  device or NULL, Ncand bytes: 1 iff steps == H
 * Asynchronous on cuda_stream. */
int mpmi_rollout_batch(mpmi_ctx *ctx, const float *d_U, const float *d_X0, int64_t x0_count,
                       int64_t Ncand, int32_t H, int32_t dump_kind, float *d_traj,
                       int32_t *d_steps, uint8_t *d_safe, uint64_t tick, void *cuda_stream);

/* One whole tick WITHOUT a context and without any allocation (csrc/noalloc.cu) -- for callers that may not call
 * cudaMalloc: code under stream capture, tight serving loops, harnesses that forbid it.  The call enqueues two kernels on
 * cuda_stream (model pack + the shared-memory-model register tick kernel, the FP32 path of Algorithm 2,
 * PAPER.md:137-173) and returns; it calls no cudaMalloc / cudaFree / cudaHostAlloc, creates no graph, stream or event.
 *   cfg       host struct as for mpmi_create, EXCEPT that the tables K (d*d), B (d*m), lift.terms (d*4, MONO), lift.W,
 *             lift.b (RFF) are DEVICE pointers here (read by the kernels, not validated: the requirements of mpmi_create
 *             on them are the caller's to keep); u_lo, u_hi, grid_counts, safe.idx / lo / hi stay host arrays, read
 *             during the call.  variant is ignored.  Runs on the CURRENT device; cfg->device must be -1 or that device.
 *   d_x0, d_u_user, d_out   device, as for mpmi_step_device; the result is the one mpmi_step_device gives for the same
 *             configuration: bit-identical where that context runs the register kernel (info.variant == 1, e.g. with
 *             MPMI_VARIANT_NARROW | MPMI_VARIANT_NO_TENSOR); against the latency kernel, whose row sums are associated
 *             differently, a candidate within rounding of the boundary may differ, as between those two kernels.
 * Limits: d <= 32 (the kernels' scratch -- the packed model and the cross-CTA selection state -- lives in ONE static
 * 8 KB __device__ array per GPU, held until the process exits), linear model, noise_sigma == 0, the whole candidate set
 * (shard 0,0).  Beyond them: MPMI_ERR_UNSUPPORTED, text in mpmi_noalloc_last_error (per host thread, valid until the
 * next call).  Every call on a GPU shares that array and re-initialises it: calls whose kernels OVERLAP on the GPU
 * (different streams, or several host threads) race on it -- serialise them.  Asynchronous. */
int mpmi_tick_noalloc(const mpmi_config *cfg, const float *d_x0, const float *d_u_user, uint64_t tick,
                      void *cuda_stream, mpmi_result *d_out);
const char *mpmi_noalloc_last_error(void);

int mpmi_get_info(const mpmi_ctx *ctx, mpmi_info *out);
const char *mpmi_strerror(int status);
const char *mpmi_last_error(const mpmi_ctx *ctx);   /* "" if none; valid until the next call on ctx */

#ifdef __cplusplus
}
#endif
#endif /* MPMI_H */
