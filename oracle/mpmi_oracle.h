/*
 * mpmi_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU restatement of Algorithm 2 (MPMI-SC) of Broad, Murphey, Argall,
 * "Highly Parallelized Data-driven MPC for Minimal Intervention Shared Control"
 * (PAPER.md:134-174), with the readings listed in DESIGN.md section 3 where the paper is silent.
 *
 * Only tests/, __graft_entry__.smoke(), bench.py's cpu_baseline leg / `--impl reference`
 * and oracle/calibrate.py may call this.  It shares no code with paper_1906_02318_b200/csrc.
 *
 * Pins (tests/test_oracle_pins.py): closed form z_H = K^H z0 + sum K^k B u, geometric series,
 * brute force on tiny inputs, Philox known-answer vectors, Eq. (2) printed value 0.0001,
 * K=0 / K=rho*I / B=0 special cases, prefix / monotone / shard invariants, lift hand values;
 * noise (NEXT-2): normal moments + Kolmogorov-Smirnov against the normal CDF, closed form
 * z_H = K^H z0 + sum K^(H-1-k) (B u + E eps_k); re-lift model (NEXT-3): reduction to the textbook
 * linear recursion x' = A x + B u when K[0:n, n:] = 0, an independent Python loop on a tiny system,
 * identity lift == linear model.
 * Functions with no pin: none ("parity unpinned" would be stated here).
 */
#ifndef MPMI_ORACLE_H
#define MPMI_ORACLE_H
#include <stdint.h>

enum { ORC_SAMPLER_PHILOX = 0, ORC_SAMPLER_GRID = 1 };
enum { ORC_LIFT_MONO = 0, ORC_LIFT_RFF = 1 };
enum { ORC_MODEL_LINEAR = 0,  /* z' = K z + B u, lifted once, x = z[0:n]                   */
       ORC_MODEL_RELIFT = 1 };/* x' = C (K Psi(x) + B u): re-lift the physical state every step */

typedef struct {
    int32_t n, m, d, N, H;
    const double *K;          /* d*d row-major (fp32 model values promoted)          */
    const double *B;          /* d*m row-major                                       */
    const float  *u_lo, *u_hi;/* m each; the sampler is DEFINED in fp32 (DESIGN G4)  */
    int32_t sampler;          /* ORC_SAMPLER_*                                       */
    const int32_t *grid_counts; /* m, product == N (grid sampler only)               */
    uint64_t seed;
    int32_t include_user;     /* 1: u_user (clamped to the box) is candidate index N */
    int32_t lift_kind;        /* ORC_LIFT_*                                          */
    const uint8_t *terms;     /* MONO: d*4 factor codes                              */
    const double *W;          /* RFF: (d-n)*n row-major                              */
    const double *b;          /* RFF: d-n                                            */
    double scale;             /* RFF: feature = scale*cos(W x + b)                   */
    int32_t nbounds;          /* box constraints: lo < x[idx] < hi  (strict)         */
    const int32_t *bidx; const double *blo; const double *bhi;
    int32_t annulus;          /* 1: rmin <= hypot(x[ix]-cx, x[iy]-cy) <= rmax (closed)*/
    int32_t ix, iy; double cx, cy, rmin, rmax;
    double inflate;           /* inflated barrier                      */
    double noise_sigma;       /* std of the additive Gaussian white noise z_i of Alg. 2 l.5
                                 (PAPER.md:132, 150), on the physical rows; 0 = none (DESIGN G6, G17) */
    int32_t model_kind;       /* ORC_MODEL_*: how f(x, u) of PAPER.md:132 is evaluated (DESIGN G5, G18) */
} orc_config;

typedef struct {
    double  u[4];             /* selected input (fp32 candidate value, promoted)     */
    int32_t index;            /* winner index in [0, N] (N = the injected u_user)    */
    int32_t safe;             /* 1: winner safe over the horizon; 0: fallback branch */
    int32_t steps;            /* safe predicted states before first violation, [0,H] */
    int32_t n_safe;           /* |store| : number of safe candidates                 */
    double  dist;             /* ||u_winner - u_h||_2                                */
    int64_t n_exec;           /* executed sample-steps: sum_i min(steps_i+1, H)      */
} orc_result;

void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void   orc_sample(const orc_config *c, uint64_t tick, int64_t i, float *u /* m */);
void   orc_clamp_user(const orc_config *c, const float *u_user, float *u_h);
void   orc_lift(const orc_config *c, const double *x /* n */, double *z /* d */);
int    orc_is_safe(const orc_config *c, const double *x /* n */, double *margin);
void   orc_noise(const orc_config *c, uint64_t tick, int64_t i, int k, double *eps /* n standard normals */);
int    orc_rollout(const orc_config *c, const double *z0, const double *u, int H, uint64_t tick, int64_t i,
                   double *margin, double *traj /* H*d or NULL */);
int    orc_step(const orc_config *c, const float *x0, const float *u_user, uint64_t tick,
                orc_result *res, int32_t *steps /* N+1 or NULL */, double *margin /* N+1 or NULL */,
                double *dist /* N+1 or NULL */, float *U /* (N+1)*m or NULL */);
int    orc_rollout_batch(const orc_config *c, const float *U /* Ncand*m */, const float *X0 /* x0_count*n */,
                         int x0_count, int64_t Ncand, int H, uint64_t tick, int32_t *steps, double *margin,
                         double *traj /* Ncand*H*d or NULL */);
int    orc_num_threads(void);
#endif
