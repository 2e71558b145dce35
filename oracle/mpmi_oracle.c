/*
 * mpmi_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See mpmi_oracle.h.
 *
 * Every function follows Algorithm 2 of the paper step by step, in FP64,
 * in the paper's order: sample (l.1) -> for each i in parallel (l.2) -> while t_p < t+T and
 * safe (l.4): predict (l.5), isSafe (l.6), advance (l.7) -> store if safe (l.9-10) ->
 * argmin cost over store (l.13).  No blocking, fusion or reordering.
 * The only OpenMP pragma is the paper's own "for i in N in parallel".
 */
#include "mpmi_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- Philox4x32-10 (Salmon et al., SC'11): counter-based generator, DESIGN G4 --------- */
static void philox_round(uint32_t c[4], const uint32_t k[2]) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c[1] ^ k[0];
    const uint32_t n2 = hi0 ^ c[3] ^ k[1];
    c[0] = n0; c[1] = lo1; c[2] = n2; c[3] = lo0;
}
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c[4] = { ctr[0], ctr[1], ctr[2], ctr[3] };
    uint32_t k[2] = { key[0], key[1] };
    for (int r = 0; r < 10; r++) {
        if (r > 0) { k[0] += 0x9E3779B9u; k[1] += 0xBB67AE85u; }
        philox_round(c, k);
    }
    memcpy(out, c, sizeof c);
}

/* ---- Algorithm 2 line 1: xi ~ U^{MxN}, or the equally spaced discretisation
 *      the paper uses in practice.  Values are DEFINED in fp32 (DESIGN G3,G4)
 *      so that both implementations test bit-identical candidates. ------------------------- */
void orc_sample(const orc_config *c, uint64_t tick, int64_t i, float *u) {
    if (c->sampler == ORC_SAMPLER_PHILOX) {
        const uint32_t ctr[4] = { (uint32_t)i, (uint32_t)((uint64_t)i >> 32), (uint32_t)tick, (uint32_t)(tick >> 32) };
        const uint32_t key[2] = { (uint32_t)c->seed, (uint32_t)(c->seed >> 32) };
        uint32_t w[4];
        orc_philox4x32_10(ctr, key, w);
        for (int j = 0; j < c->m; j++) {
            const float r = (float)(w[j] >> 8) * 0x1p-24f;            /* exact in fp32 */
            u[j] = fmaf(r, c->u_hi[j] - c->u_lo[j], c->u_lo[j]);
        }
    } else {
        /* row-major, dimension 0 slowest; endpoint-inclusive: u = lo + (k/(cnt-1))*(hi-lo);
         * k/(cnt-1) is formed first so that mid-points of odd counts are exact ("straight") */
        int64_t rem = i;
        for (int j = c->m - 1; j >= 0; j--) {
            const int cnt = c->grid_counts[j];
            const int k = (int)(rem % cnt);
            rem /= cnt;
            const float lo = c->u_lo[j], hi = c->u_hi[j];
            if (cnt == 1)          u[j] = 0.5f * (lo + hi);
            else if (k == cnt - 1) u[j] = hi;
            else                   u[j] = fmaf((float)k / (float)(cnt - 1), hi - lo, lo);
        }
    }
}

/* the joystick interval is bounded: u_h = clamp(u_user) */
void orc_clamp_user(const orc_config *c, const float *u_user, float *u_h) {
    for (int j = 0; j < c->m; j++) {
        float v = u_user[j];
        if (v < c->u_lo[j]) v = c->u_lo[j];
        if (v > c->u_hi[j]) v = c->u_hi[j];
        u_h[j] = v;
    }
}

/* ---- lift z = Psi(x): "maps functions of state to functions of state" --- */
static double factor(uint8_t code, const double *x) {
    if (code == 0xFF) return 1.0;
    const int j = code & 0x3F;
    switch (code >> 6) {
        case 0:  return x[j];
        case 1:  return sin(x[j]);
        case 2:  return cos(x[j]);
        default: return NAN;
    }
}
void orc_lift(const orc_config *c, const double *x, double *z) {
    if (c->lift_kind == ORC_LIFT_MONO) {
        for (int f = 0; f < c->d; f++) {
            double p = 1.0;
            for (int q = 0; q < 4; q++) p *= factor(c->terms[4 * f + q], x);
            z[f] = p;
        }
    } else {
        for (int f = 0; f < c->n; f++) z[f] = x[f];
        for (int r = 0; r < c->d - c->n; r++) {
            double s = c->b[r];
            for (int j = 0; j < c->n; j++) s += c->W[r * c->n + j] * x[j];
            z[c->n + r] = c->scale * cos(s);
        }
    }
}

/* ---- isSafe(x_p): geometric test with the inflated barrier.
 *      Written so that NaN/Inf => unsafe.  margin = min over constraints of |g(x)|. ------- */
int orc_is_safe(const orc_config *c, const double *x, double *margin) {
    int safe = 1;
    double mg = INFINITY;
    for (int q = 0; q < c->nbounds; q++) {
        const double v = x[c->bidx[q]];
        const double lo = c->blo[q] + c->inflate, hi = c->bhi[q] - c->inflate;
        if (!(v > lo && v < hi)) safe = 0;
        if (fabs(v - lo) < mg) mg = fabs(v - lo);
        if (fabs(hi - v) < mg) mg = fabs(hi - v);
        if (v != v) mg = 0.0;
    }
    if (c->annulus) {
        const double dx = x[c->ix] - c->cx, dy = x[c->iy] - c->cy;
        const double r2 = dx * dx + dy * dy;
        const double rmin = c->rmin + c->inflate, rmax = c->rmax - c->inflate;
        if (!(r2 >= rmin * rmin && r2 <= rmax * rmax)) safe = 0;
        const double r = sqrt(r2);
        if (fabs(r - rmin) < mg) mg = fabs(r - rmin);
        if (fabs(rmax - r) < mg) mg = fabs(rmax - r);
        if (r2 != r2) mg = 0.0;
    }
    if (margin) *margin = mg;
    return safe;
}

/* ---- the additive noise z_i of Algorithm 2 l.5, "x_p <- f(x_p, xi(i)) + z_i" with z_i i.i.d.
 *      Gaussian white noise.  The paper fixes neither the generator nor the
 *      variance; DESIGN G17: eps ~ N(0, I_n) on the n physical dims, one independent draw per
 *      (tick, candidate i, step k, dim), from the counter-based Philox4x32-10 stream
 *      key = (seed_lo, seed_hi ^ 0x6E6F6973), counter = (i, (q << 16) | k, tick_lo, tick_hi), q = dim / 4,
 *      turned into normals by the Box-Muller transform: words (w0, w1) -> dims 4q, 4q+1 and
 *      (w2, w3) -> dims 4q+2, 4q+3, with u1 = ((w >> 8) + 1) 2^-24 in (0, 1], u2 = (w' >> 8) 2^-24. */
void orc_noise(const orc_config *c, uint64_t tick, int64_t i, int k, double *eps) {
    const double two_pi = 6.283185307179586476925286766559;
    const uint32_t key[2] = { (uint32_t)c->seed, (uint32_t)(c->seed >> 32) ^ 0x6E6F6973u };
    for (int q = 0; 4 * q < c->n; q++) {
        const uint32_t ctr[4] = { (uint32_t)i, ((uint32_t)q << 16) | (uint32_t)k, (uint32_t)tick, (uint32_t)(tick >> 32) };
        uint32_t w[4];
        orc_philox4x32_10(ctr, key, w);
        for (int h = 0; h < 2; h++) {
            const double u1 = ((double)(w[2 * h] >> 8) + 1.0) * 0x1p-24;
            const double u2 = (double)(w[2 * h + 1] >> 8) * 0x1p-24;
            const double r = sqrt(-2.0 * log(u1));
            const int j = 4 * q + 2 * h;
            if (j < c->n)     eps[j]     = r * cos(two_pi * u2);
            if (j + 1 < c->n) eps[j + 1] = r * sin(two_pi * u2);
        }
    }
}

/* ---- Algorithm 2 lines 3-8 for ONE candidate.
 *      x_t itself is not tested; exactly H predicted states x_1..x_H (DESIGN G8).
 *      f(x_p, xi): ORC_MODEL_LINEAR  z' = K z + B u, x = z[0:n], lifted once (DESIGN G5);
 *                  ORC_MODEL_RELIFT  x' = C (K Psi(x) + B u): the physical state is re-lifted
 *                  before every step, the literal f(x, u) on states of PAPER.md:132 (DESIGN G18).
 *      The same input is held over the horizon.  If noise_sigma > 0 the noise
 *      sigma * eps_k is added to the n physical rows of the predicted state BEFORE isSafe, as in
 *      l.5-6 of the algorithm, and stays in the state that is carried on.
 *      Returns steps = number of safe predicted states before the first violation (H <=> safe).
 *      margin = min |g| over every state tested, including the violating one.
 *      traj (optional): z_1..z_e written at traj[k*d + f], e = min(steps+1, H); the rest NaN. */
int orc_rollout(const orc_config *c, const double *z0, const double *u, int H, uint64_t tick, int64_t i,
                double *margin, double *traj) {
    const int d = c->d, m = c->m, n = c->n;
    double *z = (double *)malloc(sizeof(double) * d), *zn = (double *)malloc(sizeof(double) * d);
    double eps[64];
    memcpy(z, z0, sizeof(double) * d);
    double mg = INFINITY;
    int steps = H, safe = 1, k = 0;
    if (traj) for (long q = 0; q < (long)H * d; q++) traj[q] = NAN;
    while (k < H && safe) {                                   /* l.4: while t_p < t+T and safe */
        for (int r = 0; r < d; r++) {                         /* l.5: x_p <- f(x_p, xi(i))     */
            double s = 0.0;
            for (int q = 0; q < d; q++) s += c->K[r * d + q] * z[q];
            for (int j = 0; j < m; j++) s += c->B[r * m + j] * u[j];
            zn[r] = s;
        }
        if (c->noise_sigma > 0.0) {                           /* l.5: ... + z_i                */
            orc_noise(c, tick, i, k, eps);
            for (int j = 0; j < n; j++) zn[j] += c->noise_sigma * eps[j];
        }
        if (c->model_kind == ORC_MODEL_RELIFT) orc_lift(c, zn, z);   /* carry x = C zn, re-lifted */
        else memcpy(z, zn, sizeof(double) * d);
        if (traj) memcpy(traj + (long)k * d, z, sizeof(double) * d);
        double g;
        safe = orc_is_safe(c, z, &g);                         /* l.6: safe = isSafe(x_p)       */
        if (g < mg) mg = g;
        if (!safe) steps = k;                                 /* k safe states came before     */
        k++;                                                  /* l.7: t_p = t_p + dt           */
    }
    free(z); free(zn);
    if (margin) *margin = mg;
    return steps;
}

/* ---- Algorithm 2, whole tick -------------------------------------- */
int orc_step(const orc_config *c, const float *x0, const float *u_user, uint64_t tick,
             orc_result *res, int32_t *steps_out, double *margin_out, double *dist_out, float *U_out) {
    const int m = c->m, d = c->d, H = c->H;
    const int64_t NC = (int64_t)c->N + (c->include_user ? 1 : 0);
    for (int j = 0; j < c->n; j++) if (!isfinite(x0[j])) return -1;
    for (int j = 0; j < m; j++) if (!isfinite(u_user[j])) return -1;

    float u_h[4];
    orc_clamp_user(c, u_user, u_h);
    double xd[64], *z0 = (double *)malloc(sizeof(double) * d);
    for (int j = 0; j < c->n; j++) xd[j] = (double)x0[j];
    orc_lift(c, xd, z0);                                       /* x_p <- x_t (l.3), lifted once */

    int32_t *steps = (int32_t *)malloc(sizeof(int32_t) * NC);
    double *dist = (double *)malloc(sizeof(double) * NC);
    double *marg = (double *)malloc(sizeof(double) * NC);
    float *U = (float *)malloc(sizeof(float) * NC * m);

    #pragma omp parallel for schedule(static)                  /* l.2: for i in N in parallel */
    for (int64_t i = 0; i < NC; i++) {
        float uf[4]; double ud[4];
        if (i < c->N) orc_sample(c, tick, i, uf);              /* l.1: xi(i)                   */
        else          memcpy(uf, u_h, sizeof(float) * m);      /* the injected u_h, DESIGN G2  */
        double s2 = 0.0;
        for (int j = 0; j < m; j++) {
            U[i * m + j] = uf[j]; ud[j] = (double)uf[j];
            const double df = ud[j] - (double)u_h[j];
            s2 += df * df;
        }
        dist[i] = sqrt(s2);                                    /* cost = Euclidean distance */
        steps[i] = orc_rollout(c, z0, ud, H, tick, i, &marg[i], NULL);  /* l.3-8 */
    }

    /* l.9-13: store <- safe xi(i);  u_r <- argmin cost over store; ties -> lower index.
     * Empty store (paper silent, DESIGN G1): most steps before violation, then lower index. */
    int64_t best = -1, n_safe = 0, n_exec = 0;
    for (int64_t i = 0; i < NC; i++) {
        n_exec += (steps[i] + 1 < H) ? steps[i] + 1 : H;
        if (steps[i] == H) {
            n_safe++;
            if (best < 0 || steps[best] != H || dist[i] < dist[best]) best = i;
        } else if (best < 0 || (steps[best] != H && steps[i] > steps[best])) {
            best = i;
        }
    }
    memset(res, 0, sizeof *res);
    for (int j = 0; j < m; j++) res->u[j] = (double)U[best * m + j];
    res->index = (int32_t)best; res->safe = steps[best] == H; res->steps = steps[best];
    res->n_safe = (int32_t)n_safe; res->dist = dist[best]; res->n_exec = n_exec;
    if (steps_out)  memcpy(steps_out, steps, sizeof(int32_t) * NC);
    if (margin_out) memcpy(margin_out, marg, sizeof(double) * NC);
    if (dist_out)   memcpy(dist_out, dist, sizeof(double) * NC);
    if (U_out)      memcpy(U_out, U, sizeof(float) * NC * m);
    free(z0); free(steps); free(dist); free(marg); free(U);
    return 0;
}

/* ---- rollouts for caller-supplied inputs (trajectory cloud of Fig. 1) ---- */
int orc_rollout_batch(const orc_config *c, const float *U, const float *X0, int x0_count,
                      int64_t Ncand, int H, uint64_t tick, int32_t *steps, double *margin, double *traj) {
    const int d = c->d, m = c->m, n = c->n;
    if (x0_count != 1 && x0_count != Ncand) return -1;
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < Ncand; i++) {
        double xd[64], ud[4], *z0 = (double *)malloc(sizeof(double) * d);
        const float *x = X0 + (x0_count == 1 ? 0 : i * n);
        for (int j = 0; j < n; j++) xd[j] = (double)x[j];
        for (int j = 0; j < m; j++) ud[j] = (double)U[i * m + j];
        orc_lift(c, xd, z0);
        double mg;
        steps[i] = orc_rollout(c, z0, ud, H, tick, i, &mg, traj ? traj + i * (int64_t)H * d : NULL);
        if (margin) margin[i] = mg;
        free(z0);
    }
    return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
