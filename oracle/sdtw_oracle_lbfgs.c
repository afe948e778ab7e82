/*
 * sdtw_oracle_lbfgs.c -- float64 CPU ORACLE of the optimiser Table 1 names (L-BFGS; DESIGN.md
 * reading C23), on the barycenter objective of eq. 7.  Part of the oracle: THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT
 * (only tests/ may call it); it shares no code, header, table or constant with the CUDA path.  It lives in a file of
 * its own so that oracle/sdtw_oracle.c -- whose SHA-256 the full-size reference outputs under tests/golden/ are keyed
 * to -- changes only when the definitions those references were computed with change.
 *
 * The pair evaluations (forward R, reverse E, contraction) are the ones of sdtw_oracle.c; this file adds the two-loop
 * recursion and the descent around them.  Pins (tests/test_oracle_pins.py): the recursion against the dense BFGS update
 * formula built in numpy (1e-12) and the secant equation; hist = 0 against oracle_barycenter_backtracking_f32 bit for
 * bit; the Armijo conditions replayed with independent evaluations; monotone objective.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG -1
#define ORACLE_ERR_MEM -2

/* sdtw_oracle.c */
int oracle_pair_full_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma, int64_t band,
                            double *value, double *grad, double *E_out, double *R_out);
int oracle_pair_checkpointed_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                                    int64_t band, double *value, double *grad);

/* ---- L-BFGS on the barycenter objective of eq. 7: the optimiser Table 1 names ("L-BFGS"; the paper
 * takes it off the shelf, so the recursion below is the textbook one -- Nocedal & Wright, Numerical Optimization,
 * Algorithm 7.4 -- and the line search is the Armijo backtracking of oracle_barycenter_backtracking_f32; C23).
 *
 * oracle_lbfgs_direction: r = H g by the two-loop recursion over the `count` stored pairs (s_i, y_i), i = 0 oldest ..
 * count-1 newest, rho_i = 1 / (s_i . y_i), initial matrix H0 = (s.y / y.y of the newest pair) I:
 *     q = g;  for i = newest..oldest: alpha_i = rho_i (s_i . q), q -= alpha_i y_i
 *     r = (s.y / y.y) q;  for i = oldest..newest: beta = rho_i (y_i . r), r += (alpha_i - beta) s_i
 * count == 0: r = g. ---- */
int oracle_lbfgs_direction(const double *S, const double *Y, int count, int64_t md, const double *g, double *r) {
    if (!g || !r || md < 1 || count < 0 || (count > 0 && (!S || !Y))) return ORACLE_ERR_ARG;
    double *alpha = (double *)malloc((size_t)(count > 0 ? count : 1) * sizeof(double));
    double *rho = (double *)malloc((size_t)(count > 0 ? count : 1) * sizeof(double));
    if (!alpha || !rho) { free(alpha); free(rho); return ORACLE_ERR_MEM; }
    for (int64_t t = 0; t < md; ++t) r[t] = g[t];
    for (int i = 0; i < count; ++i) {
        double sy = 0.0;
        for (int64_t t = 0; t < md; ++t) sy += S[(size_t)i * md + t] * Y[(size_t)i * md + t];
        rho[i] = 1.0 / sy;
    }
    for (int i = count - 1; i >= 0; --i) {
        double sq = 0.0;
        for (int64_t t = 0; t < md; ++t) sq += S[(size_t)i * md + t] * r[t];
        alpha[i] = rho[i] * sq;
        for (int64_t t = 0; t < md; ++t) r[t] -= alpha[i] * Y[(size_t)i * md + t];
    }
    if (count > 0) {
        const double *sn = S + (size_t)(count - 1) * md, *yn = Y + (size_t)(count - 1) * md;
        double sy = 0.0, yy = 0.0;
        for (int64_t t = 0; t < md; ++t) { sy += sn[t] * yn[t]; yy += yn[t] * yn[t]; }
        const double scale = sy / yy;
        for (int64_t t = 0; t < md; ++t) r[t] *= scale;
    }
    for (int i = 0; i < count; ++i) {
        double yr = 0.0;
        for (int64_t t = 0; t < md; ++t) yr += Y[(size_t)i * md + t] * r[t];
        const double beta = rho[i] * yr;
        for (int64_t t = 0; t < md; ++t) r[t] += (alpha[i] - beta) * S[(size_t)i * md + t];
    }
    free(alpha); free(rho);
    return ORACLE_OK;
}

/* The descent.  Z(0) = Z0 promoted to double; f, G as in oracle_barycenter_backtracking_f32.  Iteration it:
 *     d = -H G (two-loop recursion over the stored pairs); if G.d >= 0 the pairs are dropped and d = -G;
 *     t = step0 when no pair is stored, else 1;  up to max_trials times:  Zt = Z + t d;
 *         accept if f(Zt) <= f(Z) + c1 t (G.d), else t = shrink t;
 *     accepted: s = Zt - Z, y = G(Zt) - G(Z); the pair is stored (the oldest dropped beyond `hist`) iff
 *         s.y > 1e-10 |s| |y| (keeps H positive definite); Z = Zt, steps[it] = t.
 *     none accepted: steps[it] = 0, the descent stops (as in the backtracking loop).
 * hist == 0 is oracle_barycenter_backtracking_f32, operation for operation. ---- */
int oracle_barycenter_lbfgs_f32(const float *Z0, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                                double gamma, const double *weights, int64_t band, int iters, int hist, double step0,
                                double shrink, double c1, int max_trials, double *Z_out, double *values,
                                double *objective, double *steps, int32_t *trials, int mode, int nthreads) {
    if (!Z0 || !X || !offsets || !Z_out || !objective || !steps || !trials || m < 1 || d < 1 || N < 1 ||
        !(gamma > 0.0) || iters < 0 || hist < 0 || !(step0 > 0.0) || !(shrink > 0.0 && shrink < 1.0) || !(c1 >= 0.0) ||
        max_trials < 1)
        return ORACLE_ERR_ARG;
    const int64_t md = m * d;
    const int H = hist > 0 ? hist : 1;
    double *G = (double *)malloc((size_t)md * sizeof(double));
    double *Gold = (double *)malloc((size_t)md * sizeof(double));
    double *D = (double *)malloc((size_t)md * sizeof(double));
    double *Zt = (double *)malloc((size_t)md * sizeof(double));
    double *S = (double *)malloc((size_t)H * (size_t)md * sizeof(double));
    double *Y = (double *)malloc((size_t)H * (size_t)md * sizeof(double));
    double *vals = (double *)malloc((size_t)N * sizeof(double));
    if (!G || !Gold || !D || !Zt || !S || !Y || !vals) { free(G); free(Gold); free(D); free(Zt); free(S); free(Y); free(vals); return ORACLE_ERR_MEM; }
    for (int64_t t = 0; t < md; ++t) Z_out[t] = (double)Z0[t];
    for (int it = 0; it < iters; ++it) { steps[it] = 0.0; trials[it] = 0; }
    int rc = ORACLE_OK;
    double f = 0.0;
#define EVAL(Zptr, want_g, fout)                                                                                       \
    do {                                                                                                               \
        double *gk_ = (double *)calloc((size_t)N * (size_t)md, sizeof(double));                                        \
        if (!gk_) { rc = ORACLE_ERR_MEM; break; }                                                                      \
        _Pragma("omp parallel for schedule(dynamic, 1)") for (int k = 0; k < N; ++k) {                                 \
            const int64_t n_ = offsets[k + 1] - offsets[k];                                                            \
            double *x_ = (double *)malloc((size_t)(n_ * d) * sizeof(double));                                          \
            for (int64_t t_ = 0; t_ < n_ * d; ++t_) x_[t_] = (double)X[offsets[k] * d + t_];                           \
            double *g_ = (want_g) ? gk_ + (size_t)k * (size_t)md : NULL;                                               \
            if (mode == 1) oracle_pair_checkpointed_banded(x_, n_, (Zptr), m, d, gamma, band, &vals[k], g_);           \
            else oracle_pair_full_banded(x_, n_, (Zptr), m, d, gamma, band, &vals[k], g_, NULL, NULL);                 \
            free(x_);                                                                                                  \
        }                                                                                                              \
        double o_ = 0.0;                                                                                               \
        for (int k = 0; k < N; ++k) o_ += (weights ? weights[k] : 1.0) * vals[k];                                      \
        (fout) = o_;                                                                                                   \
        if (want_g)                                                                                                    \
            for (int64_t t_ = 0; t_ < md; ++t_) {                                                                      \
                double a_ = 0.0;                                                                                       \
                for (int k = 0; k < N; ++k) a_ += (weights ? weights[k] : 1.0) * gk_[(size_t)k * (size_t)md + t_];     \
                G[t_] = a_;                                                                                            \
            }                                                                                                          \
        free(gk_);                                                                                                     \
    } while (0)
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    EVAL(Z_out, 1, f);
    objective[0] = f;
    if (values) memcpy(values, vals, (size_t)N * sizeof(double));
    int stopped = 0, count = 0;
    for (int it = 0; it < iters && rc == ORACLE_OK; ++it) {
        if (stopped) { objective[it + 1] = f; continue; }
        rc = oracle_lbfgs_direction(S, Y, count, md, G, D);
        if (rc != ORACLE_OK) break;
        double gd = 0.0;
        for (int64_t t = 0; t < md; ++t) { D[t] = -D[t]; gd += G[t] * D[t]; }
        if (!(gd < 0.0)) {                       /* not a descent direction: restart from steepest descent */
            count = 0;
            gd = 0.0;
            for (int64_t t = 0; t < md; ++t) { D[t] = -G[t]; gd += G[t] * D[t]; }
        }
        double step = (count == 0) ? step0 : 1.0;
        int accepted = 0;
        for (int tr = 0; tr < max_trials && rc == ORACLE_OK; ++tr) {
            for (int64_t t = 0; t < md; ++t) Zt[t] = Z_out[t] + step * D[t];
            double ft = 0.0;
            EVAL(Zt, 0, ft);
            trials[it] = tr + 1;
            if (ft <= f + c1 * step * gd) {
                memcpy(Gold, G, (size_t)md * sizeof(double));
                EVAL(Zt, 1, f);                          /* gradient (and the same f) at the accepted point */
                if (values) memcpy(values, vals, (size_t)N * sizeof(double));
                if (hist > 0) {
                    double *sn, *yn;
                    if (count == hist) {                 /* drop the oldest pair */
                        memmove(S, S + md, (size_t)(hist - 1) * (size_t)md * sizeof(double));
                        memmove(Y, Y + md, (size_t)(hist - 1) * (size_t)md * sizeof(double));
                        count = hist - 1;
                    }
                    sn = S + (size_t)count * md; yn = Y + (size_t)count * md;
                    double sy = 0.0, ss = 0.0, yy = 0.0;
                    for (int64_t t = 0; t < md; ++t) {
                        sn[t] = Zt[t] - Z_out[t]; yn[t] = G[t] - Gold[t];
                        sy += sn[t] * yn[t]; ss += sn[t] * sn[t]; yy += yn[t] * yn[t];
                    }
                    if (sy > 1e-10 * sqrt(ss) * sqrt(yy)) ++count;
                }
                memcpy(Z_out, Zt, (size_t)md * sizeof(double));
                steps[it] = step;
                accepted = 1;
                break;
            }
            step *= shrink;
        }
        if (!accepted) stopped = 1;
        objective[it + 1] = f;
    }
#undef EVAL
    free(G); free(Gold); free(D); free(Zt); free(S); free(Y); free(vals);
    return rc;
}
