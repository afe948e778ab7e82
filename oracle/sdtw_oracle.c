/*
 * sdtw_oracle.c -- float64 CPU ORACLE for the Soft-DTW value / gradient / barycenter path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant with the CUDA path under paper_2404_12134_b200/csrc/.
 *
 * What it is: the plain definitions of arXiv 2404.12134, written
 * out in the paper's order and notation, in IEEE double, with no blocking / fusion /
 * reordering beyond what the definitions state:
 *
 *   Def. 3  distance matrix  Delta[i][j] = delta(x_i, z_j); delta is read
 *                               as the SQUARED Euclidean distance sum_c (x_ic - z_jc)^2
 *                               (reading C3: eq. 6 / north_star's 2(z_j - x_i)
 *                               gradient is the derivative of the squared form).
 *   eq. 3  min^gamma(a_1..a_n) = -gamma log sum_i exp(-a_i / gamma)
 *                               (the extracted text prints "e^{-a_i gamma}"; reading C1),
 *                               = min_i a_i for gamma = 0.
 *   Def. 6 / eq. 5  r_00 = 0, r_i0 = r_0j = inf,
 *                               r_ij = delta_ij + min^gamma(r_{i-1,j-1}, r_{i-1,j}, r_{i,j-1}),
 *                               Soft-DTW^gamma = r_{M,N}.
 *   eq. 6  grad = (d Delta / d Z)^T E, E by the reverse dynamic programme
 *                               "described in [19]" (not printed in the paper; reading C5, the
 *                               recurrence is fixed independently by E = d value / d Delta and
 *                               by the paper's buffer initial values 0 / 0 / 1).
 *   Def. 7 / eq. 7  barycenter objective, read (C6, C8) as the plain sum
 *                               over k minimised by fixed-step gradient descent.
 *   Def. 4 / eq. 1  classic DTW (the gamma = 0 case), used as a pin.
 *   Table 1  Sakoe-Chiba band: read (C18) as the classic adjustment
 *                               window |i - j| <= band on the cell indices; cells outside it belong
 *                               to no admissible path (Delta = +inf there, so r = +inf, E = 0).
 *                               band < 0 means no band.  The *_ex entry points take it.
 *   Def. 8 / eq. 8  similarity score d_score = DTW / |pi| (Step 3 scoring): oracle_dtw_path
 *                               (float64, the definition) and oracle_dtw_score_f32 (decisions in float32).
 *   eq. 7  per-series weights lambda_i / m_i: the *_ex entry points take one
 *                               weight w_k per pair; objective = sum_k w_k value_k and
 *                               grad = sum_k w_k grad_k (values[k] stay unweighted).
 *
 * Index convention: x has n rows (time steps) of d channels, z has m rows of d channels,
 * both row-major [t][c].  R is stored with the paper's 0-row/0-column border (and one more
 * border row/column at n+1 / m+1 for the reverse pass), i.e. (n+2) x (m+2), 1-based cells.
 *
 * parity pins: see tests/test_oracle_pins.py (brute force over all alignment paths, closed
 * forms, Delannoy counts, gamma->0 bounds, invariants of E, finite differences, symmetries).
 * Not pinned: agreement with TSLearn / the authors' code ("parity unpinned" for that item
 * only -- neither exists in this environment).
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

/* ---- eq. 3: soft minimum of three (gamma > 0), evaluated in the numerically safe
 * log-sum-exp form  mn - gamma log sum exp(-(a_p - mn)/gamma),  exp(-inf) = 0. ---- */
static double softmin3(double a, double b, double c, double gamma) {
    double mn = a;
    if (b < mn) mn = b;
    if (c < mn) mn = c;
    if (isinf(mn)) return mn; /* all three +inf */
    double s = exp(-(a - mn) / gamma) + exp(-(b - mn) / gamma) + exp(-(c - mn) / gamma);
    return mn - gamma * log(s);
}

static double min3(double a, double b, double c) {
    double mn = a;
    if (b < mn) mn = b;
    if (c < mn) mn = c;
    return mn;
}

/* ---- Sakoe-Chiba band (Table 1; reading C18): cell (i, j) is admissible iff
 * |i - j| <= band; band < 0 = no band.  Same for 0- or 1-based (i, j). ---- */
static int admissible(int64_t i, int64_t j, int64_t band) {
    if (band < 0) return 1;
    int64_t t = i - j;
    if (t < 0) t = -t;
    return t <= band;
}

/* ---- Def. 3: delta(x_i, z_j) = sum_c (x_ic - z_jc)^2 ---- */
static double delta_sq(const double *xi, const double *zj, int d) {
    double s = 0.0;
    for (int c = 0; c < d; ++c) {
        double t = xi[c] - zj[c];
        s += t * t;
    }
    return s;
}

/* Delta(X, Z) as an n x m row-major matrix (0-based). */
int oracle_cost_matrix(const double *x, int64_t n, const double *z, int64_t m, int d, double *D) {
    if (!x || !z || !D || n < 1 || m < 1 || d < 1) return ORACLE_ERR_ARG;
    for (int64_t i = 0; i < n; ++i)
        for (int64_t j = 0; j < m; ++j) D[i * m + j] = delta_sq(x + i * d, z + j * d, d);
    return ORACLE_OK;
}

/* ---- Def. 6 / eq. 5 on a given cost matrix.  R is (n+2) x (m+2); on return rows 0..n and
 * columns 0..m hold r_ij (border: r_00 = 0, r_i0 = r_0j = +inf).  gamma == 0 gives eq. 1. ---- */
int oracle_forward_R_banded(const double *D, int64_t n, int64_t m, double gamma, int64_t band, double *R);
int oracle_forward_R(const double *D, int64_t n, int64_t m, double gamma, double *R) {
    return oracle_forward_R_banded(D, n, m, gamma, -1, R);
}
/* the same with a Sakoe-Chiba band: inadmissible cells get r = +inf */
int oracle_forward_R_banded(const double *D, int64_t n, int64_t m, double gamma, int64_t band, double *R) {
    if (!D || !R || n < 1 || m < 1 || !(gamma >= 0.0)) return ORACLE_ERR_ARG;
    const int64_t ld = m + 2;
    for (int64_t j = 0; j <= m + 1; ++j) R[j] = INFINITY;
    for (int64_t i = 0; i <= n + 1; ++i) R[i * ld] = INFINITY;
    R[0] = 0.0;
    for (int64_t i = 1; i <= n; ++i)
        for (int64_t j = 1; j <= m; ++j) {
            if (!admissible(i, j, band)) { R[i * ld + j] = INFINITY; continue; }
            double rd = R[(i - 1) * ld + (j - 1)], ru = R[(i - 1) * ld + j], rl = R[i * ld + (j - 1)];
            double sm = (gamma > 0.0) ? softmin3(rd, ru, rl, gamma) : min3(rd, ru, rl);
            R[i * ld + j] = D[(i - 1) * m + (j - 1)] + sm;
        }
    return ORACLE_OK;
}

/* ---- reverse dynamic programme for E (reading C5; Algorithm 2 of the paper's ref. [19]):
 * pad  D[i][m+1] = D[n+1][j] = 0,  R[i][m+1] = R[n+1][j] = -inf,  R[n+1][m+1] = R[n][m],
 * E[n+1][m+1] = 1, other pads 0 (the paper's "0 for hbuf and vbuf, and 1 for dbuf",
 * PAPER.md:225); for j = m..1, i = n..1:
 *   E[i][j] = E[i+1][j]   exp((R[i+1][j]   - R[i][j] - D[i+1][j])   / gamma)
 *           + E[i][j+1]   exp((R[i][j+1]   - R[i][j] - D[i][j+1])   / gamma)
 *           + E[i+1][j+1] exp((R[i+1][j+1] - R[i][j] - D[i+1][j+1]) / gamma).
 * R must be the (n+2) x (m+2) array filled by oracle_forward_R (it is padded in place).
 * E is n x m row-major (0-based). ---- */
int oracle_backward_E_banded(const double *D, int64_t n, int64_t m, double gamma, int64_t band, double *R, double *E);
int oracle_backward_E(const double *D, int64_t n, int64_t m, double gamma, double *R, double *E) {
    return oracle_backward_E_banded(D, n, m, gamma, -1, R, E);
}
/* the same with a Sakoe-Chiba band: an inadmissible cell has E = 0 and contributes nothing to its
 * predecessors (it lies on no admissible path); requires |n - m| <= band (else no path exists). */
int oracle_backward_E_banded(const double *D, int64_t n, int64_t m, double gamma, int64_t band, double *R, double *E) {
    if (!D || !R || !E || n < 1 || m < 1 || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    if (!admissible(n, m, band)) return ORACLE_ERR_ARG;
    const int64_t ld = m + 2;
    double *Ep = (double *)calloc((size_t)((n + 2) * ld), sizeof(double));
    if (!Ep) return ORACLE_ERR_MEM;
    for (int64_t i = 1; i <= n; ++i) R[i * ld + (m + 1)] = -INFINITY;
    for (int64_t j = 1; j <= m; ++j) R[(n + 1) * ld + j] = -INFINITY;
    R[(n + 1) * ld + (m + 1)] = R[n * ld + m];
    Ep[(n + 1) * ld + (m + 1)] = 1.0;
#define DPAD(i, j) (((i) <= n && (j) <= m) ? D[((i)-1) * m + ((j)-1)] : 0.0)
#define OK_S(i, j) (((i) > n || (j) > m) ? 1 : admissible((i), (j), band)) /* pad cells are not masked */
    for (int64_t j = m; j >= 1; --j)
        for (int64_t i = n; i >= 1; --i) {
            if (!admissible(i, j, band)) continue; /* E = 0 */
            double r = R[i * ld + j];
            double a = OK_S(i + 1, j) ? exp((R[(i + 1) * ld + j] - r - DPAD(i + 1, j)) / gamma) : 0.0;
            double b = OK_S(i, j + 1) ? exp((R[i * ld + (j + 1)] - r - DPAD(i, j + 1)) / gamma) : 0.0;
            double c = OK_S(i + 1, j + 1) ? exp((R[(i + 1) * ld + (j + 1)] - r - DPAD(i + 1, j + 1)) / gamma) : 0.0;
            Ep[i * ld + j] = Ep[(i + 1) * ld + j] * a + Ep[i * ld + (j + 1)] * b + Ep[(i + 1) * ld + (j + 1)] * c;
        }
#undef OK_S
#undef DPAD
    for (int64_t i = 1; i <= n; ++i)
        for (int64_t j = 1; j <= m; ++j) E[(i - 1) * m + (j - 1)] = Ep[i * ld + j];
    free(Ep);
    return ORACLE_OK;
}

/* ---- the same E written as a probability flow ("normalised" form): for each cell s, the
 * weights of its three predecessors p are w_p = exp((mn_s - R[p]) / gamma) / sum_p(...), and
 * E[p] += E[s] w_p.  Mathematically identical to oracle_backward_E; kept as a standing
 * self-check (the two must agree to < 1e-8 on every configuration). ---- */
int oracle_backward_E_normalised(const double *D, int64_t n, int64_t m, double gamma, const double *R, double *E) {
    (void)D;
    if (!R || !E || n < 1 || m < 1 || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    const int64_t ld = m + 2;
    double *Ep = (double *)calloc((size_t)((n + 2) * ld), sizeof(double));
    if (!Ep) return ORACLE_ERR_MEM;
    Ep[n * ld + m] = 1.0;
    for (int64_t i = n; i >= 1; --i)
        for (int64_t j = m; j >= 1; --j) {
            double e = Ep[i * ld + j];
            double rd = R[(i - 1) * ld + (j - 1)], ru = R[(i - 1) * ld + j], rl = R[i * ld + (j - 1)];
            double mn = min3(rd, ru, rl);
            if (isinf(mn)) continue;
            double wd = exp((mn - rd) / gamma), wu = exp((mn - ru) / gamma), wl = exp((mn - rl) / gamma);
            double s = wd + wu + wl;
            Ep[(i - 1) * ld + (j - 1)] += e * wd / s;
            Ep[(i - 1) * ld + j] += e * wu / s;
            Ep[i * ld + (j - 1)] += e * wl / s;
        }
    for (int64_t i = 1; i <= n; ++i)
        for (int64_t j = 1; j <= m; ++j) E[(i - 1) * m + (j - 1)] = Ep[i * ld + j];
    free(Ep);
    return ORACLE_OK;
}

/* ---- eq. 6 with squared-Euclidean delta:  g[j][c] = sum_i E[i][j] 2 (z[j][c] - x[i][c]).
 * grad (m x d) is INCREMENTED (the paper's "gradient vector is incremented");
 * rows are visited i = n..1, the order of the reverse pass. ---- */
static void contract_gradient(const double *E, const double *x, int64_t n, const double *z, int64_t m, int d,
                              double *grad) {
    for (int64_t i = n - 1; i >= 0; --i)
        for (int64_t j = 0; j < m; ++j) {
            double e = E[i * m + j];
            for (int c = 0; c < d; ++c) grad[j * d + c] += e * 2.0 * (z[j * d + c] - x[i * d + c]);
        }
}

/* ---- one pair, full-matrix mode: value = r_{n,m}; grad (may be NULL) incremented by eq. 6;
 * E_out / R_out (may be NULL) receive the n x m E and the (n+2) x (m+2) R. ---- */
int oracle_pair_full_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                            int64_t band, double *value, double *grad, double *E_out, double *R_out);
int oracle_pair_full(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma, double *value,
                     double *grad, double *E_out, double *R_out) {
    return oracle_pair_full_banded(x, n, z, m, d, gamma, -1, value, grad, E_out, R_out);
}
int oracle_pair_full_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                            int64_t band, double *value, double *grad, double *E_out, double *R_out) {
    if (!x || !z || !value || n < 1 || m < 1 || d < 1 || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    if (!admissible(n, m, band)) return ORACLE_ERR_ARG; /* no complete path inside the band */
    double *D = (double *)malloc((size_t)(n * m) * sizeof(double));
    double *R = (double *)malloc((size_t)((n + 2) * (m + 2)) * sizeof(double));
    if (!D || !R) {
        free(D);
        free(R);
        return ORACLE_ERR_MEM;
    }
    oracle_cost_matrix(x, n, z, m, d, D);
    oracle_forward_R_banded(D, n, m, gamma, band, R);
    *value = R[n * (m + 2) + m];
    int rc = ORACLE_OK;
    if (grad || E_out) {
        double *E = E_out ? E_out : (double *)malloc((size_t)(n * m) * sizeof(double));
        if (!E) rc = ORACLE_ERR_MEM;
        if (rc == ORACLE_OK) {
            if (R_out) { /* keep the unpadded forward R for the caller */
                memcpy(R_out, R, (size_t)((n + 2) * (m + 2)) * sizeof(double));
            }
            rc = oracle_backward_E_banded(D, n, m, gamma, band, R, E);
            if (rc == ORACLE_OK && grad) contract_gradient(E, x, n, z, m, d, grad);
        }
        if (!E_out) free(E);
    } else if (R_out) {
        memcpy(R_out, R, (size_t)((n + 2) * (m + 2)) * sizeof(double));
    }
    free(D);
    free(R);
    return rc;
}

/* ---- one pair, ROW-CHECKPOINTED mode (for the 10k / 30k configurations where the full
 * float64 R is 0.8 / 7.2 GB): keep every K-th row of R (K ~ sqrt(n)), recompute K-row blocks
 * of R going backwards, hold only two rows of E.  Every cell is computed by exactly the
 * same expressions, in the same order, as in oracle_pair_full, so value and grad are
 * BITWISE identical to the full mode (tests/test_oracle_pins.py checks this). ---- */
static void forward_row(const double *xi, int64_t i /* 1-based row */, const double *z, int64_t m, int d, double gamma,
                        int64_t band, const double *Rprev, double *Rcur /* both (m+2) wide, 1-based */) {
    Rcur[0] = INFINITY;
    for (int64_t j = 1; j <= m; ++j) {
        if (!admissible(i, j, band)) { Rcur[j] = INFINITY; continue; }
        double dij = delta_sq(xi, z + (j - 1) * d, d);
        Rcur[j] = dij + softmin3(Rprev[j - 1], Rprev[j], Rcur[j - 1], gamma);
    }
}

int oracle_pair_checkpointed_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                                    int64_t band, double *value, double *grad);
int oracle_pair_checkpointed(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                             double *value, double *grad) {
    return oracle_pair_checkpointed_banded(x, n, z, m, d, gamma, -1, value, grad);
}
int oracle_pair_checkpointed_banded(const double *x, int64_t n, const double *z, int64_t m, int d, double gamma,
                                    int64_t band, double *value, double *grad) {
    if (!x || !z || !value || n < 1 || m < 1 || d < 1 || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    if (!admissible(n, m, band)) return ORACLE_ERR_ARG;
    const int64_t ld = m + 2;
    int64_t K = (int64_t)ceil(sqrt((double)n));
    if (K < 1) K = 1;
    const int64_t nck = n / K + 1; /* checkpoints hold rows 0, K, 2K, ... */
    double *ck = (double *)malloc((size_t)(nck * ld) * sizeof(double));
    double *blk = (double *)malloc((size_t)((K + 2) * ld) * sizeof(double)); /* rows b0 .. b0+K+1 */
    double *Ea = (double *)calloc((size_t)ld, sizeof(double));               /* E row i+1 */
    double *Eb = (double *)calloc((size_t)ld, sizeof(double));               /* E row i   */
    double *row = (double *)malloc((size_t)(2 * ld) * sizeof(double));
    if (!ck || !blk || !Ea || !Eb || !row) {
        free(ck); free(blk); free(Ea); free(Eb); free(row);
        return ORACLE_ERR_MEM;
    }
    /* forward sweep, keeping checkpoint rows */
    double *prev = row, *cur = row + ld;
    for (int64_t j = 0; j <= m + 1; ++j) prev[j] = INFINITY;
    prev[0] = 0.0;
    memcpy(ck, prev, (size_t)ld * sizeof(double));
    for (int64_t i = 1; i <= n; ++i) {
        forward_row(x + (i - 1) * d, i, z, m, d, gamma, band, prev, cur);
        cur[m + 1] = INFINITY;
        if (i % K == 0) memcpy(ck + (i / K) * ld, cur, (size_t)ld * sizeof(double));
        double *t = prev; prev = cur; cur = t;
    }
    *value = prev[m];
    const double Rnm = prev[m];
    if (grad) {
        /* reverse sweep over blocks of rows (b0, b0+K], b0 = last multiple of K below n, ... 0 */
        int first = 1;
        for (int64_t b0 = ((n - 1) / K) * K; b0 >= 0; b0 -= K) {
            int64_t b1 = b0 + K; /* rows b0+1 .. min(b1, n) recomputed */
            if (b1 > n) b1 = n;
            memcpy(blk, ck + (b0 / K) * ld, (size_t)ld * sizeof(double));
            for (int64_t i = b0 + 1; i <= b1; ++i)
                forward_row(x + (i - 1) * d, i, z, m, d, gamma, band, blk + (i - 1 - b0) * ld, blk + (i - b0) * ld);
            /* row b1+1 of R: the pad row (-inf, corner R[n][m]) if b1 == n, else the first row of
             * the block processed just before (kept in blk's last slot by the copy below). */
            double *Rnext = blk + (b1 - b0 + 1) * ld;
            if (first) {
                for (int64_t j = 0; j <= m + 1; ++j) Rnext[j] = -INFINITY;
                Rnext[m + 1] = Rnm;
                memset(Ea, 0, (size_t)ld * sizeof(double));
                Ea[m + 1] = 1.0;
                first = 0;
            } else {
                memcpy(Rnext, row, (size_t)ld * sizeof(double)); /* saved below */
            }
            for (int64_t i = b1; i >= b0 + 1; --i) {
                double *Ri = blk + (i - b0) * ld, *Ri1 = blk + (i + 1 - b0) * ld;
                const int last_row = (i == n);
                Ri[m + 1] = -INFINITY; /* pad column of the reverse pass */
                Eb[m + 1] = 0.0;
                for (int64_t j = m; j >= 1; --j) {
                    if (!admissible(i, j, band)) { Eb[j] = 0.0; continue; }
                    double r = Ri[j];
                    double d_dn = last_row ? 0.0 : delta_sq(x + i * d, z + (j - 1) * d, d);              /* D[i+1][j]   */
                    double d_rt = (j == m) ? 0.0 : delta_sq(x + (i - 1) * d, z + j * d, d);              /* D[i][j+1]   */
                    double d_dg = (last_row || j == m) ? 0.0 : delta_sq(x + i * d, z + j * d, d);        /* D[i+1][j+1] */
                    /* successors inside the matrix but outside the band contribute nothing */
                    const int ok_dn = last_row || admissible(i + 1, j, band);
                    const int ok_rt = (j == m) || admissible(i, j + 1, band);
                    double a = ok_dn ? exp((Ri1[j] - r - d_dn) / gamma) : 0.0;
                    double b = ok_rt ? exp((Ri[j + 1] - r - d_rt) / gamma) : 0.0;
                    double c = exp((Ri1[j + 1] - r - d_dg) / gamma); /* (i+1, j+1) has the same i - j */
                    Eb[j] = Ea[j] * a + Eb[j + 1] * b + Ea[j + 1] * c;
                }
                for (int64_t j = 0; j < m; ++j) {
                    double e = Eb[j + 1];
                    for (int c = 0; c < d; ++c) grad[j * d + c] += e * 2.0 * (z[j * d + c] - x[(i - 1) * d + c]);
                }
                double *t = Ea; Ea = Eb; Eb = t;
            }
            /* save R row b0+1 (first recomputed row) as "row b1+1" of the next (upper) block */
            memcpy(row, blk + ld, (size_t)ld * sizeof(double));
            row[m + 1] = -INFINITY;
        }
    }
    free(ck); free(blk); free(Ea); free(Eb); free(row);
    return ORACLE_OK;
}

/* ---- the call the C-ABI boundary mirrors (include/sdtw.h: sdtw_value_grad): fp32 inputs
 * promoted to double; values[k] = Soft-DTW(x_k, Z); grad = sum_k grad_k in k order (NULL =>
 * values only).  mode 0 = full matrices, 1 = row-checkpointed.  OpenMP over pairs only;
 * per-pair gradients are added into grad in ascending k whatever the thread count. ---- */
int oracle_value_grad_ex_f32(const float *Z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                             double gamma, const double *weights, int64_t band, double *values, double *grad,
                             double *objective, int mode, int nthreads);
int oracle_value_grad_f32(const float *Z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                          double gamma, double *values, double *grad, int mode, int nthreads) {
    return oracle_value_grad_ex_f32(Z, m, d, X, offsets, N, gamma, NULL, -1, values, grad, NULL, mode, nthreads);
}
/* the same with eq. 7's per-pair weights w_k (NULL = all 1) and Table 1's Sakoe-Chiba band (< 0 = none):
 * values[k] unweighted, grad = sum_k w_k grad_k (k ascending), *objective = sum_k w_k values[k]. */
int oracle_value_grad_ex_f64z(const double *z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                              double gamma, const double *weights, int64_t band, double *values, double *grad,
                              double *objective, int mode, int nthreads);
int oracle_value_grad_ex_f32(const float *Z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                             double gamma, const double *weights, int64_t band, double *values, double *grad,
                             double *objective, int mode, int nthreads) {
    if (!Z || m < 1 || d < 1) return ORACLE_ERR_ARG;
    double *z = (double *)malloc((size_t)(m * d) * sizeof(double));
    if (!z) return ORACLE_ERR_MEM;
    for (int64_t t = 0; t < m * d; ++t) z[t] = (double)Z[t];
    const int rc = oracle_value_grad_ex_f64z(z, m, d, X, offsets, N, gamma, weights, band, values, grad, objective, mode,
                                             nthreads);
    free(z);
    return rc;
}
/* the same evaluation at a barycenter given in double (an iterate of the descent below, which keeps Z in double
 * between iterations -- reading C14): lets a caller drive the loop Z <- Z - step G one evaluation at a time (the
 * full-size reference outputs of tests/golden/ are written that way, resumably). */
int oracle_value_grad_ex_f64z(const double *z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                              double gamma, const double *weights, int64_t band, double *values, double *grad,
                              double *objective, int mode, int nthreads) {
    if (!z || !X || !offsets || !values || m < 1 || d < 1 || N < 1 || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return ORACLE_ERR_ARG;
    double *gk = grad ? (double *)calloc((size_t)N * (size_t)(m * d), sizeof(double)) : NULL;
    if (grad && !gk) { free(gk); return ORACLE_ERR_MEM; }
    int rc_all = ORACLE_OK;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < N; ++k) {
        const int64_t n = offsets[k + 1] - offsets[k];
        double *x = (double *)malloc((size_t)(n * d) * sizeof(double));
        int rc = x ? ORACLE_OK : ORACLE_ERR_MEM;
        if (rc == ORACLE_OK) {
            for (int64_t t = 0; t < n * d; ++t) x[t] = (double)X[offsets[k] * d + t];
            double *g = gk ? gk + (size_t)k * (size_t)(m * d) : NULL;
            if (mode == 1) rc = oracle_pair_checkpointed_banded(x, n, z, m, d, gamma, band, &values[k], g);
            else rc = oracle_pair_full_banded(x, n, z, m, d, gamma, band, &values[k], g, NULL, NULL);
        }
        free(x);
        if (rc != ORACLE_OK) {
#pragma omp critical
            rc_all = rc;
        }
    }
    if (grad) {
        for (int64_t t = 0; t < m * d; ++t) grad[t] = 0.0;
        for (int k = 0; k < N; ++k) {
            const double w = weights ? weights[k] : 1.0;
            for (int64_t t = 0; t < m * d; ++t) grad[t] += w * gk[(size_t)k * (size_t)(m * d) + t];
        }
    }
    if (objective) {
        double obj = 0.0;
        for (int k = 0; k < N; ++k) obj += (weights ? weights[k] : 1.0) * values[k];
        *objective = obj;
    }
    free(gk);
    return rc_all;
}

/* ---- barycenter by fixed-step gradient descent ("gradient descent in a
 * straightforward manner"; readings C8, C14): Z(0) = Z0 promoted to double,
 * Z(t+1) = Z(t) - step G(Z(t)), iters times, Z kept in double between iterations.
 * objective[t] = sum_k value_k(Z(t)) (before the t-th update); values = the per-pair values
 * at the last evaluated iterate Z(iters-1).  Because the pair routines take Z as float in
 * oracle_value_grad_f32, this routine carries its own double-Z loop. ---- */
int oracle_barycenter_ex_f32(const float *Z0, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                             double gamma, const double *weights, int64_t band, int iters, double step,
                             double *Z_out, double *values, double *objective, int mode, int nthreads);
int oracle_barycenter_f32(const float *Z0, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                          double gamma, int iters, double step, double *Z_out, double *values, double *objective,
                          int mode, int nthreads) {
    return oracle_barycenter_ex_f32(Z0, m, d, X, offsets, N, gamma, NULL, -1, iters, step, Z_out, values, objective,
                                    mode, nthreads);
}
/* eq. 7 proper: objective sum_k w_k Soft-DTW(Z, x_k) (w_k = lambda_k / n_k in the paper), optional band */
int oracle_barycenter_ex_f32(const float *Z0, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                             double gamma, const double *weights, int64_t band, int iters, double step,
                             double *Z_out, double *values, double *objective, int mode, int nthreads) {
    if (!Z0 || !X || !offsets || !Z_out || m < 1 || d < 1 || N < 1 || !(gamma > 0.0) || iters < 0)
        return ORACLE_ERR_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return ORACLE_ERR_ARG;
    const int64_t md = m * d;
    double *gk = (double *)malloc((size_t)N * (size_t)md * sizeof(double));
    double *vals = (double *)malloc((size_t)N * sizeof(double));
    if (!gk || !vals) { free(gk); free(vals); return ORACLE_ERR_MEM; }
    for (int64_t t = 0; t < md; ++t) Z_out[t] = (double)Z0[t];
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    int rc_all = ORACLE_OK;
    for (int it = 0; it < iters && rc_all == ORACLE_OK; ++it) {
        memset(gk, 0, (size_t)N * (size_t)md * sizeof(double));
#pragma omp parallel for schedule(dynamic, 1)
        for (int k = 0; k < N; ++k) {
            const int64_t n = offsets[k + 1] - offsets[k];
            double *x = (double *)malloc((size_t)(n * d) * sizeof(double));
            int rc = x ? ORACLE_OK : ORACLE_ERR_MEM;
            if (rc == ORACLE_OK) {
                for (int64_t t = 0; t < n * d; ++t) x[t] = (double)X[offsets[k] * d + t];
                double *g = gk + (size_t)k * (size_t)md;
                if (mode == 1) rc = oracle_pair_checkpointed_banded(x, n, Z_out, m, d, gamma, band, &vals[k], g);
                else rc = oracle_pair_full_banded(x, n, Z_out, m, d, gamma, band, &vals[k], g, NULL, NULL);
            }
            free(x);
            if (rc != ORACLE_OK) {
#pragma omp critical
                rc_all = rc;
            }
        }
        if (rc_all != ORACLE_OK) break;
        double obj = 0.0;
        for (int k = 0; k < N; ++k) obj += (weights ? weights[k] : 1.0) * vals[k];
        if (objective) objective[it] = obj;
        if (values) memcpy(values, vals, (size_t)N * sizeof(double));
        for (int64_t t = 0; t < md; ++t) {
            double G = 0.0;
            for (int k = 0; k < N; ++k) G += (weights ? weights[k] : 1.0) * gk[(size_t)k * (size_t)md + t];
            Z_out[t] -= step * G;
        }
    }
    free(gk);
    free(vals);
    return rc_all;
}

/* ---- gradient descent with a backtracking (Armijo) line search on the barycenter objective of eq. 7 -- the
 * stand-in for the off-the-shelf optimiser of Table 1 (reading C22): it
 * removes the step-size fragility of the fixed-step loop with value-only evaluations and vector operations.
 *   f(Z) = sum_k w_k Soft-DTW(Z, x_k),  G = grad f.     Z(0) = Z0 promoted to double.
 *   iteration it:  t = step0;  up to max_trials times:  Zt = Z - t G;  accept if f(Zt) <= f(Z) - c1 t ||G||^2,
 *                  else t = shrink t.   Accepted: Z = Zt, steps[it] = t.  None accepted: steps[it] = 0 and the
 *                  descent stops (remaining entries of steps / trials are 0, objective repeats the last value).
 *   objective[it] = f(Z(it)) for it = 0..iters (iters + 1 entries),  trials[it] = evaluations of f spent. ---- */
int oracle_barycenter_backtracking_f32(const float *Z0, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                                       double gamma, const double *weights, int64_t band, int iters, double step0,
                                       double shrink, double c1, int max_trials, double *Z_out, double *values,
                                       double *objective, double *steps, int32_t *trials, int mode, int nthreads) {
    if (!Z0 || !X || !offsets || !Z_out || !objective || !steps || !trials || m < 1 || d < 1 || N < 1 ||
        !(gamma > 0.0) || iters < 0 || !(step0 > 0.0) || !(shrink > 0.0 && shrink < 1.0) || !(c1 >= 0.0) || max_trials < 1)
        return ORACLE_ERR_ARG;
    const int64_t md = m * d;
    double *G = (double *)malloc((size_t)md * sizeof(double));
    double *Zt = (double *)malloc((size_t)md * sizeof(double));
    double *vals = (double *)malloc((size_t)N * sizeof(double));
    if (!G || !Zt || !vals) { free(G); free(Zt); free(vals); return ORACLE_ERR_MEM; }
    for (int64_t t = 0; t < md; ++t) Z_out[t] = (double)Z0[t];
    for (int it = 0; it < iters; ++it) { steps[it] = 0.0; trials[it] = 0; }
    /* EVAL: f (and G) at a double-precision Z, pair by pair, summed in k order like oracle_barycenter_ex_f32 */
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
    int stopped = 0;
    for (int it = 0; it < iters && rc == ORACLE_OK; ++it) {
        if (stopped) { objective[it + 1] = f; continue; }
        double gg = 0.0;
        for (int64_t t = 0; t < md; ++t) gg += G[t] * G[t];
        double step = step0;
        int accepted = 0;
        for (int tr = 0; tr < max_trials && rc == ORACLE_OK; ++tr) {
            for (int64_t t = 0; t < md; ++t) Zt[t] = Z_out[t] - step * G[t];
            double ft = 0.0;
            EVAL(Zt, 0, ft);
            trials[it] = tr + 1;
            if (ft <= f - c1 * step * gg) {
                memcpy(Z_out, Zt, (size_t)md * sizeof(double));
                steps[it] = step;
                EVAL(Z_out, 1, f);                       /* gradient (and the same f) at the accepted point */
                if (values) memcpy(values, vals, (size_t)N * sizeof(double));
                accepted = 1;
                break;
            }
            step *= shrink;
        }
        if (!accepted) stopped = 1;
        objective[it + 1] = f;
    }
#undef EVAL
    free(G); free(Zt); free(vals);
    return rc;
}

/* ---- Def. 4 / eq. 1: classic DTW by the min-plus dynamic programme (eq. 5 with gamma = 0),
 * squared-Euclidean delta.  Used by the gamma -> 0 pin. ---- */
int oracle_dtw(const double *x, int64_t n, const double *z, int64_t m, int d, double *value) {
    if (!x || !z || !value || n < 1 || m < 1 || d < 1) return ORACLE_ERR_ARG;
    double *D = (double *)malloc((size_t)(n * m) * sizeof(double));
    double *R = (double *)malloc((size_t)((n + 2) * (m + 2)) * sizeof(double));
    if (!D || !R) { free(D); free(R); return ORACLE_ERR_MEM; }
    oracle_cost_matrix(x, n, z, m, d, D);
    oracle_forward_R(D, n, m, 0.0, R);
    *value = R[n * (m + 2) + m];
    free(D);
    free(R);
    return ORACLE_OK;
}

/* ---- Def. 8 / eq. 8: d_score(B, C_k) = DTW(B, C_k) / |pi|, pi the optimal alignment path of
 * eq. 1.  The paper does not say which optimal path is meant when several tie (reading C20): the one obtained by
 * backtracking from (n, m) preferring the diagonal predecessor, then (i-1, j), then (i, j-1) -- equivalently the
 * length is carried forward with the minimum: len[i][j] = 1 + len[argmin], ties resolved in that order.
 * float64 version (the definition): value, path length, and optionally the path itself (i, j pairs, 1-based,
 * from (1,1) to (n,m); path must hold 2 (n + m) int64). ---- */
int oracle_dtw_path(const double *x, int64_t n, const double *z, int64_t m, int d, double *value, int64_t *pathlen,
                    int64_t *path) {
    if (!x || !z || !value || !pathlen || n < 1 || m < 1 || d < 1) return ORACLE_ERR_ARG;
    const int64_t ld = m + 1;
    double *R = (double *)malloc((size_t)((n + 1) * ld) * sizeof(double));
    if (!R) return ORACLE_ERR_MEM;
    for (int64_t j = 0; j <= m; ++j) R[j] = INFINITY;
    for (int64_t i = 0; i <= n; ++i) R[i * ld] = INFINITY;
    R[0] = 0.0;
    for (int64_t i = 1; i <= n; ++i)
        for (int64_t j = 1; j <= m; ++j)
            R[i * ld + j] = delta_sq(x + (i - 1) * d, z + (j - 1) * d, d) +
                            min3(R[(i - 1) * ld + (j - 1)], R[(i - 1) * ld + j], R[i * ld + (j - 1)]);
    *value = R[n * ld + m];
    int64_t i = n, j = m, len = 0;
    int64_t *rev = path ? (int64_t *)malloc((size_t)(2 * (n + m)) * sizeof(int64_t)) : NULL;
    for (;;) {
        if (rev) { rev[2 * len] = i; rev[2 * len + 1] = j; }
        ++len;
        if (i == 1 && j == 1) break;
        const double rd = R[(i - 1) * ld + (j - 1)], ru = R[(i - 1) * ld + j], rl = R[i * ld + (j - 1)];
        const double mn = min3(rd, ru, rl);
        if (rd == mn) { --i; --j; }
        else if (ru == mn) { --i; }
        else { --j; }
    }
    *pathlen = len;
    if (rev) {
        for (int64_t t = 0; t < len; ++t) { path[2 * t] = rev[2 * (len - 1 - t)]; path[2 * t + 1] = rev[2 * (len - 1 - t) + 1]; }
        free(rev);
    }
    free(R);
    return ORACLE_OK;
}

/* ---- the same quantities with every DECISION taken in float32, the precision the CUDA path works in (the path
 * length is an integer decided by float comparisons, so both sides must compare the same numbers): per cell
 *   D = sum_c fl(fl(x_c - z_c)^2)   (c ascending, one rounding per operation, no fused multiply-add)
 *   r = fl(D + min(r_diag, r_up, r_left)),   len = 1 + len of the first of (diag, up, left) that attains the min.
 * Two rows are kept (forward only).  values[k] = DTW, pathlen[k] = |pi|, score[k] = fl(values[k] / fl(pathlen[k])).
 * Mirror of the C-ABI sdtw_dtw_score.  This file is compiled with -ffp-contract=off. ---- */
int oracle_dtw_score_f32(const float *Z, int64_t m, int d, const float *X, const int64_t *offsets, int N,
                         float *values, int32_t *pathlen, float *score, int nthreads) {
    if (!Z || !X || !offsets || !values || !pathlen || !score || m < 1 || d < 1 || N < 1) return ORACLE_ERR_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return ORACLE_ERR_ARG;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    int rc_all = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < N; ++k) {
        const int64_t n = offsets[k + 1] - offsets[k];
        const float *x = X + offsets[k] * d;
        float *r = (float *)malloc((size_t)(2 * (m + 1)) * sizeof(float));
        int32_t *l = (int32_t *)malloc((size_t)(2 * (m + 1)) * sizeof(int32_t));
        if (!r || !l) {
            free(r); free(l);
#pragma omp critical
            rc_all = ORACLE_ERR_MEM;
            continue;
        }
        float *rp = r, *rc = r + (m + 1);
        int32_t *lp = l, *lc = l + (m + 1);
        for (int64_t j = 0; j <= m; ++j) { rp[j] = INFINITY; lp[j] = 0; }
        rp[0] = 0.0f;
        for (int64_t i = 1; i <= n; ++i) {
            rc[0] = INFINITY; lc[0] = 0;
            for (int64_t j = 1; j <= m; ++j) {
                float D = 0.0f;
                for (int c = 0; c < d; ++c) {
                    const float t = x[(i - 1) * d + c] - Z[(j - 1) * d + c];
                    const float t2 = t * t;
                    D = (c == 0) ? t2 : D + t2;
                }
                const float rd = rp[j - 1], ru = rp[j], rl = rc[j - 1];
                float mn = rd;
                if (ru < mn) mn = ru;
                if (rl < mn) mn = rl;
                rc[j] = D + mn;
                lc[j] = 1 + ((rd == mn) ? lp[j - 1] : (ru == mn) ? lp[j] : lc[j - 1]);
            }
            float *tr = rp; rp = rc; rc = tr;
            int32_t *tl = lp; lp = lc; lc = tl;
        }
        values[k] = rp[m];
        pathlen[k] = lp[m];
        score[k] = rp[m] / (float)lp[m];
        free(r); free(l);
    }
    return rc_all;
}

/* ---- Sub-DTW (eq. 2): the whole reference z (m samples) against the best subsequence of a window
 * y (n samples):  min over subsequence alignment paths (all of z traversed, free first and last index along y)
 *               = min_{a <= b} DTW(z, y[a..b]).
 * In this file's index convention rows i run over y (the series with the free ends) and columns j over z:
 *   r_00 = 0, r_i0 = 0 (free start along y), r_0j = +inf (j >= 1),  r_ij = D_ij + min(r_{i-1,j-1}, r_{i-1,j}, r_{i,j-1}),
 *   value = min_i r_im,  b* = the smallest i attaining it,  a* = the row of the first cell of the path obtained by
 *   backtracking from (b*, m) with the preference diagonal, up, left (reading C20) until column 1 is left towards
 *   column 0.  a*, b* are returned 0-based, inclusive.  float64 (the definition). ---- */
int oracle_subdtw(const double *y, int64_t n, const double *z, int64_t m, int d, double *value, int64_t *a_out,
                  int64_t *b_out) {
    if (!y || !z || !value || !a_out || !b_out || n < 1 || m < 1 || d < 1) return ORACLE_ERR_ARG;
    const int64_t ld = m + 1;
    double *R = (double *)malloc((size_t)((n + 1) * ld) * sizeof(double));
    if (!R) return ORACLE_ERR_MEM;
    for (int64_t j = 1; j <= m; ++j) R[j] = INFINITY;
    for (int64_t i = 0; i <= n; ++i) R[i * ld] = 0.0;
    for (int64_t i = 1; i <= n; ++i)
        for (int64_t j = 1; j <= m; ++j)
            R[i * ld + j] = delta_sq(y + (i - 1) * d, z + (j - 1) * d, d) +
                            min3(R[(i - 1) * ld + (j - 1)], R[(i - 1) * ld + j], R[i * ld + (j - 1)]);
    int64_t b = 1;
    for (int64_t i = 2; i <= n; ++i)
        if (R[i * ld + m] < R[b * ld + m]) b = i;
    *value = R[b * ld + m];
    int64_t i = b, j = m;
    for (;;) {                                   /* walk back until the path enters the free column 0 */
        const double rd = R[(i - 1) * ld + (j - 1)], ru = R[(i - 1) * ld + j], rl = R[i * ld + (j - 1)];
        const double mn = min3(rd, ru, rl);
        if (rd == mn) { if (j == 1) break; --i; --j; }
        else if (ru == mn) { --i; }
        else { if (j == 1) break; --j; }
    }
    *a_out = i - 1;
    *b_out = b - 1;
    free(R);
    return ORACLE_OK;
}

/* ---- the same with every decision in float32 and the start row carried forward with the minimum (mirror of the
 * C-ABI sdtw_subdtw; operation order as in oracle_dtw_score_f32).  X holds N windows back to back. ---- */
int oracle_subdtw_f32(const float *Z, int64_t m, int d, const float *X, const int64_t *offsets, int N, float *values,
                      int32_t *a_out, int32_t *b_out, int nthreads) {
    if (!Z || !X || !offsets || !values || !a_out || !b_out || m < 1 || d < 1 || N < 1) return ORACLE_ERR_ARG;
    for (int k = 0; k < N; ++k)
        if (offsets[k + 1] <= offsets[k]) return ORACLE_ERR_ARG;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
    int rc_all = ORACLE_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < N; ++k) {
        const int64_t n = offsets[k + 1] - offsets[k];
        const float *x = X + offsets[k] * d;
        float *r = (float *)malloc((size_t)(2 * (m + 1)) * sizeof(float));
        int32_t *st = (int32_t *)malloc((size_t)(2 * (m + 1)) * sizeof(int32_t));
        if (!r || !st) {
            free(r); free(st);
#pragma omp critical
            rc_all = ORACLE_ERR_MEM;
            continue;
        }
        float *rp = r, *rc = r + (m + 1);
        int32_t *sp = st, *sc = st + (m + 1);
        for (int64_t j = 1; j <= m; ++j) { rp[j] = INFINITY; sp[j] = 0; }
        rp[0] = 0.0f; sp[0] = 0;                      /* column 0 of row i-1 starts a path at row i (0-based i-1 ... ) */
        float best = INFINITY; int32_t best_b = 0, best_a = 0;
        for (int64_t i = 1; i <= n; ++i) {
            sp[0] = (int32_t)(i - 1);                 /* a path entering from (i-1, 0) or (i, 0) starts at 0-based row i-1 */
            rc[0] = 0.0f; sc[0] = (int32_t)(i - 1);
            for (int64_t j = 1; j <= m; ++j) {
                float D = 0.0f;
                for (int c = 0; c < d; ++c) {
                    const float t = x[(i - 1) * d + c] - Z[(j - 1) * d + c];
                    const float t2 = t * t;
                    D = (c == 0) ? t2 : D + t2;
                }
                const float rd = rp[j - 1], ru = rp[j], rl = rc[j - 1];
                float mn = rd;
                if (ru < mn) mn = ru;
                if (rl < mn) mn = rl;
                rc[j] = D + mn;
                sc[j] = (rd == mn) ? sp[j - 1] : (ru == mn) ? sp[j] : sc[j - 1];
            }
            if (rc[m] < best) { best = rc[m]; best_b = (int32_t)(i - 1); best_a = sc[m]; }
            float *tr = rp; rp = rc; rc = tr;
            int32_t *ts = sp; sp = sc; sc = ts;
        }
        values[k] = best; a_out[k] = best_a; b_out[k] = best_b;
        free(r); free(st);
    }
    return rc_all;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
