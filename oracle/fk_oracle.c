/*
 * fk_oracle.c -- TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, obviously-correct CPU statement of what the FK-convolution hot path computes,
 * written from /root/reference/PAPER.md (P:NN = line NN):
 *
 *   hadronic  sigma^N = sum_{i,j,alpha,beta} f_alpha(x_i) f_beta(x_j) FK^N_{ij alpha beta}   P:43, Eq. (1)
 *             (meaning of f, FK and the N-vector: P:45; only a sparse list of (alpha,beta)
 *              "flavour combinations" is stored: P:100; R PDF replicas = R columns: P:81)
 *   DIS       sigma^N = sum_{i,alpha} f_alpha(x_i) FK^N_{i alpha}     (never printed in the paper, which only has
 *              "DIS" rows in Table 1; formula = BASELINE.json north_star; reading R1)
 *   gradient  "the convolution and its corresponding gradient": the vector-Jacobian product
 *              df[r][alpha][i] = d( sum_n g[n][r] sigma[n][r] ) / d f[r][alpha][i], written as the literal
 *              derivative of Eq. (1) in scatter form (reading R8).
 *
 * The method reaches exactly (up to rounding order) this plain definition, so the oracle IS the
 * definition: nested loops over (n, c, i, j) in that order, no blocking, fusion or reordering.
 * Accumulation is in `long double` (x87 80-bit here) because a plain sequential fp64 sum misses the
 * 1e-13 parity tolerance on same-sign inputs; each routine also emits the tolerance
 * denominator sum|terms| in the same pass.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call
 * this.  It shares no code with the CUDA path (paper_1909_10547_b200/csrc) and neither includes the other.
 *
 * Pins (tests/test_oracle_pins.py): exact-rational brute force, one-hot and separable tables,
 * closed forms, bilinearity, DIS-as-hadronic, numpy GEMM view, finite differences and Euler's
 * identity for the VJP.  Paper's Table 1 values: parity unpinned - inputs not published.
 *
 * Layouts (logical, BASELINE.json): FK_h[N][nx][nx][C] (i, j, channel; channel innermost),
 * FK_dis[N][nx][nA], pairs[C][2] = (a_c, b_c) ordered (i <-> a_c, j <-> b_c; reading R3),
 * f[R][nfl][nx], sigma[N][R], g[N][R], df[R][nfl][nx].
 * Returns 0, or -1 on an invalid argument (null pointer, non-positive size, flavour index out of range).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double acc_t;

static int check_index_list(const int32_t *idx, long n, int nfl) {
    for (long k = 0; k < n; ++k)
        if (idx[k] < 0 || idx[k] >= nfl) return -1;
    return 0;
}

int fk_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. (1), with two PDFs (f1 on the i/alpha leg, f2 on the j/beta leg); the paper's pp case
 * is f1 == f2 (reading R6).  The two-PDF form exists only so that bilinearity and the
 * DIS-as-hadronic special case can be checked directly. */
int fk_oracle_hadronic2(const double *fk, const int32_t *pairs, const double *f1, const double *f2,
                        double *sigma, double *scale, int N, int nx, int nfl, int C, int R) {
    if (!fk || !pairs || !f1 || !f2 || !sigma || N <= 0 || nx <= 0 || nfl <= 0 || C <= 0 || R <= 0) return -1;
    if (check_index_list(pairs, 2L * C, nfl)) return -1;
#pragma omp parallel for schedule(static)
    for (int n = 0; n < N; ++n) {
        for (int r = 0; r < R; ++r) {
            acc_t acc = 0.0L, S = 0.0L;
            for (int c = 0; c < C; ++c) {
                const int a = pairs[2 * c + 0], b = pairs[2 * c + 1];
                for (int i = 0; i < nx; ++i) {
                    for (int j = 0; j < nx; ++j) {
                        const double FK = fk[(((size_t)n * nx + i) * nx + j) * C + c];
                        const acc_t t = (acc_t)f1[((size_t)r * nfl + a) * nx + i] *
                                        (acc_t)f2[((size_t)r * nfl + b) * nx + j] * (acc_t)FK;
                        acc += t;
                        S += fabsl(t);
                    }
                }
            }
            sigma[(size_t)n * R + r] = (double)acc;
            if (scale) scale[(size_t)n * R + r] = (double)S;
        }
    }
    return 0;
}

int fk_oracle_hadronic(const double *fk, const int32_t *pairs, const double *f, double *sigma, double *scale,
                       int N, int nx, int nfl, int C, int R) {
    return fk_oracle_hadronic2(fk, pairs, f, f, sigma, scale, N, nx, nfl, C, R);
}

/* DIS: sigma^N = sum_{i,alpha} f_alpha(x_i) FK^N_{i alpha} over the active-flavour list (reading R1). */
int fk_oracle_dis(const double *fk, const int32_t *flav, const double *f, double *sigma, double *scale,
                  int N, int nx, int nfl, int nA, int R) {
    if (!fk || !flav || !f || !sigma || N <= 0 || nx <= 0 || nfl <= 0 || nA <= 0 || R <= 0) return -1;
    if (check_index_list(flav, nA, nfl)) return -1;
#pragma omp parallel for schedule(static)
    for (int n = 0; n < N; ++n) {
        for (int r = 0; r < R; ++r) {
            acc_t acc = 0.0L, S = 0.0L;
            for (int c = 0; c < nA; ++c) {
                const int a = flav[c];
                for (int i = 0; i < nx; ++i) {
                    const acc_t t = (acc_t)f[((size_t)r * nfl + a) * nx + i] *
                                    (acc_t)fk[((size_t)n * nx + i) * nA + c];
                    acc += t;
                    S += fabsl(t);
                }
            }
            sigma[(size_t)n * R + r] = (double)acc;
            if (scale) scale[(size_t)n * R + r] = (double)S;
        }
    }
    return 0;
}

/* Gradient of P:47 as a VJP: the literal derivative of Eq. (1), scatter form.  Each FK element feeds
 * df[a_c][i] (factor f[b_c][j]) and df[b_c][j] (factor f[a_c][i]); a_c == b_c with i == j therefore
 * receives both contributions automatically.  Flavours in no pair get exactly 0. */
int fk_oracle_hadronic_vjp(const double *fk, const int32_t *pairs, const double *f, const double *g,
                           double *df, double *dscale, int N, int nx, int nfl, int C, int R) {
    if (!fk || !pairs || !f || !g || !df || N <= 0 || nx <= 0 || nfl <= 0 || C <= 0 || R <= 0) return -1;
    if (check_index_list(pairs, 2L * C, nfl)) return -1;
    const size_t per = (size_t)nfl * nx;
    int fail = 0;
#pragma omp parallel for schedule(static)
    for (int r = 0; r < R; ++r) {
        acc_t *d = (acc_t *)calloc(2 * per, sizeof(acc_t));
        if (!d) { fail = 1; continue; }
        acc_t *D = d + per;
        const double *fr = f + (size_t)r * per;
        for (int n = 0; n < N; ++n) {
            const acc_t gn = (acc_t)g[(size_t)n * R + r];
            for (int c = 0; c < C; ++c) {
                const int a = pairs[2 * c + 0], b = pairs[2 * c + 1];
                for (int i = 0; i < nx; ++i) {
                    for (int j = 0; j < nx; ++j) {
                        const acc_t w = gn * (acc_t)fk[(((size_t)n * nx + i) * nx + j) * C + c];
                        const acc_t ta = w * (acc_t)fr[(size_t)b * nx + j];
                        const acc_t tb = w * (acc_t)fr[(size_t)a * nx + i];
                        d[(size_t)a * nx + i] += ta;  D[(size_t)a * nx + i] += fabsl(ta);
                        d[(size_t)b * nx + j] += tb;  D[(size_t)b * nx + j] += fabsl(tb);
                    }
                }
            }
        }
        for (size_t k = 0; k < per; ++k) {
            df[(size_t)r * per + k] = (double)d[k];
            if (dscale) dscale[(size_t)r * per + k] = (double)D[k];
        }
        free(d);
    }
    return fail ? -1 : 0;
}

/* DIS gradient (Table 1 has DIS "Gradient" rows): df[r][flav_c][i] += g[n][r] FK[n][i][c]. */
int fk_oracle_dis_vjp(const double *fk, const int32_t *flav, const double *f, const double *g,
                      double *df, double *dscale, int N, int nx, int nfl, int nA, int R) {
    (void)f; /* sigma is linear in f: the derivative does not depend on it */
    if (!fk || !flav || !g || !df || N <= 0 || nx <= 0 || nfl <= 0 || nA <= 0 || R <= 0) return -1;
    if (check_index_list(flav, nA, nfl)) return -1;
    const size_t per = (size_t)nfl * nx;
    int fail = 0;
#pragma omp parallel for schedule(static)
    for (int r = 0; r < R; ++r) {
        acc_t *d = (acc_t *)calloc(2 * per, sizeof(acc_t));
        if (!d) { fail = 1; continue; }
        acc_t *D = d + per;
        for (int n = 0; n < N; ++n) {
            const acc_t gn = (acc_t)g[(size_t)n * R + r];
            for (int c = 0; c < nA; ++c) {
                const int a = flav[c];
                for (int i = 0; i < nx; ++i) {
                    const acc_t t = gn * (acc_t)fk[((size_t)n * nx + i) * nA + c];
                    d[(size_t)a * nx + i] += t;  D[(size_t)a * nx + i] += fabsl(t);
                }
            }
        }
        for (size_t k = 0; k < per; ++k) {
            df[(size_t)r * per + k] = (double)d[k];
            if (dscale) dscale[(size_t)r * per + k] = (double)D[k];
        }
        free(d);
    }
    return fail ? -1 : 0;
}

/* Figure of merit of the fit step that follows the convolution (reading R22: the paper
 * only says "gradient descent optimization", and never prints the loss -- this is the standard quadratic
 * form over the data covariance):
 *     chi2[r] = sum_{n,m} d[n][r] Cinv[n][m] d[m][r],   d[n][r] = sigma[n][r] - data[n]
 *     g[n][r] = d chi2[r] / d sigma[n][r] = 2 sum_m Cinv[n][m] d[m][r]        (Cinv symmetric)
 * Literal double loops, long double accumulation; cscale[r] / gscale[n][r] = sum |terms| (tolerance denominators). */
int fk_oracle_chi2(const double *sigma, const double *data, const double *cinv, double *chi2, double *cscale,
                   double *g, double *gscale, int N, int R) {
    if (!sigma || !data || !cinv || !chi2 || !g || N <= 0 || R <= 0) return -1;
    for (int r = 0; r < R; ++r) {
        acc_t tot = 0, totabs = 0;
        for (int n = 0; n < N; ++n) {
            const acc_t dn = (acc_t)sigma[(size_t)n * R + r] - (acc_t)data[n];
            acc_t row = 0, rowabs = 0;
            for (int m = 0; m < N; ++m) {
                const acc_t dm = (acc_t)sigma[(size_t)m * R + r] - (acc_t)data[m];
                const acc_t t = (acc_t)cinv[(size_t)n * N + m] * dm;
                row += t;  rowabs += fabsl(t);
                tot += dn * t;  totabs += fabsl(dn * t);
            }
            g[(size_t)n * R + r] = (double)(2 * row);
            if (gscale) gscale[(size_t)n * R + r] = (double)(2 * rowabs);
        }
        chi2[r] = (double)tot;
        if (cscale) cscale[r] = (double)totabs;
    }
    return 0;
}
