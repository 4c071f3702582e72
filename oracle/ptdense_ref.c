/*
 * ptdense_ref.c -- CPU ORACLE for the dense-algebra neighbours of the Fock exchange path (TEST INFRASTRUCTURE, not
 * the product; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may use it; it shares no code
 * with paper_1905_01348_b200/).
 *
 * What it computes (plain definitions, written out; fp64 storage, long double accumulation, no blocking):
 *
 *   orbitals: n columns of N grid values, complex, C order [orbital][point]; inner product
 *       (a, b) = w * sum_r conj(a(r)) b(r),   w = Omega / N                     (reading Q11 / Q14)
 *
 *   overlap      S[m][n]   = (a_m, b_n)                                          PAPER.md:183 Alg. 3 line 2
 *                                                                                 "S_temp = Psi_f^* H_f Psi_f"
 *                                                                                 "overlap matrix of the type Psi^* Psi"
 *   rotate       out_n(r)  = sum_m a_m(r) S[m][n]                                PAPER.md:185 Alg. 3 line 4 "Psi_temp = Psi_f S"
 *   residual_n   R_n       = H Psi - Psi (Psi^* H Psi)                           PAPER.md:80 Alg. 1 line 1 (minus sign lost in the
 *                                                                                 extraction: read with Eq. (4)/(5))
 *   residual_f   R_f       = Psi_f + (i dt/2) (H Psi_f - Psi_f (Psi_f^* H Psi_f)) - Psi_half
 *                                                                                 PAPER.md:186 Alg. 3 line 5, signs from Eq. (5)
 *   density      rho(r)    = sum_i |psi_i(r)|^2                                  PAPER.md:192 Sec. 3.4
 *   cholesky     S = L L^H, L lower triangular with a real positive diagonal     PAPER.md:200 "Cholesky decomposition on the
 *                                                                                 overlap matrix"
 *   orthonormalize  Psi <- Psi L^{-H}  with  L L^H = Psi^* Psi                   PAPER.md:200 "rotate Psi_f ... via ... Trsm"
 *                   (column n: out_n = (psi_n - sum_{m<n} out_m conj(L[n][m])) / L[n][n])
 *
 * Pins (tests/test_oracle_dense_pins.py): plane-wave closed forms (S = diag, rho = n/Omega, R_n = 0 for eigenvectors of the
 * kinetic operator), orthonormal seeded orbitals give S = I, R_n is orthogonal to Psi, sum_r rho w = n, L L^H = S on a
 * hand-worked 2 x 2 case and on random Hermitian positive matrices, the orthonormalised set equals classical Gram-Schmidt
 * done with scalar Python loops, spans the same space and is a fixed point for orthonormal input.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;
typedef long double complex lcplx;

/* S[m*n_b + n] = w * sum_r conj(a[m][r]) b[n][r] */
int ptdense_ref_overlap(int64_t n_pts, double w, const double *a_, int32_t n_a, const double *b_, int32_t n_b, double *s_) {
    if (n_pts < 1 || n_a < 0 || n_b < 0 || !a_ || !b_ || !s_) return -1;
    const cplx *a = (const cplx *)a_, *b = (const cplx *)b_;
    cplx *s = (cplx *)s_;
#pragma omp parallel for collapse(2) schedule(static)
    for (int m = 0; m < n_a; ++m)
        for (int n = 0; n < n_b; ++n) {
            lcplx acc = 0.0L;
            const cplx *am = a + (size_t)m * n_pts, *bn = b + (size_t)n * n_pts;
            for (int64_t r = 0; r < n_pts; ++r) acc += (lcplx)conj(am[r]) * (lcplx)bn[r];
            s[(size_t)m * n_b + n] = (cplx)(acc * (long double)w);
        }
    return 0;
}

/* out[n][r] = sum_m a[m][r] S[m*n_out + n] */
int ptdense_ref_rotate(int64_t n_pts, const double *a_, int32_t n_a, const double *s_, int32_t n_out, double *out_) {
    if (n_pts < 1 || n_a < 0 || n_out < 0 || !a_ || !s_ || !out_) return -1;
    const cplx *a = (const cplx *)a_, *s = (const cplx *)s_;
    cplx *out = (cplx *)out_;
#pragma omp parallel for schedule(static)
    for (int n = 0; n < n_out; ++n)
        for (int64_t r = 0; r < n_pts; ++r) {
            lcplx acc = 0.0L;
            for (int m = 0; m < n_a; ++m) acc += (lcplx)a[(size_t)m * n_pts + r] * (lcplx)s[(size_t)m * n_out + n];
            out[(size_t)n * n_pts + r] = (cplx)acc;
        }
    return 0;
}

/* psi_half == NULL:  R = H Psi - Psi (Psi^* H Psi)                                        (Alg. 1 line 1)
 * else:              R = Psi + (i dt / 2) (H Psi - Psi (Psi^* H Psi)) - Psi_half          (Alg. 3 line 5) */
int ptdense_ref_residual(int64_t n_pts, double w, int32_t n, double dt, const double *psi_, const double *hpsi_,
                         const double *half_, double *r_) {
    if (n_pts < 1 || n < 1 || !psi_ || !hpsi_ || !r_) return -1;
    const cplx *psi = (const cplx *)psi_, *hpsi = (const cplx *)hpsi_, *half = (const cplx *)half_;
    cplx *r = (cplx *)r_;
    cplx *s = (cplx *)malloc(sizeof(cplx) * (size_t)n * n);
    cplx *t = (cplx *)malloc(sizeof(cplx) * (size_t)n * n_pts);
    if (!s || !t) { free(s); free(t); return -2; }
    int rc = ptdense_ref_overlap(n_pts, w, psi_, n, hpsi_, n, (double *)s);
    if (rc == 0) rc = ptdense_ref_rotate(n_pts, psi_, n, (const double *)s, n, (double *)t);
    if (rc == 0) {
        const cplx f = I * (dt / 2.0);
        for (size_t k = 0; k < (size_t)n * n_pts; ++k) {
            const cplx d = hpsi[k] - t[k];
            r[k] = half ? psi[k] + f * d - half[k] : d;
        }
    }
    free(s);
    free(t);
    return rc;
}

/* rho[r] = sum_i |psi[i][r]|^2 */
int ptdense_ref_density(int64_t n_pts, const double *psi_, int32_t n, double *rho) {
    if (n_pts < 1 || n < 0 || !psi_ || !rho) return -1;
    const cplx *psi = (const cplx *)psi_;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < n_pts; ++r) {
        long double acc = 0.0L;
        for (int i = 0; i < n; ++i) {
            const cplx z = psi[(size_t)i * n_pts + r];
            acc += (long double)creal(z) * creal(z) + (long double)cimag(z) * cimag(z);
        }
        rho[r] = (double)acc;
    }
    return 0;
}

/* S (n x n, Hermitian positive definite, row major; only the lower triangle is read) = L L^H; l gets L (upper part zero).
 * Cholesky-Banachiewicz, row by row.  Returns 1 + the failing row if S is not positive definite. */
int ptdense_ref_cholesky(int32_t n, const double *s_, double *l_) {
    if (n < 1 || !s_ || !l_) return -1;
    const cplx *s = (const cplx *)s_;
    cplx *l = (cplx *)l_;
    memset(l, 0, sizeof(cplx) * (size_t)n * n);
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j <= i; ++j) {
            lcplx acc = (lcplx)s[(size_t)i * n + j];
            for (int k = 0; k < j; ++k) acc -= (lcplx)l[(size_t)i * n + k] * (lcplx)conj(l[(size_t)j * n + k]);
            if (i == j) {
                const long double d = creall(acc);
                if (!(d > 0.0L)) return 1 + i;
                l[(size_t)i * n + i] = (double)sqrtl(d);
            } else {
                l[(size_t)i * n + j] = (cplx)(acc / (long double)creal(l[(size_t)j * n + j]));
            }
        }
    }
    return 0;
}

/* out = Psi L^{-H} with L L^H = Psi^* Psi (inner product weight w): out^* out = I.  out may not alias psi. */
int ptdense_ref_orthonormalize(int64_t n_pts, double w, const double *psi_, int32_t n, double *out_) {
    if (n_pts < 1 || n < 1 || !psi_ || !out_) return -1;
    const cplx *psi = (const cplx *)psi_;
    cplx *out = (cplx *)out_;
    cplx *s = (cplx *)malloc(sizeof(cplx) * (size_t)n * n), *l = (cplx *)malloc(sizeof(cplx) * (size_t)n * n);
    if (!s || !l) { free(s); free(l); return -2; }
    int rc = ptdense_ref_overlap(n_pts, w, psi_, n, psi_, n, (double *)s);
    if (rc == 0) rc = ptdense_ref_cholesky(n, (const double *)s, (double *)l);
    if (rc == 0) {
        /* out L^H = Psi, column by column: out_c = (psi_c - sum_{m<c} out_m conj(L[c][m])) / L[c][c] */
#pragma omp parallel for schedule(static)
        for (int64_t r = 0; r < n_pts; ++r)
            for (int c = 0; c < n; ++c) {
                lcplx acc = (lcplx)psi[(size_t)c * n_pts + r];
                for (int m = 0; m < c; ++m) acc -= (lcplx)out[(size_t)m * n_pts + r] * (lcplx)conj(l[(size_t)c * n + m]);
                out[(size_t)c * n_pts + r] = (cplx)(acc / (long double)creal(l[(size_t)c * n + c]));
            }
    }
    free(s);
    free(l);
    return rc;
}
