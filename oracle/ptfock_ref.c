/*
 * ptfock_ref.c -- CPU ORACLE for the plane-wave Fock exchange application.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no
 * code, table or constant generator with the CUDA path (paper_1905_01348_b200/csrc).
 *
 * What it computes (Sec. 2, Eq. (3); Sec. 3.2, Alg. 2;
 * readings Q1-Q16 of SURVEY.md Sec. 8(c), repeated in DESIGN.md):
 *
 *   for each target j, each orbital i:
 *       rho(r)  = conj(phi_i(r)) * psi_j(r)                          (Eq. 3: "psi_i^*(r') psi_j(r')")
 *       rho^(k) = sum_r rho(r) exp(-2 pi i sum_d k_d x_d / n_d)       (forward DFT, unnormalised)
 *       W^(k)   = v(|G(k)|^2) * rho^(k)                               ("Poisson-like equation")
 *       W(r)    = (1/N) sum_k W^(k) exp(+2 pi i sum_d k_d x_d / n_d)  (inverse DFT)
 *       out_j(r) -= alpha * phi_i(r) * W(r)                           (Alg. 2 line 8: "add the solution to (V_X Psi)_j")
 *
 *   v(G^2) = 4 pi / G^2,                         v(0) = 0          (bare Coulomb, BASELINE.json north_star)
 *   v(G^2) = 4 pi / G^2 * (1 - exp(-G^2/(4 w^2))), v(0) = pi / w^2  (HSE-screened; G->0 limit, reading Q2)
 *   E_x    = 1/2 * (Omega/N) * Re sum_j sum_r conj(psi_j(r)) out_j(r)   (reading Q11)
 *
 * G(k) = sum_d m_d b_d with m_d = k_d for k_d < n_d/2 else k_d - n_d (so m_d in [-n_d/2, n_d/2), reading Q5)
 * and b_d the reciprocal lattice vectors (b_d . a_e = 2 pi delta_de) of the cell rows a_0, a_1, a_2.
 *
 * Layout (reading Q16): C order [orbital][x0][x1][x2], x2 contiguous, interleaved (re, im) fp64.
 *
 * How it computes it: fp64 storage; the 3-D DFT is done axis by axis with a plain recursive
 * decimation-in-time Cooley-Tukey for factors 2 and 3 (anything else falls to the O(n^2) DFT);
 * twiddles are cosl/sinl in long double rounded once to double; the sum over i is carried in
 * long double.  No blocking, no fusion, no symmetry tricks: every (i, j) pair is one forward and
 * one inverse 3-D transform, in the order of Alg. 2.  OpenMP over target columns only.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): plane-wave closed form (T1), O(N^2) real-space
 * brute-force convolution (T2), Hermiticity (T3), unitary invariance (T4), E_x real and <= 0 (T5),
 * FFT vs the O(n^2) DFT / round trip / Parseval / delta (T6), periodic Poisson textbook case (T7),
 * structure: W_ji = conj(W_ij), linearity, real orbitals, grid shift (T8).
 * Parity unpinned against PWDFT itself: the paper prints no value of V_X Psi or E_x.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libptfock_ref.so ptfock_ref.c -lm      (no -ffast-math)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double re, im; } cplx;

#define REF_OK 0
#define REF_EINVAL (-1)
#define REF_ENOMEM (-2)

static const long double PI_L = 3.14159265358979323846264338327950288L;

/* ------------------------------------------------------------------------------------------
 * 1-D transforms.  sign = -1: forward  X[k] = sum_x x[x] exp(-2 pi i k x / n)   (reading Q4)
 *                  sign = +1: inverse without the 1/n.
 * ------------------------------------------------------------------------------------------ */

/* w[t] = exp(sign * 2 pi i t / n), t = 0..n-1, evaluated in long double, rounded once. */
static void fill_twiddles(int n, int sign, cplx *w) {
    for (int t = 0; t < n; ++t) {
        long double a = 2.0L * PI_L * (long double)t / (long double)n;
        w[t].re = (double)cosl(a);
        w[t].im = (double)(sign < 0 ? -sinl(a) : sinl(a));
    }
}

/* The definition itself: O(n^2), long double accumulation.  Used to test the FFT (T6). */
void ptfock_ref_dft1d_naive(int n, int sign, const double *in, double *out) {
    const cplx *x = (const cplx *)in;
    cplx *y = (cplx *)out;
    for (int k = 0; k < n; ++k) {
        long double sr = 0.0L, si = 0.0L;
        for (int t = 0; t < n; ++t) {
            long long kt = ((long long)k * t) % n;
            long double a = 2.0L * PI_L * (long double)kt / (long double)n;
            long double c = cosl(a), s = (sign < 0 ? -sinl(a) : sinl(a));
            sr += (long double)x[t].re * c - (long double)x[t].im * s;
            si += (long double)x[t].re * s + (long double)x[t].im * c;
        }
        y[k].re = (double)sr;
        y[k].im = (double)si;
    }
}

/* Recursive decimation in time.  in has stride istride, out is contiguous, w = twiddles of the
 * TOP-level length ntop (w[t] = exp(sign 2 pi i t / ntop)); a sub-transform of length n uses
 * w[t * (ntop / n)].  tmp is scratch of length n at this level. */
static void fft_rec(int n, int ntop, const cplx *w, const cplx *in, int istride, cplx *out, cplx *tmp) {
    if (n == 1) { out[0] = in[0]; return; }
    int step = ntop / n;
    if (n % 2 == 0) {
        int h = n / 2;
        /* even samples -> tmp[0..h), odd samples -> tmp[h..n) ; each needs scratch: reuse out */
        fft_rec(h, ntop, w, in, 2 * istride, tmp, out);
        fft_rec(h, ntop, w, in + istride, 2 * istride, tmp + h, out);
        for (int k = 0; k < h; ++k) {
            cplx e = tmp[k], o = tmp[h + k], t = w[k * step], p;
            p.re = t.re * o.re - t.im * o.im;
            p.im = t.re * o.im + t.im * o.re;
            out[k].re = e.re + p.re;       out[k].im = e.im + p.im;
            out[k + h].re = e.re - p.re;   out[k + h].im = e.im - p.im;
        }
    } else if (n % 3 == 0) {
        int h = n / 3;
        fft_rec(h, ntop, w, in, 3 * istride, tmp, out);
        fft_rec(h, ntop, w, in + istride, 3 * istride, tmp + h, out);
        fft_rec(h, ntop, w, in + 2 * istride, 3 * istride, tmp + 2 * h, out);
        for (int k = 0; k < n; ++k) {
            /* X[k] = A[k mod h] + w^k B[k mod h] + w^{2k} C[k mod h] */
            int kk = k % h;
            cplx a = tmp[kk], b = tmp[h + kk], c = tmp[2 * h + kk];
            cplx t1 = w[(k * step) % ntop], t2 = w[(int)(((long long)2 * k * step) % ntop)];
            out[k].re = a.re + (t1.re * b.re - t1.im * b.im) + (t2.re * c.re - t2.im * c.im);
            out[k].im = a.im + (t1.re * b.im + t1.im * b.re) + (t2.re * c.im + t2.im * c.re);
        }
    } else {
        /* plain DFT with the table (only reached for lengths with a factor other than 2, 3) */
        for (int k = 0; k < n; ++k) {
            double sr = 0.0, si = 0.0;
            for (int t = 0; t < n; ++t) {
                cplx tw = w[(int)(((long long)k * t * step) % ntop)];
                cplx x = in[(size_t)t * istride];
                sr += x.re * tw.re - x.im * tw.im;
                si += x.re * tw.im + x.im * tw.re;
            }
            out[k].re = sr; out[k].im = si;
        }
    }
}

/* Exported for T6: one 1-D transform of contiguous data, sign -1 / +1, unnormalised. */
int ptfock_ref_fft1d(int n, int sign, const double *in, double *out) {
    if (n < 1 || (sign != 1 && sign != -1)) return REF_EINVAL;
    cplx *w = (cplx *)malloc(sizeof(cplx) * n), *tmp = (cplx *)malloc(sizeof(cplx) * n);
    if (!w || !tmp) { free(w); free(tmp); return REF_ENOMEM; }
    fill_twiddles(n, sign, w);
    fft_rec(n, n, w, (const cplx *)in, 1, (cplx *)out, tmp);
    free(w); free(tmp);
    return REF_OK;
}

/* In-place 3-D transform, axis by axis (x2, then x1, then x0), unnormalised. */
typedef struct { int n[3]; cplx *w[3]; } tw3;

static int tw3_init(tw3 *t, const int n[3], int sign) {
    for (int d = 0; d < 3; ++d) { t->n[d] = n[d]; t->w[d] = NULL; }
    for (int d = 0; d < 3; ++d) {
        t->w[d] = (cplx *)malloc(sizeof(cplx) * n[d]);
        if (!t->w[d]) return REF_ENOMEM;
        fill_twiddles(n[d], sign, t->w[d]);
    }
    return REF_OK;
}
static void tw3_free(tw3 *t) { for (int d = 0; d < 3; ++d) free(t->w[d]); }

/* buf: 3 * max(n) cplx of scratch */
static void fft3d_inplace(const tw3 *t, cplx *g, cplx *buf) {
    const int n0 = t->n[0], n1 = t->n[1], n2 = t->n[2];
    int nmax = n0 > n1 ? n0 : n1; if (n2 > nmax) nmax = n2;
    cplx *pin = buf, *pout = buf + nmax, *tmp = buf + 2 * nmax;
    /* axis 2 (contiguous) */
    for (int a = 0; a < n0 * n1; ++a) {
        cplx *p = g + (size_t)a * n2;
        fft_rec(n2, n2, t->w[2], p, 1, pout, tmp);
        memcpy(p, pout, sizeof(cplx) * n2);
    }
    /* axis 1 */
    for (int x0 = 0; x0 < n0; ++x0)
        for (int x2 = 0; x2 < n2; ++x2) {
            cplx *p = g + (size_t)x0 * n1 * n2 + x2;
            for (int x1 = 0; x1 < n1; ++x1) pin[x1] = p[(size_t)x1 * n2];
            fft_rec(n1, n1, t->w[1], pin, 1, pout, tmp);
            for (int x1 = 0; x1 < n1; ++x1) p[(size_t)x1 * n2] = pout[x1];
        }
    /* axis 0 */
    for (int r = 0; r < n1 * n2; ++r) {
        cplx *p = g + r;
        for (int x0 = 0; x0 < n0; ++x0) pin[x0] = p[(size_t)x0 * n1 * n2];
        fft_rec(n0, n0, t->w[0], pin, 1, pout, tmp);
        for (int x0 = 0; x0 < n0; ++x0) p[(size_t)x0 * n1 * n2] = pout[x0];
    }
}

/* Exported for T6: in-place unnormalised 3-D transform of one grid. */
int ptfock_ref_fft3d(const int32_t n[3], int sign, double *grid) {
    if (n[0] < 1 || n[1] < 1 || n[2] < 1 || (sign != 1 && sign != -1)) return REF_EINVAL;
    int nn[3] = { n[0], n[1], n[2] };
    tw3 t;
    if (tw3_init(&t, nn, sign) != REF_OK) { tw3_free(&t); return REF_ENOMEM; }
    int nmax = nn[0] > nn[1] ? nn[0] : nn[1]; if (nn[2] > nmax) nmax = nn[2];
    cplx *buf = (cplx *)malloc(sizeof(cplx) * 3 * nmax);
    if (!buf) { tw3_free(&t); return REF_ENOMEM; }
    fft3d_inplace(&t, (cplx *)grid, buf);
    free(buf); tw3_free(&t);
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * Interaction kernel on the FFT grid ("K(r-r') ... (possibly screened)"; formulas
 * from BASELINE.json north_star; G = 0 values: reading Q2).
 * ------------------------------------------------------------------------------------------ */

static double det3(const double a[9]) {
    return a[0] * (a[4] * a[8] - a[5] * a[7]) - a[1] * (a[3] * a[8] - a[5] * a[6]) + a[2] * (a[3] * a[7] - a[4] * a[6]);
}

/* rows of b: reciprocal vectors, b_d . a_e = 2 pi delta_de */
static void reciprocal(const double a[9], double b[9]) {
    double vol = det3(a);
    const double *a0 = a, *a1 = a + 3, *a2 = a + 6;
    double c12[3] = { a1[1] * a2[2] - a1[2] * a2[1], a1[2] * a2[0] - a1[0] * a2[2], a1[0] * a2[1] - a1[1] * a2[0] };
    double c20[3] = { a2[1] * a0[2] - a2[2] * a0[1], a2[2] * a0[0] - a2[0] * a0[2], a2[0] * a0[1] - a2[1] * a0[0] };
    double c01[3] = { a0[1] * a1[2] - a0[2] * a1[1], a0[2] * a1[0] - a0[0] * a1[2], a0[0] * a1[1] - a0[1] * a1[0] };
    double f = 2.0 * (double)PI_L / vol;
    for (int c = 0; c < 3; ++c) { b[c] = f * c12[c]; b[3 + c] = f * c20[c]; b[6 + c] = f * c01[c]; }
}

/* kernel: 0 = bare Coulomb, 1 = HSE screened.  v has N doubles, C order over (k0, k1, k2). */
int ptfock_ref_vtable(const double cell[9], const int32_t n[3], int kernel, double omega, double *v) {
    if (kernel != 0 && kernel != 1) return REF_EINVAL;
    if (kernel == 1 && !(omega > 0.0)) return REF_EINVAL;
    double b[9];
    if (det3(cell) == 0.0) return REF_EINVAL;
    reciprocal(cell, b);
    const double four_pi = 4.0 * (double)PI_L;
    for (int k0 = 0; k0 < n[0]; ++k0) {
        int m0 = (k0 < (n[0] + 1) / 2) ? k0 : k0 - n[0];      /* even n: k = n/2 -> m = -n/2 */
        for (int k1 = 0; k1 < n[1]; ++k1) {
            int m1 = (k1 < (n[1] + 1) / 2) ? k1 : k1 - n[1];
            for (int k2 = 0; k2 < n[2]; ++k2) {
                int m2 = (k2 < (n[2] + 1) / 2) ? k2 : k2 - n[2];
                double gx = m0 * b[0] + m1 * b[3] + m2 * b[6];
                double gy = m0 * b[1] + m1 * b[4] + m2 * b[7];
                double gz = m0 * b[2] + m1 * b[5] + m2 * b[8];
                double g2 = gx * gx + gy * gy + gz * gz;
                double val;
                if (m0 == 0 && m1 == 0 && m2 == 0)
                    val = (kernel == 0) ? 0.0 : (double)PI_L / (omega * omega);
                else if (kernel == 0)
                    val = four_pi / g2;
                else
                    val = four_pi / g2 * (-expm1(-g2 / (4.0 * omega * omega)));
                v[((size_t)k0 * n[1] + k1) * n[2] + k2] = val;
            }
        }
    }
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * W_ij for one pair (exported for T8: W_ji = conj(W_ij)).  w_out: N cplx.
 * ------------------------------------------------------------------------------------------ */
static void pair_solve(const tw3 *tf, const tw3 *ti, const double *v, size_t N,
                       const cplx *phi_i, const cplx *psi_j, cplx *w, cplx *buf) {
    for (size_t r = 0; r < N; ++r) {           /* rho = conj(phi_i) psi_j */
        w[r].re = phi_i[r].re * psi_j[r].re + phi_i[r].im * psi_j[r].im;
        w[r].im = phi_i[r].re * psi_j[r].im - phi_i[r].im * psi_j[r].re;
    }
    fft3d_inplace(tf, w, buf);                 /* rho^(k) */
    for (size_t k = 0; k < N; ++k) { w[k].re *= v[k]; w[k].im *= v[k]; }
    fft3d_inplace(ti, w, buf);                 /* N * W(r) */
    const double inv = 1.0 / (double)N;
    for (size_t r = 0; r < N; ++r) { w[r].re *= inv; w[r].im *= inv; }
}

int ptfock_ref_pair_w(const double cell[9], const int32_t n[3], int kernel, double omega,
                      const double *phi_i, const double *psi_j, double *w_out) {
    size_t N = (size_t)n[0] * n[1] * n[2];
    int nn[3] = { n[0], n[1], n[2] };
    double *v = (double *)malloc(sizeof(double) * N);
    if (!v) return REF_ENOMEM;
    int rc = ptfock_ref_vtable(cell, n, kernel, omega, v);
    if (rc != REF_OK) { free(v); return rc; }
    tw3 tf, ti;
    int nmax = nn[0] > nn[1] ? nn[0] : nn[1]; if (nn[2] > nmax) nmax = nn[2];
    cplx *buf = (cplx *)malloc(sizeof(cplx) * 3 * nmax);
    if (tw3_init(&tf, nn, -1) != REF_OK || tw3_init(&ti, nn, +1) != REF_OK || !buf) {
        tw3_free(&tf); tw3_free(&ti); free(buf); free(v); return REF_ENOMEM;
    }
    pair_solve(&tf, &ti, v, N, (const cplx *)phi_i, (const cplx *)psi_j, (cplx *)w_out, buf);
    tw3_free(&tf); tw3_free(&ti); free(buf); free(v);
    return REF_OK;
}

/* ------------------------------------------------------------------------------------------
 * out[c] = V_X[Phi] psi_{cols[c]},  c = 0..n_cols-1  (cols == NULL: cols[c] = c).
 * phi: n_occ grids; psi: n_targets grids (may be the same pointer as phi); out: n_cols grids.
 * Each requested column sums over ALL i = 0..n_occ-1, so a subset of columns is exact for those
 * columns.  Returns the number of pair-solves executed in *pairs_done (may be NULL).
 * ------------------------------------------------------------------------------------------ */
int ptfock_ref_apply(const double cell[9], const int32_t n[3], int kernel, double omega, double alpha,
                     int32_t n_occ, const double *phi, int32_t n_targets, const double *psi,
                     const int32_t *cols, int32_t n_cols, double *out, int64_t *pairs_done) {
    if (n_occ < 0 || n_targets < 0 || n_cols < 0) return REF_EINVAL;
    for (int d = 0; d < 3; ++d) if (n[d] < 1) return REF_EINVAL;
    for (int c = 0; c < n_cols; ++c) {
        int j = cols ? cols[c] : c;
        if (j < 0 || j >= n_targets) return REF_EINVAL;
    }
    const size_t N = (size_t)n[0] * n[1] * n[2];
    int nn[3] = { n[0], n[1], n[2] };
    double *v = (double *)malloc(sizeof(double) * N);
    if (!v) return REF_ENOMEM;
    int rc = ptfock_ref_vtable(cell, n, kernel, omega, v);
    if (rc != REF_OK) { free(v); return rc; }
    tw3 tf, ti;
    if (tw3_init(&tf, nn, -1) != REF_OK || tw3_init(&ti, nn, +1) != REF_OK) {
        tw3_free(&tf); tw3_free(&ti); free(v); return REF_ENOMEM;
    }
    int nmax = nn[0] > nn[1] ? nn[0] : nn[1]; if (nn[2] > nmax) nmax = nn[2];
    int failed = 0;
    const cplx *PHI = (const cplx *)phi, *PSI = (const cplx *)psi;
    cplx *OUT = (cplx *)out;

#pragma omp parallel
    {
        cplx *w = (cplx *)malloc(sizeof(cplx) * N);
        cplx *buf = (cplx *)malloc(sizeof(cplx) * 3 * nmax);
        long double *acc = (long double *)malloc(sizeof(long double) * 2 * N);
        if (!w || !buf || !acc) {
#pragma omp atomic write
            failed = 1;
        }
#pragma omp barrier
        if (!failed) {
#pragma omp for schedule(dynamic, 1)
            for (int c = 0; c < n_cols; ++c) {
                int j = cols ? cols[c] : c;
                const cplx *psi_j = PSI + (size_t)j * N;
                for (size_t r = 0; r < 2 * N; ++r) acc[r] = 0.0L;      /* Alg. 2 line 1 */
                for (int i = 0; i < n_occ; ++i) {                       /* Alg. 2 line 2 */
                    const cplx *phi_i = PHI + (size_t)i * N;
                    pair_solve(&tf, &ti, v, N, phi_i, psi_j, w, buf);   /* Alg. 2 line 8 */
                    for (size_t r = 0; r < N; ++r) {                    /* out_j -= alpha phi_i W */
                        long double pr = (long double)phi_i[r].re * w[r].re - (long double)phi_i[r].im * w[r].im;
                        long double pi = (long double)phi_i[r].re * w[r].im + (long double)phi_i[r].im * w[r].re;
                        acc[2 * r] -= (long double)alpha * pr;
                        acc[2 * r + 1] -= (long double)alpha * pi;
                    }
                }
                cplx *o = OUT + (size_t)c * N;
                for (size_t r = 0; r < N; ++r) { o[r].re = (double)acc[2 * r]; o[r].im = (double)acc[2 * r + 1]; }
            }
        }
        free(w); free(buf); free(acc);
    }
    tw3_free(&tf); tw3_free(&ti); free(v);
    if (failed) return REF_ENOMEM;
    if (pairs_done) *pairs_done = (int64_t)n_cols * n_occ;
    return REF_OK;
}

/* E_x = 1/2 (Omega/N) Re sum_c sum_r conj(psi_{cols[c]}(r)) vx[c](r); also returns the imaginary
 * part of the same sum (should vanish, T5) in e[1].  vx: n_cols grids as written by ptfock_ref_apply. */
int ptfock_ref_exchange_energy(const double cell[9], const int32_t n[3], const double *psi,
                               const int32_t *cols, int32_t n_cols, const double *vx, double e[2]) {
    const size_t N = (size_t)n[0] * n[1] * n[2];
    const cplx *PSI = (const cplx *)psi, *VX = (const cplx *)vx;
    long double sr = 0.0L, si = 0.0L;
    for (int c = 0; c < n_cols; ++c) {
        int j = cols ? cols[c] : c;
        const cplx *p = PSI + (size_t)j * N, *q = VX + (size_t)c * N;
        for (size_t r = 0; r < N; ++r) {
            sr += (long double)p[r].re * q[r].re + (long double)p[r].im * q[r].im;
            si += (long double)p[r].re * q[r].im - (long double)p[r].im * q[r].re;
        }
    }
    long double f = 0.5L * fabsl((long double)det3(cell)) / (long double)N;
    e[0] = (double)(f * sr);
    e[1] = (double)(f * si);
    return REF_OK;
}

int ptfock_ref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
