/* Matrix-free oracle matvec (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).
 *
 * Plain C, double precision, OpenMP over target rows.  Computes, for the requested target
 * scatterers j, u_j = sum_{i != j, same window} A_ji x_i with
 *   [A_ji]_{b a} = e^{i mu phi} sum_q coef[q][b][a] h_q^(1)(k r) Pbar_q^{|mu|}(cos theta),  mu = mu_tab[b][a]
 * (PAPER.md:304-308 Eq. I17 and PAPER.md:336 Eq. I21; d = x_j - x_i = (r, theta, phi)).
 * The constant tables coef (= a5/b5 of Eq. I18) and mu come from oracle/translation.py
 * (coupling_tables); this file only evaluates h_q, Pbar_q^mu and the sums, for sizes where
 * the dense matrix of oracle/system.py does not fit.  Pinned against that dense assembly in
 * tests/test_oracle_matvec.py.  Shares nothing with the CUDA path.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QMAX 16

static double fact(int n) { double f = 1.0; for (int i = 2; i <= n; ++i) f *= i; return f; }

/* Pbar_q^m(x) = sqrt((2q+1)/2 (q-m)!/(q+m)!) (1-x^2)^{m/2} d^m P_q/dx^m, no Condon-Shortley phase */
static void pbar_all(int qmax, double ct, double st, double P[QMAX][QMAX]) {
    double U[QMAX][QMAX];                       /* unnormalised, U_m^m = (2m-1)!! sin^m */
    for (int m = 0; m <= qmax; ++m) {
        double pmm = 1.0;
        for (int i = 1; i <= m; ++i) pmm *= (2 * i - 1) * st;
        U[m][m] = pmm;
        if (m + 1 <= qmax) U[m + 1][m] = ct * (2 * m + 1) * pmm;
        for (int q = m + 2; q <= qmax; ++q)
            U[q][m] = ((2 * q - 1) * ct * U[q - 1][m] - (q + m - 1) * U[q - 2][m]) / (q - m);
    }
    for (int q = 0; q <= qmax; ++q)
        for (int m = 0; m <= q; ++m)
            P[q][m] = sqrt((2 * q + 1) / 2.0 * fact(q - m) / fact(q + m)) * U[q][m];
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_matvec_rows(int lmax, double k, int n_scat, const double *pos, const int *win_ptr, int n_win,
                        const double complex *coef, const int *mu_tab,
                        int n_rows, const int *rows, const double complex *x, double complex *y) {
    const int L = 2 * lmax * (lmax + 2);
    const int nq = 2 * lmax + 1;
    int *win_of = (int *)malloc(sizeof(int) * n_scat);
    for (int w = 0; w < n_win; ++w)
        for (int i = win_ptr[w]; i < win_ptr[w + 1]; ++i) win_of[i] = w;
#pragma omp parallel for schedule(dynamic, 1)
    for (int rr = 0; rr < n_rows; ++rr) {
        const int j = rows[rr];
        const int w = win_of[j];
        double complex *acc = y + (size_t)rr * L;
        for (int b = 0; b < L; ++b) acc[b] = 0.0;
        for (int i = win_ptr[w]; i < win_ptr[w + 1]; ++i) {
            if (i == j) continue;
            const double dx = pos[3 * j] - pos[3 * i], dy = pos[3 * j + 1] - pos[3 * i + 1],
                         dz = pos[3 * j + 2] - pos[3 * i + 2];
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            const double ct = dz / r, st = sqrt(dx * dx + dy * dy) / r;
            const double phi = atan2(dy, dx);
            const double kr = k * r;
            double complex h[QMAX];
            h[0] = -I * cexp(I * kr) / kr;
            h[1] = -(kr + I) * cexp(I * kr) / (kr * kr);
            for (int q = 1; q + 1 < nq; ++q) h[q + 1] = (2 * q + 1) / kr * h[q] - h[q - 1];
            double P[QMAX][QMAX];
            pbar_all(nq - 1, ct, st, P);
            double complex e[2 * QMAX + 1];     /* e[mu + nq] = exp(i mu phi) */
            for (int m = -(nq - 1); m <= nq - 1; ++m) e[m + nq] = cexp(I * m * phi);
            const double complex *xi = x + (size_t)i * L;
            for (int b = 0; b < L; ++b) {
                double complex s = 0.0;
                for (int a = 0; a < L; ++a) {
                    const int mu = mu_tab[b * L + a];
                    const int am = mu < 0 ? -mu : mu;
                    double complex ent = 0.0;
                    for (int q = am; q < nq; ++q) ent += coef[((size_t)q * L + b) * L + a] * h[q] * P[q][am];
                    s += ent * e[mu + nq] * xi[a];
                }
                acc[b] += s;
            }
        }
    }
    free(win_of);
}
