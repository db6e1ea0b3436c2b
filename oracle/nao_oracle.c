/*
 * nao_oracle.c -- plain, slow, obviously-correct CPU ORACLE for the nao_* hot path.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may build, load or call it.  The CUDA product
 * (paper_2606_09058_b200/csrc) shares no code with this file and never calls it.
 *
 * What it computes (each function cites the passage it follows):
 *   oracle_geneig_{d,z}        H C = S C diag(e)            Eq. 5 / 11 / 21
 *                              route: Cholesky S = L L^H, A = L^{-1} H L^{-H}, cyclic Jacobi, C = L^{-H} Z
 *                              (BASELINE.json north_star; SURVEY.md 8c "Algorithm")
 *   oracle_geneig_lowdin_{d,z} same result by the paper's own route S = U s U^H, V = U s^{-1/2},
 *                              H' = V^H H V, C = V C'
 *   oracle_fermi               Fermi level mu with sum_j w_j f((e_j - mu)/kT) = N_e, f = 1/(1+exp(x))
 *                              (Fermi-Dirac f_i: PAPER.md:42; reading C5)
 *   oracle_density_{d,z}       D = C diag(f) C^H            (north_star; Eq. 8 / 23)
 *
 * Arithmetic: FP64 storage, long double accumulation in inner products (north_star).
 * Pins (tests/test_oracle_pins.py): closed-form chains and rings, 2x2 quadratic brute force, Kronecker 4x4,
 * S = I and block-diagonal cases, invariants (C^H S C = I, residual, Tr(D S) = N_e, congruence invariance),
 * D S = I at f = 1, Fermi closed forms, Loewdin-vs-Cholesky agreement, LAPACK (scipy) cross-check.
 * No function here is "parity unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------ real instantiation ------------------------------ */
#define SCALAR double
#define LSCALAR long double
#define FN(name) name##_d
#define CONJ(x) (x)
#define REALPART(x) (x)
#define ABS2(x) ((x) * (x))
#include "oracle_impl.h"
#undef SCALAR
#undef LSCALAR
#undef FN
#undef CONJ
#undef REALPART
#undef ABS2

/* ----------------------------- complex instantiation ---------------------------- */
#define SCALAR double _Complex
#define LSCALAR long double _Complex
#define FN(name) name##_z
#define CONJ(x) conj(x)
#define REALPART(x) creal(x)
#define ABS2(x) (creal(x) * creal(x) + cimag(x) * cimag(x))
#include "oracle_impl.h"
#undef SCALAR
#undef LSCALAR
#undef FN
#undef CONJ
#undef REALPART
#undef ABS2

int oracle_geneig_d(int n, const double *H, const double *S, double *e, double *C, int *sweeps) {
    return geneig_d(n, H, S, e, C, sweeps);
}
int oracle_geneig_z(int n, const double _Complex *H, const double _Complex *S, double *e, double _Complex *C,
                    int *sweeps) {
    return geneig_z(n, H, S, e, C, sweeps);
}
int oracle_geneig_lowdin_d(int n, const double *H, const double *S, double *e, double *C) {
    return geneig_lowdin_d(n, H, S, e, C);
}
int oracle_geneig_lowdin_z(int n, const double _Complex *H, const double _Complex *S, double *e,
                           double _Complex *C) {
    return geneig_lowdin_z(n, H, S, e, C);
}
void oracle_density_d(int n, const double *C, const double *f, double *D) { density_d(n, C, f, D); }
void oracle_density_z(int n, const double _Complex *C, const double *f, double _Complex *D) {
    density_z(n, C, f, D);
}
int oracle_cholesky_d(int n, double *S) { return cholesky_d(n, S); }
int oracle_cholesky_z(int n, double _Complex *S) { return cholesky_z(n, S); }
int oracle_heev_d(int n, double *A, double *e, double *Z) { return heev_d(n, A, e, Z); }
int oracle_heev_z(int n, double _Complex *A, double *e, double _Complex *Z) { return heev_z(n, A, e, Z); }

/* ------------------------------------------------------------------------------------------------
 * Fermi level (SURVEY 8c reading C5; Fermi-Dirac occupation PAPER.md:42, degeneracy factor Eq. 3).
 * States j = 0..ns-1 with energies e[j] and weights w[j] (= g * w_k of the item the state belongs to).
 *   N(mu) = sum_j w_j f_j,   f_j = 1 / (1 + exp((e_j - mu)/kT))     strictly increasing in mu for kT > 0.
 * To resolve mu inside a gap the equation N(mu) = N_e is solved in particle/hole form: sort the states,
 * let m be the largest count with W_m = sum_{j<m} w_j <= N_e, r = N_e - W_m, and solve
 *   G(mu) = sum_{j>=m} w_j f_j  -  sum_{j<m} w_j (1 - f_j)  -  r = 0        ( == N(mu) - N_e identically ).
 * If r == 0 the root is the root of log P(mu) - log Q(mu) with P, Q the two sums, evaluated with
 * log f = -softplus(x), log(1-f) = -softplus(-x) and log-sum-exp (no cancellation, no underflow).
 * Bisection on [e_min - 50 kT, e_max + 50 kT] in long double until the interval cannot shrink.
 * Outputs *mu and f[j] (stable logistic, original state order).  Returns 0, or 1 if N_e is outside (0, sum w).
 * ------------------------------------------------------------------------------------------------ */
static long double softplusl(long double x) { /* log(1 + exp(x)) */
    return x > 0 ? x + log1pl(expl(-x)) : log1pl(expl(x));
}
static int cmp_idx_e(const void *a, const void *b, void *ctx) {
    const double *e = (const double *)ctx;
    int ia = *(const int *)a, ib = *(const int *)b;
    if (e[ia] < e[ib]) return -1;
    if (e[ia] > e[ib]) return 1;
    return ia - ib;
}
static const double *g_sort_e;
static int cmp_idx_e2(const void *a, const void *b) { return cmp_idx_e(a, b, (void *)g_sort_e); }

int oracle_fermi(int ns, const double *e, const double *w, double n_electrons, double kT, double *mu_out,
                 double *f) {
    long double wsum = 0;
    for (int j = 0; j < ns; ++j) wsum += w[j];
    if (!(n_electrons > 0) || !((long double)n_electrons < wsum) || !(kT > 0)) return 1;
    int *idx = (int *)malloc(sizeof(int) * ns);
    for (int j = 0; j < ns; ++j) idx[j] = j;
    g_sort_e = e; qsort(idx, ns, sizeof(int), cmp_idx_e2);
    int m = 0; long double W = 0;
    while (m < ns && W + (long double)w[idx[m]] <= (long double)n_electrons) { W += w[idx[m]]; ++m; }
    long double r = (long double)n_electrons - W;
    long double lo = (long double)e[idx[0]] - 50.0L * kT, hi = (long double)e[idx[ns - 1]] + 50.0L * kT;
    for (int it = 0; it < 400; ++it) {
        long double mu = 0.5L * (lo + hi);
        if (!(mu > lo && mu < hi)) break;
        int positive;
        if (r == 0.0L && m > 0) {
            /* log P = logsumexp_{j>=m} (log w_j - softplus(x_j)),  log Q = logsumexp_{j<m} (log w_j - softplus(-x_j)) */
            long double mp = -INFINITY, mq = -INFINITY;
            for (int j = 0; j < ns; ++j) {
                long double x = ((long double)e[idx[j]] - mu) / kT;
                long double t = logl((long double)w[idx[j]]) - (j >= m ? softplusl(x) : softplusl(-x));
                if (j >= m) { if (t > mp) mp = t; } else { if (t > mq) mq = t; }
            }
            long double sp = 0, sq = 0;
            for (int j = 0; j < ns; ++j) {
                long double x = ((long double)e[idx[j]] - mu) / kT;
                long double t = logl((long double)w[idx[j]]) - (j >= m ? softplusl(x) : softplusl(-x));
                if (j >= m) sp += expl(t - mp); else sq += expl(t - mq);
            }
            positive = (mp + logl(sp)) > (mq + logl(sq));
        } else {
            long double P = 0, Q = 0;
            for (int j = 0; j < ns; ++j) {
                long double x = ((long double)e[idx[j]] - mu) / kT;
                if (j >= m) P += (long double)w[idx[j]] * expl(-softplusl(x));
                else        Q += (long double)w[idx[j]] * expl(-softplusl(-x));
            }
            positive = (P - Q - r) > 0;
        }
        if (positive) hi = mu; else lo = mu;
    }
    long double mu = 0.5L * (lo + hi);
    *mu_out = (double)mu;
    for (int j = 0; j < ns; ++j) {
        long double x = ((long double)e[j] - mu) / kT;
        f[j] = (double)expl(-softplusl(x));
    }
    free(idx);
    return 0;
}
