/*
 * oracle_impl.h -- body of the CPU oracle, included twice by nao_oracle.c:
 * once with SCALAR = double (real symmetric), once with SCALAR = double _Complex
 * (complex Hermitian).  TEST INFRASTRUCTURE ONLY -- see nao_oracle.c header.
 *
 * Column-major storage: element (i,j) of an n*n matrix M is M[j*n + i].
 * FP64 storage, long double accumulation in every inner product (north_star).
 */

/* ---- 1. Cholesky S = L L^H, unblocked, column by column (north_star) ----
 * Overwrites the lower triangle of S with L, zeroes the strict upper triangle.
 * Returns 0, or j+1 if the j-th pivot (0-based j) is not positive (LAPACK potrf convention). */
static int FN(cholesky)(int n, SCALAR *S) {
    for (int j = 0; j < n; ++j) {
        long double acc = (long double)REALPART(S[(size_t)j * n + j]);
        for (int k = 0; k < j; ++k) acc -= (long double)ABS2(S[(size_t)k * n + j]);
        if (!(acc > 0.0L)) return j + 1;
        double ljj = (double)sqrtl(acc);
        S[(size_t)j * n + j] = ljj;
        #pragma omp parallel for schedule(static)
        for (int i = j + 1; i < n; ++i) {
            LSCALAR s = (LSCALAR)S[(size_t)j * n + i];
            for (int k = 0; k < j; ++k)
                s -= (LSCALAR)S[(size_t)k * n + i] * (LSCALAR)CONJ(S[(size_t)k * n + j]);
            S[(size_t)j * n + i] = (SCALAR)(s / (long double)ljj);
        }
    }
    for (int j = 1; j < n; ++j)
        for (int i = 0; i < j; ++i) S[(size_t)j * n + i] = 0;
    return 0;
}

/* ---- 2. A = L^{-1} H L^{-H}: forward substitution on the columns of H,
 * then on the rows of the result; finally symmetrise A <- (A + A^H)/2.  H is overwritten by A. */
static void FN(reduce_to_standard)(int n, const SCALAR *L, SCALAR *H) {
    /* X = L^{-1} H : for each column c solve L x = h_c */
    #pragma omp parallel for schedule(static)
    for (int c = 0; c < n; ++c) {
        SCALAR *x = H + (size_t)c * n;
        for (int i = 0; i < n; ++i) {
            LSCALAR s = (LSCALAR)x[i];
            for (int k = 0; k < i; ++k) s -= (LSCALAR)L[(size_t)k * n + i] * (LSCALAR)x[k];
            x[i] = (SCALAR)(s / (long double)REALPART(L[(size_t)i * n + i]));
        }
    }
    /* A = X L^{-H} : for each row r solve a_r L^H = x_r, i.e. a_r[j] = (x_r[j] - sum_{k<j} a_r[k] conj(L[j,k])) / L[j,j] */
    #pragma omp parallel for schedule(static)
    for (int r = 0; r < n; ++r) {
        for (int j = 0; j < n; ++j) {
            LSCALAR s = (LSCALAR)H[(size_t)j * n + r];
            for (int k = 0; k < j; ++k)
                s -= (LSCALAR)H[(size_t)k * n + r] * (LSCALAR)CONJ(L[(size_t)k * n + j]);
            H[(size_t)j * n + r] = (SCALAR)(s / (long double)REALPART(L[(size_t)j * n + j]));
        }
    }
    for (int j = 0; j < n; ++j) {
        H[(size_t)j * n + j] = REALPART(H[(size_t)j * n + j]);
        for (int i = j + 1; i < n; ++i) {
            SCALAR a = 0.5 * (H[(size_t)j * n + i] + CONJ(H[(size_t)i * n + j]));
            H[(size_t)j * n + i] = a;
            H[(size_t)i * n + j] = CONJ(a);
        }
    }
}

/* ---- 3. cyclic two-sided Jacobi on Hermitian A ----
 * Round-robin (tournament) ordering: every round holds n/2 disjoint pairs (p,q).  The rotation
 *     J = [ c , s*phi ; -s*conj(phi) , c ],   phi = a_pq/|a_pq|,
 *     zeta = (a_qq - a_pp) / (2|a_pq|),  t = sign(zeta)/(|zeta| + sqrt(1+zeta^2)),  c = 1/sqrt(1+t^2), s = t c
 * annihilates a_pq in A <- J^H A J.  Per round: all rotation parameters from the current A (disjoint pairs do
 * not touch each other's 2x2 blocks), then all row updates (A <- J^H A), then all column updates (A <- A J,
 * Z <- Z J).  The product of disjoint rotations commutes, so the result equals applying them one by one and is
 * independent of the thread count.  On exit diag(A) holds the eigenvalues and Z (n*n) the eigenvectors.
 * Returns the number of sweeps done. */
static int FN(jacobi)(int n, SCALAR *A, SCALAR *Z, int max_sweeps) {
    int m = n + (n & 1);              /* players in the tournament (one dummy if n is odd) */
    int half = m / 2;
    int *top = (int *)malloc(sizeof(int) * half), *bot = (int *)malloc(sizeof(int) * half);
    double *cs = (double *)malloc(sizeof(double) * half), *sn = (double *)malloc(sizeof(double) * half);
    SCALAR *ph = (SCALAR *)malloc(sizeof(SCALAR) * half);
    int *pp = (int *)malloc(sizeof(int) * half), *qq = (int *)malloc(sizeof(int) * half);
    for (size_t i = 0; i < (size_t)n * n; ++i) Z[i] = 0;
    for (int i = 0; i < n; ++i) Z[(size_t)i * n + i] = 1.0;
    long double fro = 0;
    for (size_t i = 0; i < (size_t)n * n; ++i) fro += (long double)ABS2(A[i]);
    double normA = (double)sqrtl(fro);
    double prev_off = -1.0;
    int sweep = 0;
    for (; sweep < max_sweeps; ++sweep) {
        long double off2 = 0;
        for (int j = 0; j < n; ++j)
            for (int i = 0; i < n; ++i)
                if (i != j) off2 += (long double)ABS2(A[(size_t)j * n + i]);
        double off = (double)sqrtl(off2);
        if (off <= 1e-15 * normA) break;
        if (sweep >= 5 && prev_off >= 0 && off > 0.5 * prev_off) break;   /* rounding floor reached */
        prev_off = off;
        for (int i = 0; i < half; ++i) { top[i] = i; bot[i] = m - 1 - i; }
        for (int round = 0; round < m - 1; ++round) {
            int np = 0;
            for (int i = 0; i < half; ++i) {
                int p = top[i], q = bot[i];
                if (p >= n || q >= n) continue;
                if (p > q) { int t = p; p = q; q = t; }
                SCALAR apq = A[(size_t)q * n + p];
                double g = sqrt(ABS2(apq));
                if (g == 0.0) continue;
                double app = REALPART(A[(size_t)p * n + p]), aqq = REALPART(A[(size_t)q * n + q]);
                double zeta = (aqq - app) / (2.0 * g);
                double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
                double c = 1.0 / sqrt(1.0 + t * t);
                pp[np] = p; qq[np] = q; cs[np] = c; sn[np] = t * c; ph[np] = apq / g; ++np;
            }
            /* rows: A <- J^H A :  row_p' = c row_p - s phi row_q ;  row_q' = s conj(phi) row_p + c row_q */
            #pragma omp parallel for schedule(static)
            for (int j = 0; j < n; ++j) {
                SCALAR *col = A + (size_t)j * n;
                for (int r = 0; r < np; ++r) {
                    SCALAR ap = col[pp[r]], aq = col[qq[r]];
                    col[pp[r]] = cs[r] * ap - sn[r] * ph[r] * aq;
                    col[qq[r]] = sn[r] * CONJ(ph[r]) * ap + cs[r] * aq;
                }
            }
            /* columns: A <- A J, Z <- Z J :  col_p' = c col_p - s conj(phi) col_q ;  col_q' = s phi col_p + c col_q */
            #pragma omp parallel for schedule(static)
            for (int r = 0; r < np; ++r) {
                SCALAR *cp = A + (size_t)pp[r] * n, *cq = A + (size_t)qq[r] * n;
                SCALAR *zp = Z + (size_t)pp[r] * n, *zq = Z + (size_t)qq[r] * n;
                for (int i = 0; i < n; ++i) {
                    SCALAR ap = cp[i], aq = cq[i];
                    cp[i] = cs[r] * ap - sn[r] * CONJ(ph[r]) * aq;
                    cq[i] = sn[r] * ph[r] * ap + cs[r] * aq;
                    SCALAR vp = zp[i], vq = zq[i];
                    zp[i] = cs[r] * vp - sn[r] * CONJ(ph[r]) * vq;
                    zq[i] = sn[r] * ph[r] * vp + cs[r] * vq;
                }
            }
            /* the annihilated entries are exactly zero in exact arithmetic; set them so */
            for (int r = 0; r < np; ++r) {
                A[(size_t)qq[r] * n + pp[r]] = 0; A[(size_t)pp[r] * n + qq[r]] = 0;
                A[(size_t)pp[r] * n + pp[r]] = REALPART(A[(size_t)pp[r] * n + pp[r]]);
                A[(size_t)qq[r] * n + qq[r]] = REALPART(A[(size_t)qq[r] * n + qq[r]]);
            }
            /* rotate the tournament: player top[0] stays, the others move one seat */
            int last_top = top[half - 1], first_bot = bot[0];
            for (int i = half - 1; i > 1; --i) top[i] = top[i - 1];
            if (half > 1) top[1] = first_bot;
            for (int i = 0; i < half - 1; ++i) bot[i] = bot[i + 1];
            bot[half - 1] = last_top;
            if (half == 1) { /* n == 2: single pair, nothing to rotate */ bot[0] = first_bot; }
        }
    }
    free(top); free(bot); free(cs); free(sn); free(ph); free(pp); free(qq);
    return sweep;
}

/* ---- Hermitian eigen-decomposition A = Z diag(e) Z^H, ascending (steps 3-4) ---- */
static int FN(heev)(int n, SCALAR *A, double *e, SCALAR *Z) {
    int sweeps = FN(jacobi)(n, A, Z, 30);
    int *idx = (int *)malloc(sizeof(int) * n);
    for (int i = 0; i < n; ++i) idx[i] = i;
    /* insertion sort of indices by eigenvalue (stable) */
    for (int i = 1; i < n; ++i) {
        int k = idx[i]; double v = REALPART(A[(size_t)k * n + k]); int j = i - 1;
        while (j >= 0 && REALPART(A[(size_t)idx[j] * n + idx[j]]) > v) { idx[j + 1] = idx[j]; --j; }
        idx[j + 1] = k;
    }
    SCALAR *tmp = (SCALAR *)malloc(sizeof(SCALAR) * (size_t)n * n);
    for (int j = 0; j < n; ++j) {
        e[j] = REALPART(A[(size_t)idx[j] * n + idx[j]]);
        memcpy(tmp + (size_t)j * n, Z + (size_t)idx[j] * n, sizeof(SCALAR) * n);
    }
    memcpy(Z, tmp, sizeof(SCALAR) * (size_t)n * n);
    free(tmp); free(idx);
    return sweeps;
}

/* ---- 4. C = L^{-H} Z by back substitution ---- */
static void FN(back_substitute)(int n, const SCALAR *L, SCALAR *Z) {
    #pragma omp parallel for schedule(static)
    for (int c = 0; c < n; ++c) {
        SCALAR *x = Z + (size_t)c * n;
        for (int i = n - 1; i >= 0; --i) {
            LSCALAR s = (LSCALAR)x[i];
            for (int k = i + 1; k < n; ++k) s -= (LSCALAR)CONJ(L[(size_t)i * n + k]) * (LSCALAR)x[k];
            x[i] = (SCALAR)(s / (long double)REALPART(L[(size_t)i * n + i]));
        }
    }
}

/* Generalized Hermitian-definite eigenproblem H C = S C diag(e), Cholesky route (Eq. 5/11/21:
 * PAPER.md:50, 75, 113-115).  H, S: n*n inputs (not modified).  Outputs e[n] ascending, C n*n with C^H S C = I.
 * Returns 0 ok, j>0 if the leading minor j of S is not positive definite. */
static int FN(geneig)(int n, const SCALAR *H, const SCALAR *S, double *e, SCALAR *C, int *sweeps_out) {
    size_t nn = (size_t)n * n;
    SCALAR *L = (SCALAR *)malloc(sizeof(SCALAR) * nn), *A = (SCALAR *)malloc(sizeof(SCALAR) * nn);
    memcpy(L, S, sizeof(SCALAR) * nn); memcpy(A, H, sizeof(SCALAR) * nn);
    int info = FN(cholesky)(n, L);
    if (info) { free(L); free(A); return info; }
    FN(reduce_to_standard)(n, L, A);
    int sw = FN(heev)(n, A, e, C);
    if (sweeps_out) *sweeps_out = sw;
    FN(back_substitute)(n, L, C);
    free(L); free(A);
    return 0;
}

/* Loewdin route of the paper (section 3.1 Part 2-1..2-5):
 * S = U s U^H, V = U s^{-1/2}, H' = V^H H V, H' C' = C' e, C = V C'.  Cross-check of the Cholesky route. */
static int FN(geneig_lowdin)(int n, const SCALAR *H, const SCALAR *S, double *e, SCALAR *C) {
    size_t nn = (size_t)n * n;
    SCALAR *W = (SCALAR *)malloc(sizeof(SCALAR) * nn), *U = (SCALAR *)malloc(sizeof(SCALAR) * nn);
    SCALAR *T = (SCALAR *)malloc(sizeof(SCALAR) * nn), *Cp = (SCALAR *)malloc(sizeof(SCALAR) * nn);
    double *s = (double *)malloc(sizeof(double) * n);
    memcpy(W, S, sizeof(SCALAR) * nn);
    FN(heev)(n, W, s, U);
    for (int j = 0; j < n; ++j) {
        if (!(s[j] > 0)) { free(W); free(U); free(T); free(Cp); free(s); return j + 1; }
        double f = 1.0 / sqrt(s[j]);
        for (int i = 0; i < n; ++i) U[(size_t)j * n + i] *= f;          /* U now holds V */
    }
    /* T = H V */
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            LSCALAR acc = 0;
            for (int k = 0; k < n; ++k) acc += (LSCALAR)H[(size_t)k * n + i] * (LSCALAR)U[(size_t)j * n + k];
            T[(size_t)j * n + i] = (SCALAR)acc;
        }
    /* W = V^H T, symmetrised */
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            LSCALAR acc = 0;
            for (int k = 0; k < n; ++k) acc += (LSCALAR)CONJ(U[(size_t)i * n + k]) * (LSCALAR)T[(size_t)j * n + k];
            W[(size_t)j * n + i] = (SCALAR)acc;
        }
    for (int j = 0; j < n; ++j) {
        W[(size_t)j * n + j] = REALPART(W[(size_t)j * n + j]);
        for (int i = j + 1; i < n; ++i) {
            SCALAR a = 0.5 * (W[(size_t)j * n + i] + CONJ(W[(size_t)i * n + j]));
            W[(size_t)j * n + i] = a; W[(size_t)i * n + j] = CONJ(a);
        }
    }
    FN(heev)(n, W, e, Cp);
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < n; ++j)
        for (int i = 0; i < n; ++i) {
            LSCALAR acc = 0;
            for (int k = 0; k < n; ++k) acc += (LSCALAR)U[(size_t)k * n + i] * (LSCALAR)Cp[(size_t)j * n + k];
            C[(size_t)j * n + i] = (SCALAR)acc;
        }
    free(W); free(U); free(T); free(Cp); free(s);
    return 0;
}

/* ---- 6. density matrix D = C diag(f) C^H = sum_i f_i c_i c_i^H (north_star; Eq. 8/23 PAPER.md:63, 129 is its
 * complex conjugate, reading C3).  Long double accumulation. ---- */
static void FN(density)(int n, const SCALAR *C, const double *f, SCALAR *D) {
    #pragma omp parallel for schedule(dynamic, 4)
    for (int m = 0; m < n; ++m)
        for (int l = 0; l < n; ++l) {
            LSCALAR acc = 0;
            for (int i = 0; i < n; ++i)
                acc += (long double)f[i] * ((LSCALAR)C[(size_t)i * n + l] * (LSCALAR)CONJ(C[(size_t)i * n + m]));
            D[(size_t)m * n + l] = (SCALAR)acc;
        }
}
