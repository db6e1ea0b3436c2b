// stedc_core.cuh -- scalar building blocks of the tridiagonal divide-and-conquer eigensolver (
// the paper names the method -- "divide-and-conquer ... dominated by matrix multiplications", PAPER.md:744 -- the
// algorithm itself is Cuppen's rank-one tearing with Gu/Eisenstat deflation and Loewner-formula eigenvectors, restated
// here from the published algorithm).  The formulations followed are the ones the reference libraries made standard:
// `deflate_range` is the deflation loop of LAPACK dlaed2 (its column types 1-4 and index names are kept so that the two can be
// read side by side), `secular_root` follows LAPACK dlaed4's scheme (origin shifted to the nearer pole, the `erretm` stopping
// test, the two-pole "middle way" step), and `ql_implicit` is the implicit QL iteration of EISPACK tql2 / imtql2 in its
// textbook form.  No library source is copied; the code is written from the published descriptions of those routines.
//
//   T = [T1 0; 0 T2] + rho v v^T  ->  D + rho z z^T  ->  deflation  ->  secular equation  ->  eigenvectors.
//
// Everything in this header is __host__ __device__ and free of CUDA intrinsics except through the `Lanes` policy,
// so that the numerics can be exercised on the host (the product only ever calls them from kernels).
#pragma once
#include <math.h>
#include <float.h>

namespace nao {
namespace dc {

#define NAO_HD __host__ __device__ __forceinline__

static const double DC_EPS = 1.1102230246251565e-16;      // 2^-53, unit roundoff

// ---------------------------------------------------------------------------------------------------------------
// Lane policies: a "team" of cooperating lanes evaluates the sums of the secular function.
//   SerialLanes: one lane (host tests, or one thread per root).   WarpLanes (stedc.cu): 32 lanes + xor-shuffle.
// ---------------------------------------------------------------------------------------------------------------
struct SerialLanes {
    NAO_HD int lane() const { return 0; }
    NAO_HD int count() const { return 1; }
    NAO_HD double sum(double v) const { return v; }
};

// ---------------------------------------------------------------------------------------------------------------
// Secular equation.  Poles d[0] < d[1] < ... < d[K-1] (strictly increasing after deflation), weights z[i] != 0,
// rho > 0.  Root number j of
//        f(lambda) = 1/rho + sum_i z_i^2 / (d_i - lambda)
// lies in (d_j, d_{j+1}) for j < K-1 and in (d_{K-1}, d_{K-1} + rho |z|^2] for j = K-1.
// The unknown is tau = lambda - d_org with the origin d_org the nearer pole, so that every difference
//        delta_i = (d_i - d_org) - tau = d_i - lambda
// is obtained to high RELATIVE accuracy (this is what makes the Loewner eigenvector formula work).
// Iteration: osculatory two-pole rational interpolation ("middle way"), safeguarded by a bracket [lo, hi] that
// always contains the root; a step that leaves the bracket, or too many steps, falls back to bisection.
// On exit: *lambda = d_org + tau; delta[i] = d_i - lambda for all i (written by the lanes, stride lanes.count()).
// Returns the number of iterations used (>= 0), or -1 if the residual test was not met within the cap (the
// bracket has then been bisected to working precision, so the root is still accurate).
// ---------------------------------------------------------------------------------------------------------------
template <class Lanes>
NAO_HD int secular_root(const Lanes &L, int K, int j, const double *__restrict__ d, const double *__restrict__ z,
                        double rho, double *__restrict__ delta, double *lambda) {
    const double rhoinv = 1.0 / rho;
    const int ln = L.lane(), nl = L.count();
    if (K == 1) {
        double tau = rho * z[0] * z[0];
        if (ln == 0) delta[0] = -tau;
        *lambda = d[0] + tau;
        return 0;
    }
    const bool last = (j == K - 1);
    int org;            // origin pole
    double lo, hi, tau;
    const int jl = last ? K - 2 : j, jr = jl + 1;          // the two poles that bracket (or precede) the root
    const double del = d[jr] - d[jl];
    if (!last) {
        // f at the midpoint decides which half holds the root
        const double mid = 0.5 * del;                      // relative to d[j]
        double s = 0.0;
        for (int i = ln; i < K; i += nl)
            if (i != jl && i != jr) s += z[i] * z[i] / ((d[i] - d[jl]) - mid);
        const double c0 = rhoinv + L.sum(s);
        const double fmid = c0 + z[jl] * z[jl] / (-mid) + z[jr] * z[jr] / (del - mid);
        const double zl2 = z[jl] * z[jl], zr2 = z[jr] * z[jr];
        if (fmid > 0.0) {          // root in the left half: origin d[j], tau in (0, del/2]
            org = jl; lo = 0.0; hi = mid;
            const double a = c0 * del + zl2 + zr2, b = zl2 * del;
            const double disc = sqrt(fabs(a * a - 4.0 * b * c0));
            tau = (a > 0.0) ? 2.0 * b / (a + disc) : (a - disc) / (2.0 * c0);
        } else {                   // right half: origin d[j+1], tau in [-del/2, 0)
            org = jr; lo = -mid; hi = 0.0;
            const double a = zl2 + zr2 - c0 * del, b = -zr2 * del;
            const double disc = sqrt(fabs(a * a - 4.0 * b * c0));
            tau = (a > 0.0) ? 2.0 * b / (a + disc) : (a - disc) / (2.0 * c0);
        }
        if (!(tau > lo && tau < hi)) tau = 0.5 * (lo + hi);
    } else {
        // last root: origin d[K-1], tau in (0, rho |z|^2]
        double s = 0.0;
        for (int i = ln; i < K; i += nl) s += z[i] * z[i];
        const double znorm2 = L.sum(s);
        org = K - 1; lo = 0.0; hi = rho * znorm2;
        // two-pole start: c0 + zl2/(-del - tau) + zr2/(-tau) = 0 with the other poles frozen at tau = hi/2
        const double mid = 0.5 * hi;
        s = 0.0;
        for (int i = ln; i < K - 2; i += nl) s += z[i] * z[i] / ((d[i] - d[K - 1]) - mid);
        const double c0 = rhoinv + L.sum(s);
        const double zl2 = z[jl] * z[jl], zr2 = z[jr] * z[jr];
        // c0 tau^2 + (c0 del - zl2 - zr2) tau - zr2 del = 0   (positive root wanted)
        const double a = zl2 + zr2 - c0 * del, b = -zr2 * del;     // c0 eta^2 - a eta + b = 0
        const double disc = sqrt(fabs(a * a - 4.0 * b * c0));
        if (c0 > 0.0) tau = (a < 0.0) ? 2.0 * b / (a - disc) : (a + disc) / (2.0 * c0);
        else tau = mid;
        if (!(tau > lo && tau <= hi)) tau = mid;
    }
    const double dorg = d[org];
    const double klog = 8.0 + 2.0 * log2((double)K);
    int it = 0, status = -1;
    const int ITMAX = 80;
    double prev_absw = HUGE_VAL;
    for (; it < ITMAX; ++it) {
        // psi: poles i <= jl (left of the root), phi: poles i >= jr;  for the last root all poles are "left"
        double psi = 0.0, dpsi = 0.0, phi = 0.0, dphi = 0.0;
        for (int i = ln; i < K; i += nl) {
            const double dl = (d[i] - dorg) - tau;
            const double t = z[i] / dl, tt = z[i] * t;     // z^2/delta
            if (last ? true : (i <= jl)) { psi += tt; dpsi += t * t; } else { phi += tt; dphi += t * t; }
        }
        psi = L.sum(psi); dpsi = L.sum(dpsi); phi = L.sum(phi); dphi = L.sum(dphi);
        const double w = rhoinv + psi + phi, dw = dpsi + dphi;
        const double erretm = klog * (phi - psi) + 2.0 * rhoinv + fabs(tau) * dw;
        if (fabs(w) <= DC_EPS * erretm) { status = it; break; }
        if (w <= 0.0) lo = fmax(lo, tau); else hi = fmin(hi, tau);
        if (!(hi - lo > 2.0 * DC_EPS * fmax(fabs(lo), fabs(hi)))) { status = it; break; }   // bracket exhausted
        double eta;
        const bool bisect = (it >= 20) || (it >= 4 && fabs(w) > 0.5 * prev_absw && (it & 1));
        prev_absw = fabs(w);
        if (bisect) {
            eta = 0.5 * (lo + hi) - tau;
        } else if (last) {
            // one-sided: all poles left; fit psi(x) ~ s + a/(Dr - x) at the nearest pole (delta of pole K-1)
            const double Dr = (d[K - 1] - dorg) - tau;          // = -tau
            const double Dl = (d[K - 2] - dorg) - tau;
            // two-pole fit: poles K-2 (with everything left of it) and K-1
            const double zr = z[K - 1] / Dr, tr = z[K - 1] * zr;          // exact nearest-pole term
            const double psi_l = psi - tr, dpsi_l = dpsi - zr * zr;
            const double c = w - Dl * dpsi_l - Dr * (zr * zr);
            const double a = (Dl + Dr) * w - Dl * Dr * dw;
            const double b = Dl * Dr * w;
            (void)psi_l;
            if (c == 0.0) eta = b / a;
            else {
                const double disc = sqrt(fabs(a * a - 4.0 * b * c));
                eta = (a >= 0.0) ? (a + disc) / (2.0 * c) : 2.0 * b / (a - disc);
            }
            if (w * eta >= 0.0) eta = -w / dw;
        } else {
            const double Dl = (d[jl] - dorg) - tau, Dr = (d[jr] - dorg) - tau;
            const double c = w - Dl * dpsi - Dr * dphi;
            const double a = (Dl + Dr) * w - Dl * Dr * dw;
            const double b = Dl * Dr * w;
            if (c == 0.0) eta = b / a;
            else {
                const double disc = sqrt(fabs(a * a - 4.0 * b * c));
                eta = (a <= 0.0) ? (a - disc) / (2.0 * c) : 2.0 * b / (a + disc);
            }
            if (w * eta >= 0.0) eta = -w / dw;       // f is increasing: the step must oppose the sign of f
        }
        double tnew = tau + eta;
        if (!(tnew > lo && tnew < hi)) tnew = 0.5 * (lo + hi);
        tau = tnew;
    }
    for (int i = ln; i < K; i += nl) delta[i] = (d[i] - dorg) - tau;
    *lambda = dorg + tau;
    return status;
}

// ---------------------------------------------------------------------------------------------------------------
// Deflation scan (sequential; one thread per merge).  Inputs in SORTED order: ds[j], zs[j] (z already scaled by
// 1/sqrt(2) and sign-fixed), src[j] = index (0..N-1) of the column the j-th sorted entry belongs to.
// State is carried across calls so that the caller can stage the inputs through shared memory in chunks.
// Outputs (global arrays of length N):
//   dlam[0..K), wz[0..K)      poles and weights of the secular problem, poles ascending
//   indxp[0..K)               column of the j-th secular pole;  indxp[K..N) columns of the deflated values, whose d
//                             are DESCENDING with position
//   coltyp[col]               1 top-only, 2 dense, 3 bottom-only, 4 deflated
//   dcol[col]                 updated d of a column (changes only through rotations)
//   rot_*[0..nrot)            Givens rotations to apply, in order, to columns (rot_p, rot_q) of Q:
//                             [x y] <- [c x + s y, c y - s x]
// ---------------------------------------------------------------------------------------------------------------
struct DeflateState {
    int K, K2, pj, nrot;
    double d_pj, z_pj, tol, rho;
    int typ_pj;
};

NAO_HD void deflate_init(DeflateState &s, int N, double rho, double tol) {
    s.K = 0; s.K2 = N; s.pj = -1; s.nrot = 0; s.d_pj = 0.0; s.z_pj = 0.0; s.tol = tol; s.rho = rho; s.typ_pj = 0;
}

NAO_HD void deflate_range(DeflateState &s, int N, int n1, int jb, int je, const double *ds, const double *zs,
                          const int *src, double *dlam, double *wz, int *indxp, int *coltyp, double *dcol,
                          int *rot_p, int *rot_q, double *rot_c, double *rot_s) {
    for (int j = jb; j < je; ++j) {
        const int nj = src[j - jb];
        const double dj = ds[j - jb], zj = zs[j - jb];
        const int typ_nj = nj < n1 ? 1 : 3;
        if (s.rho * fabs(zj) <= s.tol) {           // negligible weight: deflate
            s.K2--; coltyp[nj] = 4; indxp[s.K2] = nj; dcol[nj] = dj;
            continue;
        }
        if (s.pj < 0) { s.pj = nj; s.d_pj = dj; s.z_pj = zj; s.typ_pj = typ_nj; continue; }
        // try to rotate z_pj into z_nj
        double sn = s.z_pj, cs = zj;
        const double tau = hypot(cs, sn);
        const double t = dj - s.d_pj;
        cs /= tau; sn = -sn / tau;
        if (fabs(t * cs * sn) <= s.tol) {
            // deflate pj; nj carries the combined weight
            const double znew = tau;
            int typ_new = typ_nj;
            if (typ_nj != s.typ_pj) typ_new = 2;
            coltyp[s.pj] = 4;
            rot_p[s.nrot] = s.pj; rot_q[s.nrot] = nj; rot_c[s.nrot] = cs; rot_s[s.nrot] = sn; s.nrot++;
            const double dp = s.d_pj * cs * cs + dj * sn * sn;
            const double dn = s.d_pj * sn * sn + dj * cs * cs;
            dcol[s.pj] = dp;
            s.K2--;
            // insert pj among the deflated so that their d stay descending with position
            int pos = s.K2;
            while (pos + 1 < N && dp < dcol[indxp[pos + 1]]) { indxp[pos] = indxp[pos + 1]; ++pos; }
            indxp[pos] = s.pj;
            s.pj = nj; s.d_pj = dn; s.z_pj = znew; s.typ_pj = typ_new;
        } else {
            dlam[s.K] = s.d_pj; wz[s.K] = s.z_pj; indxp[s.K] = s.pj; coltyp[s.pj] = s.typ_pj; dcol[s.pj] = s.d_pj;
            s.K++;
            s.pj = nj; s.d_pj = dj; s.z_pj = zj; s.typ_pj = typ_nj;
        }
    }
}

NAO_HD void deflate_finish(DeflateState &s, double *dlam, double *wz, int *indxp, int *coltyp, double *dcol) {
    if (s.pj >= 0) {
        dlam[s.K] = s.d_pj; wz[s.K] = s.z_pj; indxp[s.K] = s.pj; coltyp[s.pj] = s.typ_pj; dcol[s.pj] = s.d_pj;
        s.K++;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Implicit QL on a small symmetric tridiagonal (leaf solver), split into the scalar recurrence (one lane) that
// emits plane rotations and their application to the rows of Z (all lanes).  tql2-style; d[0..m), e[0..m-1]
// (e[i] couples i and i+1; e[m-1] is scratch).  `emit(i, c, s)` must apply, to every row k of Z:
//      f = Z[k][i+1];  Z[k][i+1] = s Z[k][i] + c f;  Z[k][i] = c Z[k][i] - s f.
// Returns 0, or l+1 if eigenvalue l failed to converge in 60 sweeps.
// ---------------------------------------------------------------------------------------------------------------
template <class Emit> NAO_HD int ql_implicit(int m, double *d, double *e, Emit &emit) {
    if (m > 0) e[m - 1] = 0.0;
    for (int l = 0; l < m; ++l) {
        int iter = 0, mm;
        do {
            for (mm = l; mm < m - 1; ++mm) {
                const double dd = fabs(d[mm]) + fabs(d[mm + 1]);
                if (fabs(e[mm]) <= DC_EPS * dd) break;
            }
            if (mm != l) {
                if (iter++ == 60) return l + 1;
                double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                double r = hypot(g, 1.0);
                g = d[mm] - d[l] + e[l] / (g + (g >= 0.0 ? fabs(r) : -fabs(r)));
                double s = 1.0, c = 1.0, p = 0.0;
                int i;
                for (i = mm - 1; i >= l; --i) {
                    double f = s * e[i];
                    const double b = c * e[i];
                    e[i + 1] = (r = hypot(f, g));
                    if (r == 0.0) { d[i + 1] -= p; e[mm] = 0.0; break; }
                    s = f / r; c = g / r;
                    g = d[i + 1] - p;
                    r = (d[i] - g) * s + 2.0 * c * b;
                    p = s * r;
                    d[i + 1] = g + p;
                    g = c * r - b;
                    emit(i, c, s);
                }
                if (r == 0.0 && i >= l) continue;
                d[l] -= p; e[l] = g; e[mm] = 0.0;
            }
        } while (mm != l);
    }
    return 0;
}

}  // namespace dc
}  // namespace nao
