/*
 * nao_synth.c -- seeded synthetic NAO-shaped H and S matrices (input generator).
 *
 * This module serves BOTH the CPU oracle and the CUDA path as their common source
 * of inputs.  It contains none of the method's arithmetic (no factorisation, no
 * eigen-solve, no Fermi function, no density matrix): it only writes matrices.
 *
 * Recipe: BASELINE.json "configs" / DESIGN.md section "Input recipe".
 *   - atoms uniform in a cubic box of side L (bohr); 13 orbitals per atom in the
 *     order s,s,p*3,p*3,d*5  (s2 p2 d1; paper: 13 basis functions per Si atom,
 *     PAPER.md:224, section 4).
 *   - pair terms within a 10 bohr cut-off:  S_ij = exp(-d^2/12.5) * u,
 *     H_ij = -0.3 exp(-d/3) * v,  u,v ~ U[-1,1] drawn per unordered (pair,image).
 *   - S made SPD by diagonal dominance: d_i = 1 + sum |S_ij(R)|, then
 *     S(R) <- S(R) / sqrt(d_i d_j)  (unit diagonal).
 *   - periodic cells: images R in {-1,0,1}^3, Bloch sum
 *     M_ij(k) = sum_R exp(+i k.R) M_ij(R)   (Eq. 12).
 * Every random number is a pure function of (seed, stream tag, canonical index
 * tuple) through a counter-based 64-bit mix hash, so the result does not depend
 * on thread count or evaluation order.
 *
 * All matrices are written COLUMN-MAJOR: element (i,j) at [j*n + i]; complex
 * matrices interleaved (re,im).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#define NORB 13
#define CUTOFF 10.0

enum { TAG_POS = 1, TAG_ONSITE = 2, TAG_S = 3, TAG_H = 4, TAG_MOM = 5, TAG_AX = 6, TAG_AY = 7, TAG_AZ = 8 };

static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static inline uint64_t key4(uint64_t seed, uint64_t tag, uint64_t a, uint64_t b, uint64_t c) {
    uint64_t h = mix64(seed * 0x2545F4914F6CDD1DULL + tag);
    h = mix64(h ^ (a + 0x1000000ULL));
    h = mix64(h ^ (b + 0x2000000ULL));
    h = mix64(h ^ (c + 0x3000000ULL));
    return h;
}
static inline double u01(uint64_t h) { return (double)(h >> 11) * (1.0 / 9007199254740992.0); }
static inline double usym(uint64_t h) { return 2.0 * u01(h) - 1.0; }
/* standard normal by Box-Muller from two hashed uniforms */
static double gauss(uint64_t seed, uint64_t tag, uint64_t a, uint64_t b) {
    double u1 = u01(key4(seed, tag, a, b, 0));
    double u2 = u01(key4(seed, tag, a, b, 1));
    if (u1 < 1e-300) u1 = 1e-300;
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* orbital type within an atom: 0 = s, 1 = p, 2 = d */
static inline int orb_type(int o) { return o < 2 ? 0 : (o < 8 ? 1 : 2); }
static const double ONSITE_E[3] = { -0.5, -0.2, 0.0 };

int nao_synth_norb(void) { return NORB; }

/* positions: pos[3*nat], uniform in [0,L)^3 */
void nao_synth_positions(uint64_t seed, int nat, double L, double *pos) {
    for (int a = 0; a < nat; ++a)
        for (int c = 0; c < 3; ++c)
            pos[3 * a + c] = L * u01(key4(seed, TAG_POS, (uint64_t)a, (uint64_t)c, 0));
}

/* canonical unordered key for the pair (i, j, R) == (j, i, -R); rc = image code 0..26 (13 = home cell) */
static inline void canon(int i, int j, int rc, uint64_t *a, uint64_t *b, uint64_t *c) {
    if (i > j || (i == j && rc > 13)) { int t = i; i = j; j = t; rc = 26 - rc; }
    *a = (uint64_t)i; *b = (uint64_t)j; *c = (uint64_t)rc;
}
static inline double raw_S(uint64_t seed, int i, int j, int rc, double d) {
    uint64_t a, b, c; canon(i, j, rc, &a, &b, &c);
    return exp(-d * d / 12.5) * usym(key4(seed, TAG_S, a, b, c));
}
static inline double raw_H(uint64_t seed, int i, int j, int rc, double d) {
    uint64_t a, b, c; canon(i, j, rc, &a, &b, &c);
    return -0.3 * exp(-d / 3.0) * usym(key4(seed, TAG_H, a, b, c));
}

/* distance between atom a (home cell) and atom b displaced by image rc; returns -1 if beyond cut-off */
static inline double pair_dist(const double *pos, double L, int a, int b, int rc, int periodic) {
    int rx = rc / 9 - 1, ry = (rc / 3) % 3 - 1, rz = rc % 3 - 1;
    if (!periodic && rc != 13) return -1.0;
    double dx = pos[3 * b] + rx * L - pos[3 * a];
    double dy = pos[3 * b + 1] + ry * L - pos[3 * a + 1];
    double dz = pos[3 * b + 2] + rz * L - pos[3 * a + 2];
    double d2 = dx * dx + dy * dy + dz * dz;
    if (d2 > CUTOFF * CUTOFF) return -1.0;
    return sqrt(d2);
}

/* diagonal-dominance scale d_i = 1 + sum_{(j,R) != (i,0)} |S_ij(R)| */
static void row_scales(uint64_t seed, int nat, double L, int periodic, const double *pos, double *dsc) {
    int n = nat * NORB;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int a = 0; a < nat; ++a) {
        double acc[NORB];
        for (int o = 0; o < NORB; ++o) acc[o] = 1.0;
        for (int b = 0; b < nat; ++b)
            for (int rc = 0; rc < 27; ++rc) {
                double d = pair_dist(pos, L, a, b, rc, periodic);
                if (d < 0) continue;
                for (int o = 0; o < NORB; ++o)
                    for (int q = 0; q < NORB; ++q) {
                        int i = a * NORB + o, j = b * NORB + q;
                        if (i == j && rc == 13) continue;
                        acc[o] += fabs(raw_S(seed, i, j, rc, d));
                    }
            }
        for (int o = 0; o < NORB; ++o) dsc[a * NORB + o] = acc[o];
    }
    (void)n;
}

/*
 * Bloch-summed H(k), S(k) for one k-point (fractional kfrac[3]; phase = 2*pi*kfrac.R).
 * is_complex = 0: kfrac must be 0 and Hout/Sout are real n*n; otherwise complex interleaved.
 * d_shift is added to the diagonal of H on d orbitals (collinear spin splitting).
 * Column-major output.
 */
void nao_synth_hs(uint64_t seed, int nat, double L, int periodic, const double *kfrac, int is_complex,
                  double d_shift, double *Hout, double *Sout) {
    int n = nat * NORB;
    double *pos = (double *)malloc(sizeof(double) * 3 * nat);
    double *dsc = (double *)malloc(sizeof(double) * n);
    nao_synth_positions(seed, nat, L, pos);
    row_scales(seed, nat, L, periodic, pos, dsc);
    size_t es = is_complex ? 2 : 1;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int b = 0; b < nat; ++b) {           /* column atom (orbital j lives on atom b's image) */
        for (int a = 0; a < nat; ++a) {
            double hs[NORB][NORB][2], ss[NORB][NORB][2];
            memset(hs, 0, sizeof hs); memset(ss, 0, sizeof ss);
            for (int rc = 0; rc < 27; ++rc) {
                double d = pair_dist(pos, L, a, b, rc, periodic);
                if (d < 0) continue;
                int rx = rc / 9 - 1, ry = (rc / 3) % 3 - 1, rz = rc % 3 - 1;
                double ph = 6.283185307179586476925286766559 * (kfrac[0] * rx + kfrac[1] * ry + kfrac[2] * rz);
                double cr = is_complex ? cos(ph) : 1.0, ci = is_complex ? sin(ph) : 0.0;
                if (rc == 13) { cr = 1.0; ci = 0.0; }
                for (int o = 0; o < NORB; ++o)
                    for (int q = 0; q < NORB; ++q) {
                        int i = a * NORB + o, j = b * NORB + q;
                        double sv, hv;
                        if (i == j && rc == 13) {
                            sv = 1.0;
                            hv = ONSITE_E[orb_type(o)] + 0.05 * gauss(seed, TAG_ONSITE, (uint64_t)i, 0)
                                 + (orb_type(o) == 2 ? d_shift : 0.0);
                        } else {
                            sv = raw_S(seed, i, j, rc, d) / sqrt(dsc[i] * dsc[j]);
                            hv = raw_H(seed, i, j, rc, d);
                        }
                        ss[o][q][0] += sv * cr; ss[o][q][1] += sv * ci;
                        hs[o][q][0] += hv * cr; hs[o][q][1] += hv * ci;
                    }
            }
            for (int o = 0; o < NORB; ++o)
                for (int q = 0; q < NORB; ++q) {
                    size_t i = (size_t)a * NORB + o, j = (size_t)b * NORB + q;
                    size_t off = (j * (size_t)n + i) * es;
                    Hout[off] = hs[o][q][0]; Sout[off] = ss[o][q][0];
                    if (is_complex) { Hout[off + 1] = hs[o][q][1]; Sout[off + 1] = ss[o][q][1]; }
                }
        }
    }
    free(pos); free(dsc);
}

/*
 * Noncollinear Hamiltonian (spin-major basis [alpha; beta], Eq. 21, 175-179 Eq. 25-27):
 *   H_NC = [H0 + J m_z + i lam A_z ,  J(m_x - i m_y) + i lam A_x + lam A_y ;  h.c. , H0 - J m_z - i lam A_z]
 * H0, S real N*N Gamma-point matrices of the same recipe; J m on the orbital diagonal of each atom with that
 * atom's random unit vector m; A_x,A_y,A_z real antisymmetric, non-zero only between p/d orbitals of one atom.
 * Hnc: complex (2N)*(2N) column-major interleaved; S: real N*N column-major.
 */
void nao_synth_nc(uint64_t seed, int nat, double L, int periodic, double J, double lam, double *Hnc, double *S) {
    int N = nat * NORB;
    size_t n2 = 2 * (size_t)N;
    double kz[3] = { 0, 0, 0 };
    double *H0 = (double *)malloc(sizeof(double) * (size_t)N * N);
    nao_synth_hs(seed, nat, L, periodic, kz, 0, 0.0, H0, S);
    #pragma omp parallel for schedule(static)
    for (int j = 0; j < N; ++j)
        for (int i = 0; i < N; ++i) {
            double h = H0[(size_t)j * N + i];
            size_t aa = ((size_t)j * n2 + i) * 2, bb = (((size_t)j + N) * n2 + (i + N)) * 2;
            size_t ab = (((size_t)j + N) * n2 + i) * 2, ba = ((size_t)j * n2 + (i + N)) * 2;
            Hnc[aa] = h; Hnc[aa + 1] = 0; Hnc[bb] = h; Hnc[bb + 1] = 0;
            Hnc[ab] = 0; Hnc[ab + 1] = 0; Hnc[ba] = 0; Hnc[ba + 1] = 0;
        }
    free(H0);
    for (int a = 0; a < nat; ++a) {
        double m[3], nrm = 0;
        for (int c = 0; c < 3; ++c) { m[c] = gauss(seed, TAG_MOM, (uint64_t)a, (uint64_t)c); nrm += m[c] * m[c]; }
        nrm = sqrt(nrm);
        for (int c = 0; c < 3; ++c) m[c] /= nrm;
        for (int o = 0; o < NORB; ++o) {
            size_t i = (size_t)a * NORB + o;
            Hnc[(i * n2 + i) * 2] += J * m[2];
            Hnc[((i + N) * n2 + (i + N)) * 2] -= J * m[2];
            /* alpha-beta block element (i, i+N) = J (m_x - i m_y); beta-alpha = conjugate */
            Hnc[((i + N) * n2 + i) * 2] += J * m[0]; Hnc[((i + N) * n2 + i) * 2 + 1] += -J * m[1];
            Hnc[(i * n2 + (i + N)) * 2] += J * m[0]; Hnc[(i * n2 + (i + N)) * 2 + 1] += J * m[1];
        }
        for (int o = 2; o < NORB; ++o)
            for (int q = o + 1; q < NORB; ++q) {
                size_t i = (size_t)a * NORB + o, j = (size_t)a * NORB + q;
                double ax = usym(key4(seed, TAG_AX, i, j, 0));
                double ay = usym(key4(seed, TAG_AY, i, j, 0));
                double az = usym(key4(seed, TAG_AZ, i, j, 0));
                /* A(i,j) = +a, A(j,i) = -a */
                /* alpha-alpha: + i lam A_z ; beta-beta: - i lam A_z */
                Hnc[(j * n2 + i) * 2 + 1] += lam * az;            Hnc[(i * n2 + j) * 2 + 1] -= lam * az;
                Hnc[((j + N) * n2 + i + N) * 2 + 1] -= lam * az;  Hnc[((i + N) * n2 + j + N) * 2 + 1] += lam * az;
                /* alpha-beta block B = i lam A_x + lam A_y: B(i,j) = lam(ay + i ax), B(j,i) = -lam(ay + i ax) */
                Hnc[((j + N) * n2 + i) * 2] += lam * ay;  Hnc[((j + N) * n2 + i) * 2 + 1] += lam * ax;
                Hnc[((i + N) * n2 + j) * 2] -= lam * ay;  Hnc[((i + N) * n2 + j) * 2 + 1] -= lam * ax;
                /* beta-alpha block = B^H: (B^H)(j,i) = conj(B(i,j)), (B^H)(i,j) = conj(B(j,i)) */
                Hnc[(i * n2 + j + N) * 2] += lam * ay;    Hnc[(i * n2 + j + N) * 2 + 1] -= lam * ax;
                Hnc[(j * n2 + i + N) * 2] -= lam * ay;    Hnc[(j * n2 + i + N) * 2 + 1] += lam * ax;
            }
    }
}
