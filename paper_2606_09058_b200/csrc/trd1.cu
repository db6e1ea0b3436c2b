// trd1.cu -- one-stage Householder tridiagonalisation (SURVEY.md 8a row a3/a4 role, 8d ambiguity M1: this is the
// HBM-bound "BLAS2 half" the paper describes for the one-stage reduction) and the blocked
// back-transformation Z <- Q Z (row a6).
//
// Algorithm: LAPACK xHETRD/xLATRD, lower storage, panels of NB columns.  Inside a panel the trailing matrix is NOT
// updated; column j is brought up to date with the panel's (V, W), a reflector is generated, and
//   w = tau (A22 v - V (W^H v) - W (V^H v)) - 1/2 |tau|^2 (v^H A22 v - 2 Re (W^H v)^H (V^H v)) v
// is appended.  After the panel A22 -= V W^H + W V^H runs on the DMMA GEMM core.
//
// B200 design: ONE cooperative persistent kernel per panel.  The G CTAs that work on an item are co-resident and meet
// at a software grid barrier only TWICE per column:
//   phase A: finalise w of the previous column for the CTA's own rows, update column j, partial norm   | barrier
//   phase B: reflector scalars (every CTA, redundantly), v written to A, partial W^H v / V^H v,
//            HEMV over 64x64 tiles of the lower triangle (each element read from HBM exactly once per column,
//            both its row and its column contribution formed from registers), partial v^H A v          | barrier
// Every cross-CTA reduction goes through per-CTA partial buffers summed in a fixed order: results are bit-reproducible
// (no floating-point atomics).  HEMV tile loads are 512 B (real) / 1 KB (complex) contiguous per column and the
// next tile is prefetched into registers while the current one is reduced, so the kernel runs at HBM speed once the
// trailing matrix exceeds L2.
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <cooperative_groups.h>

namespace nao {

static const int TRD_NB = 32;        // panel width
static const int TRD_NT = 512;       // threads per CTA
static const int TRD_TB = 64;        // HEMV tile edge

template <class T> struct TrdArgs {
    T *A; long lda, sA;
    double *d, *e; T *tau;           // per item: n each
    T *Wp;                           // per item: n x NB (ld n)
    T *acol;                         // per item: n
    double *pn;                      // per item: G
    T *pt;                           // per item: G x 2NB
    double *pvav;                    // per item: G
    T *Prow, *Pcol;                  // per item: nblk x n each
    unsigned *bar;                   // per item: one counter for this launch
    int n, j0, nbp, G, nblk;
};

template <class T> __device__ __forceinline__ T block_sum_T(T v, T *red /* TRD_NT/32 */) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    T s = Ops<T>::zero();
    for (int w = 0; w < TRD_NT / 32; ++w) s = Ops<T>::add(s, red[w]);
    __syncthreads();
    return s;
}
__device__ __forceinline__ double block_sum_d(double v, double *red) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < TRD_NT / 32; ++w) s += red[w];
    __syncthreads();
    return s;
}

template <class T>
__global__ void __launch_bounds__(TRD_NT, 1) hetrd_panel_kernel(TrdArgs<T> p) {
    typedef Ops<T> O;
    const int G = p.G;
    const int item = blockIdx.x / G, g = blockIdx.x % G;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = p.n, j0 = p.j0, nblk = p.nblk;
    const long lda = p.lda;
    T *A = p.A + (long)item * p.sA;
    double *dd = p.d + (long)item * n, *ee = p.e + (long)item * n;
    T *tauv = p.tau + (long)item * n;
    T *Wp = p.Wp + (long)item * n * TRD_NB;
    T *acol = p.acol + (long)item * n;
    double *pn = p.pn + (long)item * G;
    T *pt = p.pt + (long)item * G * 2 * TRD_NB;
    double *pvav = p.pvav + (long)item * G;
    T *Prow = p.Prow + (long)item * nblk * n, *Pcol = p.Pcol + (long)item * nblk * n;
    unsigned *bar = p.bar + item;
    unsigned bar_ord = 0;

    const int m = n - j0;
    const int chunk = (m + G - 1) / G;
    const int r0 = j0 + g * chunk, r1 = min(n, r0 + chunk);     // rows owned by this CTA

    __shared__ T s_t[2 * TRD_NB];          // t1 = W^H v at [0,NB), t2 = V^H v at [NB,2NB)
    __shared__ T s_wrow[TRD_NB], s_vrow[TRD_NB];
    __shared__ T s_tau, s_scale;
    __shared__ double s_alpha, s_dred[TRD_NT / 32];
    __shared__ T s_red[TRD_NT / 32];
    __shared__ T xs_row[TRD_TB], xs_col[TRD_TB];
    __shared__ T red_row[8][TRD_TB];
    __shared__ T red_col[TRD_NT / 32][8];
    __shared__ T s_wpart[TRD_NT / 32][2 * TRD_NB];

    for (int i = 0; i <= p.nbp; ++i) {
        const int j = j0 + i;
        // =============================== phase A ===============================
        if (i > 0) {
            // reduce the partials of phase B(i-1): t1, t2 (k < i-1) and v^H A v
            const int nk = i - 1;
            if (tid < 2 * TRD_NB) {
                T s = O::zero();
                int k = tid < TRD_NB ? tid : tid - TRD_NB;
                if (k < nk)
                    for (int q = 0; q < G; ++q) s = O::add(s, ldcg(pt + (long)q * 2 * TRD_NB + tid));
                s_t[tid] = s;
            }
            if (warp == 4) {
                double s = 0.0;
                for (int q = lane; q < G; q += 32) s += ldcg(pvav + q);
                s = warp_sum(s);
                if (lane == 0) s_dred[0] = s;
            }
            __syncthreads();
            if (tid == 0) {
                double s = s_dred[0];
                for (int k = 0; k < nk; ++k) s -= 2.0 * O::real(O::conj_mul(s_t[k], s_t[TRD_NB + k]));
                s_alpha = -0.5 * O::abs2(s_tau) * s;
            }
            __syncthreads();
        }
        // w_{i-1}(r) for a row r >= j, from the tile partials of phase B(i-1)
        auto wfinal = [&](int r, bool own) -> T {
            const int jm1 = j - 1, nk = i - 1;
            const int bmin = (jm1 + 1) / TRD_TB, br = r / TRD_TB;
            T acc = O::zero();
            for (int J = bmin; J <= br; ++J) acc = O::add(acc, ldcg(Prow + (long)J * n + r));
            for (int I = br; I < nblk; ++I) acc = O::add(acc, ldcg(Pcol + (long)I * n + r));
            for (int k = 0; k < nk; ++k) {
                T v = own ? A[r + (long)(j0 + k) * lda] : ldcg(A + r + (long)(j0 + k) * lda);
                T w = own ? Wp[r + (long)k * n] : ldcg(Wp + r + (long)k * n);
                acc = O::sub(acc, O::add(O::mul(v, s_t[k]), O::mul(w, s_t[TRD_NB + k])));
            }
            T vr = (r == j) ? O::one() : (own ? A[r + (long)jm1 * lda] : ldcg(A + r + (long)jm1 * lda));
            return O::add(O::mul(s_tau, acc), O::scale(vr, s_alpha));
        };
        if (i > 0) {
            if (tid == 0) s_wrow[i - 1] = wfinal(j, false);
            for (int r = max(r0, j) + tid; r < r1; r += TRD_NT) Wp[r + (long)(i - 1) * n] = wfinal(r, true);
        }
        const bool do_col = (i < p.nbp) || (j == n - 1);
        if (do_col) {
            if (tid < i) {
                s_vrow[tid] = ldcg(A + j + (long)(j0 + tid) * lda);
                if (tid < i - 1) s_wrow[tid] = ldcg(Wp + j + (long)tid * n);
            }
        }
        __syncthreads();
        if (do_col) {
            double nrm = 0.0;
            for (int r = max(r0, j) + tid; r < r1; r += TRD_NT) {
                T a = A[r + (long)j * lda];
                if (r == j) a = O::from_real(O::real(a));
                for (int k = 0; k < i; ++k) {
                    T v = A[r + (long)(j0 + k) * lda], w = Wp[r + (long)k * n];
                    a = O::sub(a, O::add(O::mul_conj(v, s_wrow[k]), O::mul_conj(w, s_vrow[k])));
                }
                if (r == j) dd[j] = O::real(a);
                else { acol[r] = a; if (r >= j + 2) nrm += O::abs2(a); }
            }
            nrm = block_sum_d(nrm, s_dred);
            if (tid == 0) pn[g] = nrm;
        }
        if (i == p.nbp) break;
        group_barrier(bar, G, ++bar_ord);

        // =============================== phase B ===============================
        if (warp == 0) {
            double s = 0.0;
            for (int q = lane; q < G; q += 32) s += ldcg(pn + q);
            s = warp_sum(s);
            if (lane == 0) {
                T alpha0 = ldcg(acol + j + 1);
                double ar = O::real(alpha0), ai = O::imag(alpha0);
                T tau, scale; double beta;
                if (s == 0.0 && ai == 0.0) { tau = O::zero(); scale = O::zero(); beta = ar; }
                else {
                    double nrm = sqrt(ar * ar + ai * ai + s);
                    beta = ar >= 0.0 ? -nrm : nrm;
                    if (O::is_complex) {
                        cplx t = make_double2((beta - ar) / beta, -ai / beta);
                        double dr = ar - beta, di = ai, den = dr * dr + di * di;     // 1/(alpha0 - beta)
                        cplx sc = make_double2(dr / den, -di / den);
                        tau = *(T *)&t; scale = *(T *)&sc;
                    } else {
                        tau = O::from_real((beta - ar) / beta); scale = O::from_real(1.0 / (ar - beta));
                    }
                }
                s_tau = tau; s_scale = scale;
                if (g == 0) { ee[j] = beta; tauv[j] = tau; }
            }
        }
        __syncthreads();
        const T scale = s_scale;
        auto vval = [&](int x) -> T {
            if (x < j + 1 || x >= n) return O::zero();
            if (x == j + 1) return O::one();
            return O::mul(ldcg(acol + x), scale);
        };
        // v into column j of A (own rows), and partial t1 = W^H v, t2 = V^H v over own rows
        {
            const int rb = max(r0, j + 1);
            for (int k = tid; k < 2 * TRD_NB * (TRD_NT / 32); k += TRD_NT) (&s_wpart[0][0])[k] = O::zero();
            __syncthreads();
            for (int base = rb + warp * 32; base < r1; base += TRD_NT) {
                int r = base + lane;
                T v = O::zero();
                if (r < r1) { v = vval(r); A[r + (long)j * lda] = v; }
                for (int k = 0; k < i; ++k) {
                    T w = r < r1 ? Wp[r + (long)k * n] : O::zero();
                    T a = r < r1 ? A[r + (long)(j0 + k) * lda] : O::zero();
                    T p1 = warp_sum(O::conj_mul(w, v)), p2 = warp_sum(O::conj_mul(a, v));
                    if (lane == 0) {
                        s_wpart[warp][k] = O::add(s_wpart[warp][k], p1);
                        s_wpart[warp][TRD_NB + k] = O::add(s_wpart[warp][TRD_NB + k], p2);
                    }
                }
            }
            __syncthreads();
            if (tid < 2 * TRD_NB) {
                T s = O::zero();
                for (int w = 0; w < TRD_NT / 32; ++w) s = O::add(s, s_wpart[w][tid]);
                pt[(long)g * 2 * TRD_NB + tid] = s;
            }
        }
        // HEMV over the 64x64 tiles (I >= J >= bmin) of the lower triangle of A[j+1:, j+1:]
        double vav = 0.0;
        {
            const int bmin = (j + 1) / TRD_TB, nbk = nblk - bmin, ntiles = nbk * (nbk + 1) / 2;
            const int r = tid & 63, cg = tid >> 6;
            auto decode = [&](int t, int &I, int &J) {
                int ii = (int)((sqrt(8.0 * (double)t + 1.0) - 1.0) * 0.5);
                while ((ii + 1) * (ii + 2) / 2 <= t) ++ii;
                while (ii * (ii + 1) / 2 > t) --ii;
                I = bmin + ii; J = bmin + (t - ii * (ii + 1) / 2);
            };
            auto load = [&](T a[8], int t) {
                int I, J; decode(t, I, J);
                const int gr = I * TRD_TB + r;
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const int gc = J * TRD_TB + cg * 8 + q;
                    T v = O::zero();
                    if (gr < n && gc >= j + 1 && gr >= gc) {
                        v = A[gr + (long)gc * lda];
                        if (gr == gc) v = O::from_real(O::real(v));
                    }
                    a[q] = v;
                }
            };
            T cur[8], nxt[8];
            int t = g;
            if (t < ntiles) load(cur, t);
            while (t < ntiles) {
                const int tn = t + G;
                if (tn < ntiles) load(nxt, tn);
                int I, J; decode(t, I, J);
                if (tid < TRD_TB) xs_col[tid] = vval(J * TRD_TB + tid);
                else if (tid < 2 * TRD_TB) xs_row[tid - TRD_TB] = vval(I * TRD_TB + tid - TRD_TB);
                __syncthreads();
                const T xr = xs_row[r];
                T rs = O::zero();
                T cs[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const int c = cg * 8 + q;
                    rs = O::fma(cur[q], xs_col[c], rs);
                    const bool strict = (I > J) || (r > c);
                    cs[q] = strict ? O::conj_mul(cur[q], xr) : O::zero();
                }
                red_row[cg][r] = rs;
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    T s = warp_sum(cs[q]);
                    if (lane == 0) red_col[warp][q] = s;
                }
                __syncthreads();
                if (tid < TRD_TB) {
                    T s = O::zero();
#pragma unroll
                    for (int q = 0; q < 8; ++q) s = O::add(s, red_row[q][tid]);
                    const int gr = I * TRD_TB + tid;
                    if (gr < n) Prow[(long)J * n + gr] = s;
                    vav += O::real(O::conj_mul(xs_row[tid], s));
                } else if (tid < 2 * TRD_TB) {
                    const int c = tid - TRD_TB, cg2 = c >> 3, q = c & 7;
                    T s = O::add(red_col[2 * cg2][q], red_col[2 * cg2 + 1][q]);
                    const int gc = J * TRD_TB + c;
                    if (gc < n) Pcol[(long)I * n + gc] = s;
                    vav += O::real(O::conj_mul(xs_col[c], s));
                }
                __syncthreads();
#pragma unroll
                for (int q = 0; q < 8; ++q) cur[q] = nxt[q];
                t = tn;
            }
        }
        vav = block_sum_d(vav, s_dred);
        if (tid == 0) pvav[g] = vav;
        group_barrier(bar, G, ++bar_ord);
    }
}

// workspace layout per call (all items)
struct TrdWork {
    void *Wp, *acol, *pt, *Prow, *Pcol; double *pn, *pvav; unsigned *bar; int G, nblk, items_per_launch; size_t bytes;
};
static int trd_G(int n, int batch, int nsm) {
    int per = nsm / (batch < nsm ? batch : nsm);
    if (per < 1) per = 1;
    int want = ceil_div(n, 64);
    return per < want ? per : want;
}
static int num_sms() {
    static int nsm = 0;
    if (!nsm) {
        int dev = 0; cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) nsm = 148;
    }
    return nsm;
}
static TrdWork trd_plan(int dtype, int n, int batch, void *work) {
    TrdWork w;
    const size_t es = esize(dtype);
    const int nsm = num_sms();
    w.G = trd_G(n, batch, nsm);
    w.nblk = ceil_div(n, TRD_TB);
    w.items_per_launch = batch < nsm ? batch : nsm;
    const int npanels = ceil_div(n, TRD_NB) + 1;
    Arena ar(work, (size_t)-1);
    w.Wp = ar.take((size_t)batch * n * TRD_NB * es);
    w.acol = ar.take((size_t)batch * n * es);
    w.pt = ar.take((size_t)batch * w.G * 2 * TRD_NB * es);
    w.Prow = ar.take((size_t)batch * w.nblk * n * es);
    w.Pcol = ar.take((size_t)batch * w.nblk * n * es);
    w.pn = (double *)ar.take((size_t)batch * w.G * 8);
    w.pvav = (double *)ar.take((size_t)batch * w.G * 8);
    w.bar = (unsigned *)ar.take((size_t)batch * npanels * 4);
    w.bytes = ar.off;
    return w;
}
size_t hetrd_workspace(int dtype, int n, int batch) { return trd_plan(dtype, n, batch, nullptr).bytes; }

template <class T>
static int hetrd_impl(int dtype, int n, int batch, T *A, long lda, long sA, double *d, double *e, T *tau, void *work,
                      cudaStream_t st) {
    TrdWork w = trd_plan(dtype, n, batch, work);
    const int npanels = ceil_div(n, TRD_NB) + 1;
    NAO_CUDA_CHECK(cudaMemsetAsync(w.bar, 0, (size_t)batch * npanels * 4, st));
    int panel = 0;
    for (int j0 = 0; j0 == 0 || j0 < n - 1; j0 += TRD_NB, ++panel) {
        const int nbp = max(0, min(TRD_NB, n - 1 - j0));
        for (int b0 = 0; b0 < batch; b0 += w.items_per_launch) {
            const int nb_items = min(w.items_per_launch, batch - b0);
            TrdArgs<T> a;
            a.A = A + (long)b0 * sA; a.lda = lda; a.sA = sA;
            a.d = d + (long)b0 * n; a.e = e + (long)b0 * n; a.tau = tau + (long)b0 * n;
            a.Wp = (T *)w.Wp + (long)b0 * n * TRD_NB; a.acol = (T *)w.acol + (long)b0 * n;
            a.pn = w.pn + (long)b0 * w.G; a.pt = (T *)w.pt + (long)b0 * w.G * 2 * TRD_NB; a.pvav = w.pvav + (long)b0 * w.G;
            a.Prow = (T *)w.Prow + (long)b0 * w.nblk * n; a.Pcol = (T *)w.Pcol + (long)b0 * w.nblk * n;
            a.bar = w.bar + (size_t)panel * batch + b0;
            a.n = n; a.j0 = j0; a.nbp = nbp; a.G = w.G; a.nblk = w.nblk;
            // algorithmic bytes of this launch: the lower triangle of the trailing matrix once per column
            double bytes = 0.0;
            for (int i = 0; i < nbp; ++i) { double mm = n - (j0 + i) - 1; bytes += 0.5 * mm * (mm + 1) * sizeof(T); }
            const int pk = prof_kernel_begin(0, bytes * nb_items, st);
            void *args[] = {&a};
            NAO_CUDA_CHECK(cudaLaunchCooperativeKernel((void *)hetrd_panel_kernel<T>, dim3(nb_items * w.G), dim3(TRD_NT), args, 0, st));
            NAO_LAUNCHED();
            prof_kernel_end(0, pk, st);
        }
        const int jn = j0 + nbp;             // first row/column of the trailing matrix
        if (nbp > 0 && jn < n) {
            const int mt = n - jn;
            GemmDesc g1 = gemm_desc(OP_N, OP_C, mt, mt, nbp, -1.0, A + jn + (long)j0 * lda, lda, (T *)w.Wp + jn, n, 1.0,
                                    A + jn + (long)jn * lda, lda);
            g1.sA = sA; g1.sB = (long)n * TRD_NB; g1.sC = sA; g1.cmode = 1;
            if (int rc = gemm_launch(dtype, g1, batch, st)) return rc;
            GemmDesc g2 = gemm_desc(OP_N, OP_C, mt, mt, nbp, -1.0, (T *)w.Wp + jn, n, A + jn + (long)j0 * lda, lda, 1.0,
                                    A + jn + (long)jn * lda, lda);
            g2.sA = (long)n * TRD_NB; g2.sB = sA; g2.sC = sA; g2.cmode = 1;
            if (int rc = gemm_launch(dtype, g2, batch, st)) return rc;
        }
        if (n == 1) break;
    }
    return NAO_OK;
}

int hetrd(int dtype, int n, int batch, void *A, long lda, long sA, double *d, double *e, void *tau, void *work,
          cudaStream_t st) {
    return dtype == NAO_COMPLEX ? hetrd_impl<cplx>(dtype, n, batch, (cplx *)A, lda, sA, d, e, (cplx *)tau, work, st)
                                : hetrd_impl<double>(dtype, n, batch, (double *)A, lda, sA, d, e, (double *)tau, work, st);
}

// ----------------------------------------------------------------------------------------------------------------
// Back-transformation: Z <- Q Z, Q = H(0) H(1) ... H(n-2), H(j) = I - tau_j v_j v_j^H, v_j = A[j+1:, j] (unit first
// element stored explicitly by hetrd).  Blocks of KB reflectors, last block first:
//   Vb (explicit, zeros above the unit diagonal), G = Vb^H Vb, T by the xLARFT recurrence, then three GEMMs
//   X = Vb^H Z ; X <- T X ; Z -= Vb X.
// ----------------------------------------------------------------------------------------------------------------
static const int ORM_KB = 64;

template <class T>
__global__ void build_v_kernel(int n, int jb, int kb, const T *A, long lda, long sA, T *V, long ldv, long sV) {
    // V (m x kb), m = n - jb - 1, row r <-> global row jb+1+r; column k <-> reflector jb+k whose unit sits at r == k
    A += (long)blockIdx.z * sA; V += (long)blockIdx.z * sV;
    const int m = n - jb - 1;
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= m) return;
    for (int k = blockIdx.y; k < kb; k += gridDim.y) {
        T v;
        if (r < k) v = Ops<T>::zero();
        else if (r == k) v = Ops<T>::one();
        else v = A[(jb + 1 + r) + (long)(jb + k) * lda];
        V[r + (long)k * ldv] = v;
    }
}

// T (kb x kb upper) from G = V^H V and tau: T(i,i) = tau_i ; T(0:i, i) = -tau_i T(0:i,0:i) G(0:i, i)
template <class T>
__global__ void __launch_bounds__(256) larft_kernel(int kb, const T *G, long sG, const T *tau, long sTau, T *Tm, long sT) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *sT_ = (T *)smem_raw;             // kb x kb, column-major
    __shared__ T s_g[ORM_KB];
    G += (long)blockIdx.x * sG; tau += (long)blockIdx.x * sTau; Tm += (long)blockIdx.x * sT;
    const int tid = threadIdx.x;
    for (int e = tid; e < kb * kb; e += blockDim.x) sT_[e] = Ops<T>::zero();
    __syncthreads();
    for (int i = 0; i < kb; ++i) {
        const T ti = tau[i];
        if (tid < i) s_g[tid] = G[tid + (long)i * kb];
        __syncthreads();
        if (tid < i) {
            // row tid of T(0:i,0:i) times g  (T upper: columns c >= tid)
            T acc = Ops<T>::zero();
            for (int c = tid; c < i; ++c) acc = Ops<T>::fma(sT_[tid + c * kb], s_g[c], acc);
            T v = Ops<T>::mul(ti, acc);
            sT_[tid + i * kb] = Ops<T>::sub(Ops<T>::zero(), v);
        }
        if (tid == 0) sT_[i + i * kb] = ti;
        __syncthreads();
    }
    for (int e = tid; e < kb * kb; e += blockDim.x) Tm[e] = sT_[e];
}

struct OrmWork { void *V, *G, *T, *X, *X2; size_t bytes; };
static OrmWork orm_plan(int dtype, int n, int ncols, int batch, void *work) {
    OrmWork w; const size_t es = esize(dtype);
    Arena ar(work, (size_t)-1);
    w.V = ar.take((size_t)batch * n * ORM_KB * es);
    w.G = ar.take((size_t)batch * ORM_KB * ORM_KB * es);
    w.T = ar.take((size_t)batch * ORM_KB * ORM_KB * es);
    w.X = ar.take((size_t)batch * ORM_KB * ncols * es);
    w.X2 = ar.take((size_t)batch * ORM_KB * ncols * es);
    w.bytes = ar.off;
    return w;
}
size_t ormtr_workspace(int dtype, int n, int batch) { return orm_plan(dtype, n, n, batch, nullptr).bytes; }

template <class T>
static int ormtr_impl(int dtype, int n, int ncols, int batch, const T *A, long lda, long sA, const T *tau, T *Z, long ldz,
                      long sZ, void *work, cudaStream_t st) {
    if (n < 2) return NAO_OK;
    OrmWork w = orm_plan(dtype, n, ncols, batch, work);
    const int nref = n - 1;
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(larft_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)(ORM_KB * ORM_KB * sizeof(T))));
        attr = true;
    }
    const int nblocks = ceil_div(nref, ORM_KB);
    for (int blk = nblocks - 1; blk >= 0; --blk) {
        const int jb = blk * ORM_KB, kb = min(ORM_KB, nref - jb), m = n - jb - 1;
        const long ldv = m, sV = (long)n * ORM_KB;
        build_v_kernel<T><<<dim3(ceil_div(m, 256), kb, batch), 256, 0, st>>>(n, jb, kb, A, lda, sA, (T *)w.V, ldv, sV);
        NAO_LAUNCHED();
        // G = V^H V
        GemmDesc g = gemm_desc(OP_C, OP_N, kb, kb, m, 1.0, w.V, ldv, w.V, ldv, 0.0, w.G, kb);
        g.sA = sV; g.sB = sV; g.sC = ORM_KB * ORM_KB;
        if (int rc = gemm_launch(dtype, g, batch, st)) return rc;
        larft_kernel<T><<<batch, 256, kb * kb * sizeof(T), st>>>(kb, (const T *)w.G, ORM_KB * ORM_KB, tau + jb, n, (T *)w.T, ORM_KB * ORM_KB);
        NAO_LAUNCHED();
        // X = V^H Z[jb+1:, :]
        GemmDesc x = gemm_desc(OP_C, OP_N, kb, ncols, m, 1.0, w.V, ldv, Z + jb + 1, ldz, 0.0, w.X, kb);
        x.sA = sV; x.sB = sZ; x.sC = (long)ORM_KB * ncols;
        if (int rc = gemm_launch(dtype, x, batch, st)) return rc;
        // X2 = T X
        GemmDesc t = gemm_desc(OP_N, OP_N, kb, ncols, kb, 1.0, w.T, kb, w.X, kb, 0.0, w.X2, kb);
        t.sA = ORM_KB * ORM_KB; t.sB = (long)ORM_KB * ncols; t.sC = (long)ORM_KB * ncols; t.maskA = MASK_UPPER;
        if (int rc = gemm_launch(dtype, t, batch, st)) return rc;
        // Z[jb+1:, :] -= V X2
        GemmDesc u = gemm_desc(OP_N, OP_N, m, ncols, kb, -1.0, w.V, ldv, w.X2, kb, 1.0, Z + jb + 1, ldz);
        u.sA = sV; u.sB = (long)ORM_KB * ncols; u.sC = sZ;
        if (int rc = gemm_launch(dtype, u, batch, st)) return rc;
    }
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int ormtr(int dtype, int n, int ncols, int batch, const void *A, long lda, long sA, const void *tau, void *Z, long ldz,
          long sZ, void *work, cudaStream_t st) {
    return dtype == NAO_COMPLEX
               ? ormtr_impl<cplx>(dtype, n, ncols, batch, (const cplx *)A, lda, sA, (const cplx *)tau, (cplx *)Z, ldz, sZ, work, st)
               : ormtr_impl<double>(dtype, n, ncols, batch, (const double *)A, lda, sA, (const double *)tau, (double *)Z, ldz, sZ, work, st);
}

}  // namespace nao
