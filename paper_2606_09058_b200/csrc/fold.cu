// fold.cu -- the step after the hot path: the energy-weighted density matrix and the k-folded
// real-space density matrix.  The paper leaves both on the CPU inside its Part 4/5 ("calculating the density matrix",
// PAPER.md:163-169), where the redistribution alone costs 9-10 % of the step.
//
//   * energy weights    fe[b,i] = f[b,i] * e[b,i]; nao_density_matrix with these weights gives C diag(f e) C^H
//   * folding           D(R) = sum_k w_k exp(-i k.R) D(k)      (inverse of the Bloch sum, Eq. 12)
//
// The fold is a streaming kernel: every D(k) element is read once (up to 16 k-points are held in registers), every D(R)
// element written once; the nk x nR phase table w_k exp(-i k.R) is formed on the device and broadcast from shared memory.
#include "nao_internal.cuh"
#include "scalar.cuh"

namespace nao {

static const int FOLD_NT = 128;      // threads per CTA = rows per tile
static const int FOLD_COLS = 8;      // columns per CTA
static const int FOLD_RMAX = 128;    // lattice vectors per pass (phase table of 128 x KC complex in shared memory)

__global__ void energy_weights_kernel(long total, const double *E, const double *F, double *FE) {
    long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < total) FE[i] = F[i] * E[i];
}

// table[r * kc_pad + q] = w_k exp(-i k.R_r) for k = k0 + q (zero for the padding q >= kc)
__global__ void fold_phase_kernel(int nk, int nR, int k0, int kc, int kc_pad, const double *kpt, const double *wk,
                                  const double *Rv, cplx *table) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nR * kc_pad) return;
    int r = e / kc_pad, q = e % kc_pad;
    cplx v = make_double2(0.0, 0.0);
    if (q < kc) {
        int k = k0 + q;
        double phi = -(kpt[3 * k] * Rv[3 * r] + kpt[3 * k + 1] * Rv[3 * r + 1] + kpt[3 * k + 2] * Rv[3 * r + 2]);
        double s, c;
        sincos(phi, &s, &c);
        v = make_double2(wk[k] * c, wk[k] * s);
    }
    table[e] = v;
}

// One CTA: 128 rows x 8 columns of every D(R), R in [r0, r0 + nr).  KC k-points per pass; accumulate != 0 adds to D(R).
template <bool REAL_OUT, int KC>
__global__ void __launch_bounds__(FOLD_NT) fold_kernel(int n, int k0, int kc, int r0, int nr, const cplx *Dk, long ldd,
                                                       long sD, const cplx *table, void *DR, long lddr, long sDR,
                                                       int accumulate) {
    __shared__ cplx s_ph[FOLD_RMAX * KC];
    for (int e = threadIdx.x; e < nr * KC; e += FOLD_NT) s_ph[e] = table[(long)r0 * KC + e];
    __syncthreads();
    const int i = blockIdx.x * FOLD_NT + threadIdx.x;
    if (i >= n) return;
    const int jbeg = blockIdx.y * FOLD_COLS, jend = min(n, jbeg + FOLD_COLS);
    for (int j = jbeg; j < jend; ++j) {
        cplx d[KC];
#pragma unroll
        for (int q = 0; q < KC; ++q) d[q] = q < kc ? ldcg(Dk + (long)(k0 + q) * sD + i + (long)j * ldd) : make_double2(0.0, 0.0);
        for (int r = 0; r < nr; ++r) {
            double ar = 0.0, ai = 0.0;
#pragma unroll
            for (int q = 0; q < KC; ++q) {
                const cplx p = s_ph[r * KC + q];
                ar = fma(p.x, d[q].x, ar); ar = fma(-p.y, d[q].y, ar);
                if (!REAL_OUT) { ai = fma(p.x, d[q].y, ai); ai = fma(p.y, d[q].x, ai); }
            }
            const long o = (long)(r0 + r) * sDR + i + (long)j * lddr;
            if (REAL_OUT) {
                double *out = (double *)DR + o;
                *out = accumulate ? *out + ar : ar;
            } else {
                cplx *out = (cplx *)DR + o;
                cplx v = make_double2(ar, ai);
                if (accumulate) { cplx c = *out; v.x += c.x; v.y += c.y; }
                *out = v;
            }
        }
    }
}

template <bool REAL_OUT, int KC>
static void fold_launch(int n, int k0, int kc, int nR, const cplx *Dk, long ldd, long sD, const cplx *table, void *DR,
                        long lddr, long sDR, int accumulate, cudaStream_t st) {
    dim3 grid(ceil_div(n, FOLD_NT), ceil_div(n, FOLD_COLS));
    for (int r0 = 0; r0 < nR; r0 += FOLD_RMAX) {
        fold_kernel<REAL_OUT, KC><<<grid, FOLD_NT, 0, st>>>(n, k0, kc, r0, min(FOLD_RMAX, nR - r0), Dk, ldd, sD, table, DR,
                                                            lddr, sDR, accumulate);
        NAO_LAUNCHED();
    }
}

}  // namespace nao

NAO_EXPORT int nao_energy_weights(int n, int batch, const double *dE, const double *dF, double *dFE, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!dE) return -3;
    if (!dF) return -4;
    if (!dFE) return -5;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    long total = (long)n * batch;
    energy_weights_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(total, dE, dF, dFE);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

NAO_EXPORT int nao_fold_workspace(int nk, int nR, size_t *bytes) {
    if (nk < 1) return -1;
    if (nR < 1) return -2;
    if (!bytes) return -3;
    // k (3 nk) + w (nk) + R (3 nR) doubles, then the phase table of one pass (nR x 16 complex)
    *bytes = nao::align_up(sizeof(double) * (4 * (size_t)nk + 3 * (size_t)nR)) + nao::align_up(sizeof(nao::cplx) * 16 * (size_t)nR);
    return NAO_OK;
}

NAO_EXPORT int nao_fold_density(int n, int nk, int nR, int out_dtype, const void *dDk, long ldd, long strideD,
                                const double *h_k, const double *h_w, const double *h_R, void *dDR, long lddr,
                                long strideDR, void *dwork, size_t work_bytes, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (nk < 1) return -2;
    if (nR < 1) return -3;
    if (out_dtype != NAO_REAL && out_dtype != NAO_COMPLEX) return -4;
    if (!dDk) return -5;
    if (ldd < n) return -6;
    if (nk > 1 && strideD < (long)ldd * n) return -7;
    if (!h_k) return -8;
    if (!h_w) return -9;
    if (!h_R) return -10;
    if (!dDR) return -11;
    if (lddr < n) return -12;
    if (nR > 1 && strideDR < (long)lddr * n) return -13;
    if (!dwork) return -14;
    size_t need; nao_fold_workspace(nk, nR, &need);
    if (work_bytes < need) return NAO_ERR_WORKSPACE;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *d_k = (double *)dwork, *d_w = d_k + 3 * (size_t)nk, *d_R = d_w + nk;
    cplx *table = (cplx *)((char *)dwork + align_up(sizeof(double) * (4 * (size_t)nk + 3 * (size_t)nR)));
    // pageable host memory: the copies are staged before the calls return, the host arrays may be reused at once
    NAO_CUDA_CHECK(cudaMemcpyAsync(d_k, h_k, sizeof(double) * 3 * nk, cudaMemcpyHostToDevice, st));
    NAO_CUDA_CHECK(cudaMemcpyAsync(d_w, h_w, sizeof(double) * nk, cudaMemcpyHostToDevice, st));
    NAO_CUDA_CHECK(cudaMemcpyAsync(d_R, h_R, sizeof(double) * 3 * nR, cudaMemcpyHostToDevice, st));
    const bool real_out = out_dtype == NAO_REAL;
    for (int k0 = 0; k0 < nk; k0 += 16) {
        const int kc = nk - k0 < 16 ? nk - k0 : 16;
        const int kc_pad = kc <= 8 ? 8 : 16;
        fold_phase_kernel<<<ceil_div(nR * kc_pad, 128), 128, 0, st>>>(nk, nR, k0, kc, kc_pad, d_k, d_w, d_R, table);
        NAO_LAUNCHED();
        const int acc = k0 > 0;
        const cplx *Dk = (const cplx *)dDk;
        if (real_out) {
            if (kc_pad == 8) fold_launch<true, 8>(n, k0, kc, nR, Dk, ldd, strideD, table, dDR, lddr, strideDR, acc, st);
            else fold_launch<true, 16>(n, k0, kc, nR, Dk, ldd, strideD, table, dDR, lddr, strideDR, acc, st);
        } else {
            if (kc_pad == 8) fold_launch<false, 8>(n, k0, kc, nR, Dk, ldd, strideD, table, dDR, lddr, strideDR, acc, st);
            else fold_launch<false, 16>(n, k0, kc, nR, Dk, ldd, strideD, table, dDR, lddr, strideDR, acc, st);
        }
    }
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}
