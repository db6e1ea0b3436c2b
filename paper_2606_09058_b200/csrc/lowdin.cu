// lowdin.cu -- the paper's own orthogonalisation (Part 2-1/2-2, 3-1/3-2):
// S = U s U^H by the library's eigensolver, W = s^{-1/2} U^H (the paper's V^H, V = U s^{-1/2}), then A = W H W^H and
// C = W^H Z exactly as on the Cholesky route, with a dense W instead of a triangular one.  Optional pruning of
// near-dependent directions (s_i <= rel * s_max) for ill-conditioned S: the rows of W of the pruned directions are zero, the
// reduced matrix gets NAO_PRUNED_LEVEL on their diagonal entries, so these levels sort to the top with zero vectors C.
#include "nao_internal.cuh"
#include "scalar.cuh"

namespace nao {

// W(i, j) = g_i conj(U(j, i)),  g_i = s_i^{-1/2}, or 0 for a pruned direction.  32x32 tiles through shared memory.
template <class T>
__global__ void lowdin_w_kernel(int n, const T *U, long ldu, long sU, const double *s, double rel, T *W, long ldw, long sW,
                                int *info) {
    typedef Ops<T> O;
    __shared__ T tile[32][33];
    const int b = blockIdx.z;
    U += (long)b * sU; W += (long)b * sW; s += (long)b * n;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const double smax = s[n - 1];
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        const int r = j0 + threadIdx.x, cc = i0 + c;                 // tile[c][x] = U(j0 + x, i0 + c)
        tile[c][threadIdx.x] = (r < n && cc < n) ? U[r + (long)cc * ldu] : O::zero();
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        const int i = i0 + threadIdx.x, j = j0 + c;
        if (i < n && j < n) {
            const double si = s[i];
            const double g = (si > 0.0 && si > rel * smax) ? 1.0 / sqrt(si) : 0.0;
            W[i + (long)j * ldw] = O::scale(O::conj(tile[threadIdx.x][c]), g);
        }
    }
    // without pruning a non-positive eigenvalue of S is an error (S not positive definite)
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0 && threadIdx.y == 0 && rel == 0.0 && !(s[0] > 0.0) && info[b] == 0)
        info[b] = n + 2;
}

int lowdin_w(int dtype, int n, int batch, const void *U, long ldu, long sU, const double *s, double rel, void *W, long ldw,
             long sW, int *d_info, cudaStream_t st) {
    dim3 grid(ceil_div(n, 32), ceil_div(n, 32), batch), block(32, 8);
    if (dtype == NAO_COMPLEX) lowdin_w_kernel<cplx><<<grid, block, 0, st>>>(n, (const cplx *)U, ldu, sU, s, rel, (cplx *)W, ldw, sW, d_info);
    else lowdin_w_kernel<double><<<grid, block, 0, st>>>(n, (const double *)U, ldu, sU, s, rel, (double *)W, ldw, sW, d_info);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

// Pruned direction i <=> row i of W is identically zero: A(i, i) = big (in every one of the nrep diagonal blocks of order nS).
// ew / ea = doubles per element of W / A.
__global__ void lowdin_shift_kernel(int nS, int nrep, double *A, long lda, long sA, int ea, const double *W, long ldw, long sW,
                                    int ew, double big) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nS) return;
    A += (long)blockIdx.y * sA * ea; W += (long)blockIdx.y * sW * ew;
    bool zero = true;
    for (int j = 0; j < nS; ++j) {
        const double *p = W + (i + (long)j * ldw) * ew;
        if (p[0] != 0.0 || (ew == 2 && p[1] != 0.0)) zero = false;
    }
    if (zero)
        for (int r = 0; r < nrep; ++r) {
            double *d = A + ((long)(i + r * nS) * (lda + 1)) * ea;
            d[0] = big;
            if (ea == 2) d[1] = 0.0;
        }
}

int lowdin_shift(int dtype, int n, int nS, int batch, void *A, long lda, long sA, const void *W, int wdtype, long ldw, long sW,
                 double big, cudaStream_t st) {
    lowdin_shift_kernel<<<dim3(ceil_div(nS, 128), batch), 128, 0, st>>>(nS, n / nS, (double *)A, lda, sA,
                                                                       dtype == NAO_COMPLEX ? 2 : 1, (const double *)W, ldw, sW,
                                                                       wdtype == NAO_COMPLEX ? 2 : 1, big);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

}  // namespace nao
