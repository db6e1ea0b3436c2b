// util.cu -- element-wise helper kernels (copies, Hermitian completion, packing of the S factor).
// All are HBM/L2-bound streaming kernels: consecutive threads walk a column (coalesced), grid-stride over columns.
#include "nao_internal.cuh"

namespace nao {

template <class T> __device__ __forceinline__ T conj_(T x);
template <> __device__ __forceinline__ double conj_<double>(double x) { return x; }
template <> __device__ __forceinline__ cplx conj_<cplx>(cplx x) { return make_double2(x.x, -x.y); }
template <class T> __device__ __forceinline__ T zero_();
template <> __device__ __forceinline__ double zero_<double>() { return 0.0; }
template <> __device__ __forceinline__ cplx zero_<cplx>() { return make_double2(0.0, 0.0); }

static inline dim3 grid2d(int m, int n, int batch) {
    return dim3((unsigned)ceil_div(m, 256), (unsigned)min(n, 65535), (unsigned)batch);
}

template <class T>
__global__ void copy_kernel(int m, int n, const T *A, long lda, long sA, T *B, long ldb, long sB, int uplo) {
    A += (long)blockIdx.z * sA; B += (long)blockIdx.z * sB;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    for (int j = blockIdx.y; j < n; j += gridDim.y) {
        if (uplo == 1 && i < j) continue;
        if (uplo == 2 && i >= j) continue;
        B[i + (long)j * ldb] = A[i + (long)j * lda];
    }
}
int copy_matrix(int dtype, int m, int n, const void *A, long lda, long sA, void *B, long ldb, long sB, int batch,
                int uplo, cudaStream_t st) {
    if (m <= 0 || n <= 0 || batch <= 0) return NAO_OK;
    if (dtype == NAO_COMPLEX) copy_kernel<cplx><<<grid2d(m, n, batch), 256, 0, st>>>(m, n, (const cplx *)A, lda, sA, (cplx *)B, ldb, sB, uplo);
    else copy_kernel<double><<<grid2d(m, n, batch), 256, 0, st>>>(m, n, (const double *)A, lda, sA, (double *)B, ldb, sB, uplo);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

// B <- Hermitian completion of tril(A).  32x32 tiles through shared memory so both the read of the lower tile and
// the write of its mirrored upper tile are coalesced.  In-place (B == A) is safe: a tile pair is owned by one CTA.
template <class T>
__global__ void herm_fill_kernel(int n, const T *A, long lda, long sA, T *B, long ldb, long sB);
template <> __global__ void herm_fill_kernel<double>(int n, const double *A, long lda, long sA, double *B, long ldb, long sB) {
    __shared__ double tile[32][33];
    A += (long)blockIdx.z * sA; B += (long)blockIdx.z * sB;
    int ti = blockIdx.x, tj = blockIdx.y;
    if (tj > ti) return;
    int i0 = ti * 32, j0 = tj * 32;
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        tile[c][threadIdx.x] = (i < n && j < n) ? A[i + (long)j * lda] : 0.0;
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        if (i < n && j < n && i >= j) B[i + (long)j * ldb] = tile[c][threadIdx.x];
        int mi = j0 + threadIdx.x, mj = i0 + c;
        if (mi < n && mj < n && mi < mj) B[mi + (long)mj * ldb] = tile[threadIdx.x][c];
    }
}
template <> __global__ void herm_fill_kernel<cplx>(int n, const cplx *A, long lda, long sA, cplx *B, long ldb, long sB) {
    __shared__ cplx tile[32][33];
    A += (long)blockIdx.z * sA; B += (long)blockIdx.z * sB;
    int ti = blockIdx.x, tj = blockIdx.y;
    if (tj > ti) return;
    int i0 = ti * 32, j0 = tj * 32;
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        cplx v = make_double2(0.0, 0.0);
        if (i < n && j < n) { v = A[i + (long)j * lda]; if (i == j) v.y = 0.0; }
        tile[c][threadIdx.x] = v;
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        if (i < n && j < n && i >= j) B[i + (long)j * ldb] = tile[c][threadIdx.x];
        int mi = j0 + threadIdx.x, mj = i0 + c;
        if (mi < n && mj < n && mi < mj) { cplx v = tile[threadIdx.x][c]; v.y = -v.y; B[mi + (long)mj * ldb] = v; }
    }
}
int herm_fill(int dtype, int n, const void *A, long lda, long sA, void *B, long ldb, long sB, int batch, cudaStream_t st) {
    if (n <= 0 || batch <= 0) return NAO_OK;
    int t = ceil_div(n, 32);
    dim3 grid(t, t, batch), block(32, 8);
    if (dtype == NAO_COMPLEX) herm_fill_kernel<cplx><<<grid, block, 0, st>>>(n, (const cplx *)A, lda, sA, (cplx *)B, ldb, sB);
    else herm_fill_kernel<double><<<grid, block, 0, st>>>(n, (const double *)A, lda, sA, (double *)B, ldb, sB);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int set_zero(void *p, size_t bytes, cudaStream_t st) {
    if (bytes == 0) return NAO_OK;
    NAO_CUDA_CHECK(cudaMemsetAsync(p, 0, bytes, st));
    return NAO_OK;
}

__global__ void r2c_kernel(int m, int n, const double *Q, long ldq, long sQ, cplx *Z, long ldz, long sZ) {
    Q += (long)blockIdx.z * sQ; Z += (long)blockIdx.z * sZ;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    for (int j = blockIdx.y; j < n; j += gridDim.y) Z[i + (long)j * ldz] = make_double2(Q[i + (long)j * ldq], 0.0);
}
int real_to_complex(int m, int n, const double *Q, long ldq, long sQ, cplx *Z, long ldz, long sZ, int batch, cudaStream_t st) {
    if (m <= 0 || n <= 0 || batch <= 0) return NAO_OK;
    r2c_kernel<<<grid2d(m, n, batch), 256, 0, st>>>(m, n, Q, ldq, sQ, Z, ldz, sZ);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

// B (n x m, ldb) <- A^H for a complex m x n matrix A (lda): 32x32 tiles through shared memory, both sides coalesced
__global__ void conj_transpose_kernel(int m, int n, const cplx *A, long lda, long sA, cplx *B, long ldb, long sB) {
    __shared__ cplx tile[32][33];
    A += (long)blockIdx.z * sA; B += (long)blockIdx.z * sB;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        const int i = i0 + threadIdx.x, j = j0 + c;
        if (i < m && j < n) tile[c][threadIdx.x] = A[i + (long)j * lda];
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        const int j = j0 + threadIdx.x, i = i0 + c;          // B(j, i) = conj(A(i, j))
        if (i < m && j < n) { const cplx v = tile[threadIdx.x][c]; B[j + (long)i * ldb] = make_double2(v.x, -v.y); }
    }
}
int conj_transpose(int m, int n, const cplx *A, long lda, long sA, cplx *B, long ldb, long sB, int batch, cudaStream_t st) {
    if (m <= 0 || n <= 0 || batch <= 0) return NAO_OK;
    conj_transpose_kernel<<<dim3(ceil_div(m, 32), ceil_div(n, 32), batch), dim3(32, 8), 0, st>>>(m, n, A, lda, sA, B, ldb, sB);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

// S holds L in its lower triangle and the strict upper triangle of L^{-H} above it (nao.h).  W <- L^{-1}:
//   W(i,j) = conj(S(j,i)) for i > j ; W(i,i) = 1/S(i,i) ; 0 above.       (reads go through 32x32 smem tiles)
template <class T> __device__ __forceinline__ T recip_diag(T x);
template <> __device__ __forceinline__ double recip_diag<double>(double x) { return 1.0 / x; }
template <> __device__ __forceinline__ cplx recip_diag<cplx>(cplx x) { return make_double2(1.0 / x.x, 0.0); }

template <class T>
__global__ void unpack_linv_kernel(int n, const T *S, long lds, long sS, T *W, long ldw, long sW) {
    __shared__ T tile[32][33];
    S += (long)blockIdx.z * sS; W += (long)blockIdx.z * sW;
    int ti = blockIdx.x, tj = blockIdx.y;      // output tile (rows ti, cols tj)
    int i0 = ti * 32, j0 = tj * 32;
    if (tj > ti) {                              // strictly upper tile of W: zeros
        for (int c = threadIdx.y; c < 32; c += blockDim.y) {
            int i = i0 + threadIdx.x, j = j0 + c;
            if (i < n && j < n) W[i + (long)j * ldw] = zero_<T>();
        }
        return;
    }
    // read S tile (rows tj, cols ti) = mirrored position
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int r = j0 + threadIdx.x, cc = i0 + c;
        tile[c][threadIdx.x] = (r < n && cc < n) ? S[r + (long)cc * lds] : zero_<T>();   // tile[col - i0][row - j0]
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        if (i >= n || j >= n) continue;
        T v;
        if (i > j) v = conj_(tile[threadIdx.x][c]);          // S(j, i): row j = j0 + c, col i = i0 + x
        else if (i == j) v = recip_diag(tile[threadIdx.x][c]);
        else v = zero_<T>();
        W[i + (long)j * ldw] = v;
    }
}
// inverse direction: S(j,i) <- conj(W(i,j)) for i > j (strict upper of S), lower of S untouched
template <class T>
__global__ void pack_linv_kernel(int n, T *S, long lds, long sS, const T *W, long ldw, long sW) {
    __shared__ T tile[32][33];
    S += (long)blockIdx.z * sS; W += (long)blockIdx.z * sW;
    int ti = blockIdx.x, tj = blockIdx.y;      // W tile (rows ti, cols tj), ti >= tj
    if (tj > ti) return;
    int i0 = ti * 32, j0 = tj * 32;
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int i = i0 + threadIdx.x, j = j0 + c;
        tile[c][threadIdx.x] = (i < n && j < n) ? W[i + (long)j * ldw] : zero_<T>();   // tile[j - j0][i - i0]
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += blockDim.y) {
        int r = j0 + threadIdx.x, cc = i0 + c;      // S(r, cc) with r = j, cc = i
        if (r < n && cc < n && cc > r) S[r + (long)cc * lds] = conj_(tile[threadIdx.x][c]);
    }
}
int unpack_linv(int dtype, int n, const void *S, long lds, long sS, void *W, long ldw, long sW, int batch, cudaStream_t st) {
    if (n <= 0 || batch <= 0) return NAO_OK;
    int t = ceil_div(n, 32);
    dim3 grid(t, t, batch), block(32, 8);
    if (dtype == NAO_COMPLEX) unpack_linv_kernel<cplx><<<grid, block, 0, st>>>(n, (const cplx *)S, lds, sS, (cplx *)W, ldw, sW);
    else unpack_linv_kernel<double><<<grid, block, 0, st>>>(n, (const double *)S, lds, sS, (double *)W, ldw, sW);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}
int pack_linv(int dtype, int n, void *S, long lds, long sS, const void *W, long ldw, long sW, int batch, cudaStream_t st) {
    if (n <= 0 || batch <= 0) return NAO_OK;
    int t = ceil_div(n, 32);
    dim3 grid(t, t, batch), block(32, 8);
    if (dtype == NAO_COMPLEX) pack_linv_kernel<cplx><<<grid, block, 0, st>>>(n, (cplx *)S, lds, sS, (const cplx *)W, ldw, sW);
    else pack_linv_kernel<double><<<grid, block, 0, st>>>(n, (double *)S, lds, sS, (const double *)W, ldw, sW);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

}  // namespace nao
