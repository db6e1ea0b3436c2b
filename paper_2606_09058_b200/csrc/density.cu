// density.cu -- D = C diag(f) C^H (Eq. 8, Eq. 23; north_star form).
//
// HERK-shaped: only the tiles touching the lower triangle are computed on the DMMA GEMM core, with the Fermi
// weights f[k] fused into the A-fragment load (scaleK) and the k-range cut at the last column with |f| >= 1e-17
// (decided on the device: the GEMM descriptor lives in device memory and a one-warp kernel writes its k).  The upper
// triangle is then filled by a coalesced Hermitian mirror.
#include "nao_internal.cuh"

namespace nao {

__global__ void dm_setup_kernel(int n, int dtype, const void *C, long ldc, long sC, const double *F, void *D, long ldd,
                                long sD, GemmDesc *descs) {
    const int b = blockIdx.x;
    const double *f = F + (long)b * n;
    int last = -1;
    for (int k = threadIdx.x; k < n; k += 32)
        if (fabs(f[k]) >= 1e-17) last = k;
    for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    if (threadIdx.x == 0) {
        size_t es = dtype == NAO_COMPLEX ? 16 : 8;
        GemmDesc d;
        d.A = (const char *)C + (size_t)b * sC * es; d.B = d.A; d.C = (char *)D + (size_t)b * sD * es;
        d.lda = ldc; d.ldb = ldc; d.ldc = ldd; d.sA = d.sB = d.sC = 0;
        d.m = n; d.n = n; d.k = last + 1;
        d.opA = OP_N; d.opB = OP_C; d.maskA = d.maskB = MASK_NONE; d.offA = d.offB = 0;
        d.cmode = 1; d.conjC = 0; d.alpha = 1.0; d.beta = 0.0; d.scaleK = f; d.sScale = 0; d.ksplit = 1; d.sSplit = 0;
        descs[b] = d;
    }
}

}  // namespace nao

NAO_EXPORT int nao_density_workspace(int n, int batch, int dtype, size_t *bytes) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if (!bytes) return -4;
    *bytes = nao::align_up(sizeof(nao::GemmDesc) * (size_t)batch);
    return NAO_OK;
}

NAO_EXPORT int nao_density_matrix(int n, int batch, int dtype, const void *dC, long ldc, long strideC, const double *dF,
                                  void *dD, long ldd, long strideD, void *dwork, size_t work_bytes, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if (!dC) return -4;
    if (ldc < n) return -5;
    if (batch > 1 && strideC < (long)ldc * n) return -6;
    if (!dF) return -7;
    if (!dD) return -8;
    if (ldd < n) return -9;
    if (batch > 1 && strideD < (long)ldd * n) return -10;
    if (!dwork) return -11;
    size_t need; nao_density_workspace(n, batch, dtype, &need);
    if (work_bytes < need) return NAO_ERR_WORKSPACE;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    GemmDesc *descs = (GemmDesc *)dwork;
    dm_setup_kernel<<<batch, 32, 0, st>>>(n, dtype, dC, ldc, strideC, dF, dD, ldd, strideD, descs);
    NAO_LAUNCHED();
    int rc = gemm_launch_grouped(dtype, descs, batch, n, n, 1, OP_N, OP_C, true, st);
    if (rc) return rc;
    return herm_fill(dtype, n, dD, ldd, strideD, dD, ldd, strideD, batch, st);
}

// ---------------------------------------------------------------------------------------------------------------------
// nao_occupied_count: 1 + last level (over all items) with f >= threshold
// ---------------------------------------------------------------------------------------------------------------------
namespace nao {
// one CTA; the result goes straight to a pinned, device-mapped HOST word (the library allocates no device memory)
__global__ void __launch_bounds__(1024) occupied_count_kernel(int n, int batch, const double *F, double thr, int *out) {
    __shared__ int red[32];
    int last = -1;
    for (long e = threadIdx.x; e < (long)n * batch; e += blockDim.x)
        if (F[e] >= thr) last = max(last, (int)(e % n));
    for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = last;
    __syncthreads();
    if (threadIdx.x < 32) {
        last = red[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
        if (threadIdx.x == 0) *out = last + 1;
    }
}
}  // namespace nao

NAO_EXPORT int nao_occupied_count(int n, int batch, const double *dF, double threshold, int *h_count, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!dF) return -3;
    if (!h_count) return -5;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    static int *h_pinned = nullptr, *d_mapped = nullptr;
    if (!h_pinned) {
        if (cudaHostAlloc((void **)&h_pinned, sizeof(int), cudaHostAllocMapped) != cudaSuccess) return NAO_ERR_CUDA;
        if (cudaHostGetDevicePointer((void **)&d_mapped, h_pinned, 0) != cudaSuccess) return NAO_ERR_CUDA;
    }
    occupied_count_kernel<<<1, 1024, 0, st>>>(n, batch, dF, threshold, d_mapped);
    NAO_LAUNCHED();
    if (cudaStreamSynchronize(st) != cudaSuccess) return NAO_ERR_CUDA;
    *h_count = *h_pinned;
    return NAO_OK;
}
