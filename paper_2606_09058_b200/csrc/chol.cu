// chol.cu -- Cholesky factor S = L L^H and its inverse W = L^{-1} (the paper's role for it is
// Part 2-1/2-2 and 3-1/3-2, "diagonalise S, form V", PAPER.md:159-163, 189-193 -- computed once and reused in every
// later SCF step).
//
// Recursive blocked algorithm in which everything above the leaves is a DMMA GEMM:
//   [S11 .; S21 S22]:  (L11, W11) <- rec(S11);  L21 = S21 W11^H;  S22 -= L21 L21^H (lower tiles only);
//                      (L22, W22) <- rec(S22);  W21 = -W22 (L21 W11).
// Leaves (order <= 64) are factored and inverted inside shared memory by one CTA per batch item.
// L^{-1} is formed explicitly because the per-step reduction A = L^{-1} H L^{-H} and the back-substitution
// C = L^{-H} Z then become plain (triangular-masked) GEMMs -- the same choice the paper makes with its explicit
// V = U s^{-1/2} and V^H H V / V C' products.
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>

namespace nao {

static const int CHOL_LEAF = 64;

// One CTA per batch item.  nb <= 64.  S block (lower referenced) -> L in place; W block <- L^{-1} (lower; the
// strict upper part of the W block is zeroed).  info: first failing pivot (1-based, global index).
// Right-looking factorisation with ONE barrier per column: the scaled column j of L goes to a second array while the
// trailing update reads the unscaled column (a(i,k) -= a(i,j) conj(a(k,j)) / a(j,j)); thread <-> (row i, every 4th column).
// The inverse is a forward substitution per column, 4 adjacent lanes per column, so it needs warp-level barriers only.
template <class T>
__global__ void __launch_bounds__(256) chol_leaf_kernel(int nb, int off, T *S, long lds, long sS, T *W, long ldw,
                                                        long sW, int *info) {
    typedef Ops<T> O;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int ld = CHOL_LEAF + 1;
    T *sA = (T *)smem_raw;                 // [64][65] working copy a(i,j) at sA[i*ld + j]; later the inverse X
    T *sF = sA + CHOL_LEAF * ld;           // [64][65] the factor L
    const int b = blockIdx.x;
    S += (long)b * sS + off + (long)off * lds;
    W += (long)b * sW + off + (long)off * ldw;
    const int tid = threadIdx.x;
    for (int e = tid; e < CHOL_LEAF * CHOL_LEAF; e += 256) {
        const int i = e & (CHOL_LEAF - 1), j = e >> 6;
        sA[i * ld + j] = (i < nb && j < nb && i >= j) ? S[i + (long)j * lds] : O::zero();
        sF[i * ld + j] = O::zero();
    }
    __syncthreads();
    const int ti = tid & (CHOL_LEAF - 1), tq = tid >> 6;
    for (int j = 0; j < nb; ++j) {
        double ajj = O::real(sA[j * ld + j]);
        if (!(ajj > 0.0)) {
            if (tid == 0 && info[b] == 0) info[b] = off + j + 1;
            ajj = 1.0;
        }
        const double piv = sqrt(ajj), rinv = 1.0 / piv, ainv = 1.0 / ajj;
        if (ti >= j && ti < nb) {
            const T aij = sA[ti * ld + j];
            if (tq == 0) sF[ti * ld + j] = ti == j ? O::from_real(piv) : O::scale(aij, rinv);
            if (ti > j) {
                const T l = O::scale(aij, ainv);
                for (int k = j + 1 + tq; k <= ti; k += 4)
                    sA[ti * ld + k] = O::sub(sA[ti * ld + k], O::mul_conj(l, sA[k * ld + j]));
            }
        }
        __syncthreads();
    }
    // inverse by forward substitution, X(i,c) = (delta_ic - sum_{k=c}^{i-1} L(i,k) X(k,c)) / L(i,i): 4 adjacent lanes
    // split the k-sum of one column, nobody else touches that column of X
    {
        T *sX = sA;
        const int c = tid >> 2, part = tid & 3;
        for (int i = 0; i < nb; ++i) {
            T acc = O::zero();
            if (c < nb && i > c)
                for (int k = c + part; k < i; k += 4) acc = O::sub(acc, O::mul(sF[i * ld + k], sX[k * ld + c]));
            double *a = (double *)&acc;
#pragma unroll
            for (int w = 0; w < (int)(sizeof(T) / 8); ++w) {
                a[w] += __shfl_xor_sync(0xffffffffu, a[w], 1);
                a[w] += __shfl_xor_sync(0xffffffffu, a[w], 2);
            }
            if (c < nb && part == 0) {
                const double dinv = 1.0 / O::real(sF[i * ld + i]);
                T v;
                if (i < c) v = O::zero();
                else if (i == c) v = O::from_real(dinv);
                else v = O::scale(acc, dinv);
                sX[i * ld + c] = v;
            }
            __syncwarp();
        }
    }
    __syncthreads();
    for (int e = tid; e < CHOL_LEAF * CHOL_LEAF; e += 256) {
        const int i = e & (CHOL_LEAF - 1), j = e >> 6;
        if (i < nb && j < nb) {
            if (i >= j) S[i + (long)j * lds] = sF[i * ld + j];
            W[i + (long)j * ldw] = sA[i * ld + j];
        }
    }
}

template <class T>
static int leaf(int nb, int off, int batch, void *S, long lds, long sS, void *W, long ldw, long sW, int *info,
                cudaStream_t st) {
    size_t smem = 2 * (size_t)CHOL_LEAF * (CHOL_LEAF + 1) * sizeof(T);
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(chol_leaf_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            (int)(2 * CHOL_LEAF * (CHOL_LEAF + 1) * sizeof(T))));
        attr = true;
    }
    chol_leaf_kernel<T><<<batch, 256, smem, st>>>(nb, off, (T *)S, lds, sS, (T *)W, ldw, sW, info);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

struct CholCtx {
    int dtype, batch; size_t es;
    char *S; long lds, sS; char *W; long ldw, sW; char *T; long ldt, sT; int *info; cudaStream_t st;
    void *scratch; size_t scratch_elems; int nsm;       // split-K partial sums of the mid-level products (optional)
    void *s(int i, int j) const { return S + ((size_t)i + (size_t)j * lds) * es; }
    void *w(int i, int j) const { return W + ((size_t)i + (size_t)j * ldw) * es; }
    void *t(int i, int j) const { return T + ((size_t)i + (size_t)j * ldt) * es; }
};

// A product of the recursion.  Mid-level nodes have few output tiles and a long k: with scratch they are split along k so
// that the launch covers the SMs (n = 6656: the 16 products of order 832 take 185 us each on 49 CTAs).
static int chol_gemm(const CholCtx &c, const GemmDesc &d) {
    const long tiles = (long)ceil_div(d.m, 128) * ceil_div(d.n, c.dtype == NAO_COMPLEX ? 64 : 128) * c.batch;
    if (c.scratch && d.cmode == 0 && d.beta == 0.0 && d.k >= 256 && 2 * tiles <= c.nsm) {
        int ks = (int)std::min<long>(std::min<long>(c.nsm / tiles, d.k / 128), 16);
        while (ks >= 2 && (size_t)ks * d.m * d.n * c.batch > c.scratch_elems) --ks;
        if (ks >= 2) return gemm_splitk(c.dtype, d, c.batch, ks, c.scratch, c.st);
    }
    return gemm_launch(c.dtype, d, c.batch, c.st);
}

static int rec(const CholCtx &c, int off, int n) {
    int rc;
    if (n <= CHOL_LEAF) {
        return c.dtype == NAO_COMPLEX ? leaf<cplx>(n, off, c.batch, c.S, c.lds, c.sS, c.W, c.ldw, c.sW, c.info, c.st)
                                      : leaf<double>(n, off, c.batch, c.S, c.lds, c.sS, c.W, c.ldw, c.sW, c.info, c.st);
    }
    int n1 = ((n / 2 + CHOL_LEAF - 1) / CHOL_LEAF) * CHOL_LEAF;
    if (n1 >= n) n1 = n / 2;
    int n2 = n - n1, o2 = off + n1;
    if ((rc = rec(c, off, n1))) return rc;
    // T21 = S21 * W11^H
    GemmDesc d = gemm_desc(OP_N, OP_C, n2, n1, n1, 1.0, c.s(o2, off), c.lds, c.w(off, off), c.ldw, 0.0, c.t(o2, off), c.ldt);
    d.sA = c.sS; d.sB = c.sW; d.sC = c.sT; d.maskB = MASK_LOWER;
    if ((rc = chol_gemm(c, d))) return rc;
    if ((rc = copy_matrix(c.dtype, n2, n1, c.t(o2, off), c.ldt, c.sT, c.s(o2, off), c.lds, c.sS, c.batch, 0, c.st))) return rc;
    // S22 -= L21 L21^H  (lower tiles)
    d = gemm_desc(OP_N, OP_C, n2, n2, n1, -1.0, c.s(o2, off), c.lds, c.s(o2, off), c.lds, 1.0, c.s(o2, o2), c.lds);
    d.sA = c.sS; d.sB = c.sS; d.sC = c.sS; d.cmode = 1;
    if ((rc = gemm_launch(c.dtype, d, c.batch, c.st))) return rc;
    if ((rc = rec(c, o2, n2))) return rc;
    // T21 = L21 * W11
    d = gemm_desc(OP_N, OP_N, n2, n1, n1, 1.0, c.s(o2, off), c.lds, c.w(off, off), c.ldw, 0.0, c.t(o2, off), c.ldt);
    d.sA = c.sS; d.sB = c.sW; d.sC = c.sT; d.maskB = MASK_LOWER;
    if ((rc = chol_gemm(c, d))) return rc;
    // W21 = -W22 * T21
    d = gemm_desc(OP_N, OP_N, n2, n1, n2, -1.0, c.w(o2, o2), c.ldw, c.t(o2, off), c.ldt, 0.0, c.w(o2, off), c.ldw);
    d.sA = c.sW; d.sB = c.sT; d.sC = c.sW; d.maskA = MASK_LOWER;
    return chol_gemm(c, d);
}

int potrf_trtri(int dtype, int n, int batch, void *S, long lds, long sS, void *W, long ldw, long sW, void *T, long ldt,
                long sT, int *d_info, cudaStream_t st, void *scratch, size_t scratch_bytes) {
    int nsm = 148, dev = 0;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    CholCtx c{dtype, batch, esize(dtype), (char *)S, lds, sS, (char *)W, ldw, sW, (char *)T, ldt, sT, d_info, st,
              scratch, scratch ? scratch_bytes / esize(dtype) : 0, nsm};
    // W's strict upper triangle must read as zero: leaves write their own blocks, the rest is cleared here
    for (int b = 0; b < batch; ++b) {
        // clear column by column only if ldw != n; the common case is a dense n x n buffer
        if (ldw == n) { if (int rc = set_zero((char *)W + (size_t)b * sW * c.es, (size_t)n * n * c.es, st)) return rc; }
        else for (int j = 0; j < n; ++j) if (int rc = set_zero((char *)W + ((size_t)b * sW + (size_t)j * ldw) * c.es, (size_t)n * c.es, st)) return rc;
    }
    return rec(c, 0, n);
}

}  // namespace nao

NAO_EXPORT int nao_potrf_trtri(int n, int batch, int dtype, void *dS, long lds, long strideS, void *dLinv, void *dtmp,
                               int *d_info, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if (!dS) return -4;
    if (lds < n) return -5;
    if (batch > 1 && strideS < (long)lds * n) return -6;
    if (!dLinv) return -7;
    if (!dtmp) return -8;
    if (!d_info) return -9;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(d_info, 0, sizeof(int) * batch, st) != cudaSuccess) return NAO_ERR_CUDA;
    int rc = potrf_trtri(dtype, n, batch, dS, lds, strideS, dLinv, n, (long)n * n, dtmp, n, (long)n * n, d_info, st);
    if (rc) return rc;
    return pack_linv(dtype, n, dS, lds, strideS, dLinv, n, (long)n * n, batch, st);
}
