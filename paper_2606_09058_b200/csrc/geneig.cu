// geneig.cu -- drivers: nao_heev (standard Hermitian problem) and nao_geneig (H C = S C diag(e)).
//
// nao_geneig (Eq. 5/11/21; the paper's Part 2 / Part 3):
//   1. S = L L^H, W = L^{-1}                (skipped with NAO_S_FACTORED: W is unpacked from dS)
//   2. A = W H W^H                          (paper: H' = V^H H V, Part 2-3 / 3-3; here V = W^H)
//   3. A = Z diag(e) Z^H                    (Part 2-4 / 3-5)
//   4. C = W^H Z                            (Part 2-5 / 3-6)
// With NAO_NC_BLOCK_S the overlap is S_NC = diag(S, S) with S real N x N (Eq. 25-27): only the
// real N x N S is factored and steps 2 and 4 run block-wise on the four N x N spin blocks.
#include "nao_internal.cuh"
#include <algorithm>

namespace nao {

// ----------------------------------------------------------------------------------------------------- heev
struct HeevPlan { size_t d, e, tau, qt, sub, v2, tau2, sub2, bytes; bool two_stage; };
// Default switch-over (flags force either path), from `microbench heev` on B200 with all eigenvectors, one-stage vs
// two-stage in ms: real n = 1664 x 2 items 41.6 vs 40.3, 3328 x 2 106.8 vs 102.3, 3328 x 1 97.6 vs 88.9, 4992 x 2 222.7 vs
// 211.0, 6656 x 1 309.7 vs 262.2, 6656 x 2 413.6 vs 351, 9984 x 1 698 vs 617; complex n = 9984 1.29 s vs 1.5 s (the second
// back-transformation runs at a lower rate in complex arithmetic, and the chase cannot double-buffer complex blocks).
static const int TWO_STAGE_MIN_N_REAL = 1536;
static bool use_two_stage(int dtype, int n, int batch, unsigned flags) {
    if (flags & NAO_TRD_ONE_STAGE) return false;
    if (!he2hb_supported(dtype, n, batch)) return false;
    if (flags & NAO_TRD_TWO_STAGE) return true;
    return dtype == NAO_REAL && n >= TWO_STAGE_MIN_N_REAL;
}
static HeevPlan heev_plan(int dtype, int n, int batch, unsigned flags) {
    HeevPlan p; size_t off = 0;
    auto take = [&](size_t b) { size_t o = off; off += align_up(b); return o; };
    p.two_stage = use_two_stage(dtype, n, batch, flags);
    p.d = take((size_t)batch * n * 8); p.e = take((size_t)batch * n * 8); p.tau = take((size_t)batch * n * esize(dtype));
    p.qt = take(dtype == NAO_COMPLEX ? (size_t)batch * n * n * 8 : 0);
    p.v2 = p.tau2 = p.sub2 = 0;
    if (p.two_stage) {
        p.v2 = take((size_t)batch * n * n * esize(dtype));
        p.tau2 = take((size_t)batch * hb2st_nk(n) * n * esize(dtype));
        const size_t s2 = std::max(std::max(he2hb_workspace(dtype, n, batch), hb2st_workspace(dtype, n, batch)),
                                   std::max(std::max(stedc_workspace(n, batch), q2_workspace(dtype, n, batch)),
                                            ormtr_workspace(dtype, n, batch)));
        p.sub = take(s2);
    } else {
        p.sub = take(std::max(hetrd_workspace(dtype, n, batch), std::max(stedc_workspace(n, batch), ormtr_workspace(dtype, n, batch))));
    }
    p.bytes = off;
    return p;
}

static int heev(int dtype, int n, int batch, unsigned flags, void *A, long lda, long sA, double *E, void *Z, long ldz,
                long sZ, void *work, int *d_info, cudaStream_t st, int nvec = -1, int phase = 3) {
    // phase bit 0: reduction to tridiagonal form + D&C (eigenvalues; Q_T and the reflectors stay in the workspace)
    // phase bit 1: back-transformation of the nvec lowest eigenvectors
    if (nvec < 0 || nvec > n) nvec = n;
    HeevPlan p = heev_plan(dtype, n, batch, flags);
    char *w = (char *)work;
    double *d = (double *)(w + p.d), *e = (double *)(w + p.e);
    void *tau = w + p.tau, *sub = w + p.sub;
    void *V2 = w + p.v2, *tau2 = w + p.tau2;
    int rc = NAO_OK;
    if (phase & 1) {
        prof_mark(2, st);
        if (p.two_stage) {
            if ((rc = he2hb(dtype, n, batch, A, lda, sA, tau, sub, st))) return rc;
            prof_mark(3, st);
            if ((rc = hb2st(dtype, n, batch, A, lda, sA, d, e, V2, n, (long)n * n, tau2, sub, st))) return rc;
        } else {
            if ((rc = hetrd(dtype, n, batch, A, lda, sA, d, e, tau, sub, st))) return rc;
            prof_mark(3, st);
        }
        prof_mark(4, st);
        // with both phases in one call the D&C runs through; otherwise it stops at the eigenvalues and is continued below
        const int dc_phase = (phase & 2) ? 3 : 1;
        if (dtype == NAO_COMPLEX) {
            double *qt = (double *)(w + p.qt);
            if ((rc = stedc(n, batch, d, e, E, qt, n, (long)n * n, sub, d_info, st, nvec, dc_phase))) return rc;
        } else {
            if ((rc = stedc(n, batch, d, e, E, (double *)Z, ldz, sZ, sub, d_info, st, nvec, dc_phase))) return rc;
        }
        prof_mark(5, st);
    }
    if (!(phase & 2)) return rc;
    if (!(phase & 1)) {        // eigenvectors of the tridiagonal matrix: only the nvec lowest (top merge restricted)
        if (dtype == NAO_COMPLEX) {
            if ((rc = stedc(n, batch, d, e, E, (double *)(w + p.qt), n, (long)n * n, sub, d_info, st, nvec, 2))) return rc;
        } else {
            if ((rc = stedc(n, batch, d, e, E, (double *)Z, ldz, sZ, sub, d_info, st, nvec, 2))) return rc;
        }
    }
    if (dtype == NAO_COMPLEX)
        if ((rc = real_to_complex(n, nvec, (const double *)(w + p.qt), n, (long)n * n, (cplx *)Z, ldz, sZ, batch, st))) return rc;
    if (p.two_stage) {
        if ((rc = q2_apply(dtype, n, nvec, batch, V2, n, (long)n * n, tau2, Z, ldz, sZ, sub, st))) return rc;
        prof_mark(6, st);
        rc = ormtr(dtype, n, nvec, batch, TRD2_B, A, lda, sA, tau, Z, ldz, sZ, sub, st);
    } else {
        prof_mark(6, st);
        rc = ormtr(dtype, n, nvec, batch, 1, A, lda, sA, tau, Z, ldz, sZ, sub, st);
    }
    prof_mark(7, st);
    return rc;
}

// ----------------------------------------------------------------------------------------------------- geneig
static double g_lowdin_rel = 0.0;      // nao_set_lowdin_threshold

// NAO_STREAM_GROUPS_2/4/8: number of internal streams the batch of nao_geneig is spread over
static int stream_groups(unsigned flags, int batch) {
    int g = 1 << ((flags & NAO_STREAM_GROUPS_MASK) >> 5);
    while (g > 1 && batch < g) g >>= 1;
    return g;
}

struct GePlan { size_t W, Wc, A, X, heev, bytes; int nS, sdtype, nitemsS; };
static GePlan ge_plan(int n, int batch, int dtype, unsigned flags, bool shared_S) {
    GePlan p; size_t off = 0;
    auto take = [&](size_t b) { size_t o = off; off += align_up(b); return o; };
    const bool nc = flags & NAO_NC_BLOCK_S;
    p.nS = nc ? n / 2 : n; p.sdtype = nc ? NAO_REAL : dtype; p.nitemsS = shared_S ? 1 : batch;
    p.W = take((size_t)p.nitemsS * p.nS * p.nS * esize(p.sdtype));
    p.Wc = take(nc ? (size_t)p.nitemsS * p.nS * p.nS * 16 : 0);
    p.A = take((size_t)batch * n * n * esize(dtype));
    p.X = take((size_t)batch * n * n * esize(dtype));
    size_t hb = heev_plan(dtype, n, batch, flags).bytes;
    if (flags & NAO_LOWDIN) hb = std::max(hb, heev_plan(p.sdtype, p.nS, p.nitemsS, flags).bytes);
    p.heev = take(hb);
    p.bytes = off;
    return p;
}

}  // namespace nao

NAO_EXPORT int nao_heev_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if (!bytes) return -5;
    *bytes = nao::heev_plan(dtype, n, batch, flags).bytes;
    return NAO_OK;
}

NAO_EXPORT int nao_heev(int n, int batch, int dtype, unsigned flags, void *dA, long lda, long strideA, double *dE, void *dZ,
                        long ldz, long strideZ, void *dwork, size_t work_bytes, int *d_info, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if (!dA) return -5;
    if (lda < n) return -6;
    if (batch > 1 && strideA < lda * (long)n) return -7;
    if (!dE) return -8;
    if (!dZ) return -9;
    if (ldz < n) return -10;
    if (batch > 1 && strideZ < ldz * (long)n) return -11;
    if (!dwork) return -12;
    if (work_bytes < heev_plan(dtype, n, batch, flags).bytes) return NAO_ERR_WORKSPACE;
    if (!d_info) return -14;
    if (int rcb = bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(d_info, 0, sizeof(int) * batch, st) != cudaSuccess) return NAO_ERR_CUDA;
    return heev(dtype, n, batch, flags, dA, lda, strideA, dE, dZ, ldz, strideZ, dwork, d_info, st);
}

NAO_EXPORT int nao_geneig_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if ((flags & NAO_NC_BLOCK_S) && (dtype != NAO_COMPLEX || (n & 1))) return -4;
    if (!bytes) return -5;
    const int groups = nao::stream_groups(flags, batch);
    flags &= ~NAO_STREAM_GROUPS_MASK;
    size_t plain = nao::ge_plan(n, batch, dtype, flags, false).bytes;
    if (groups > 1) {
        // every group carves its own slice, planned with the group's share of the SMs
        nao::set_sm_limit(nao::sm_count() / groups);
        size_t total = 0;
        for (int g = 0; g < groups; ++g) {
            const int b0 = (int)((long)batch * g / groups), b1 = (int)((long)batch * (g + 1) / groups);
            total += nao::align_up(nao::ge_plan(n, b1 - b0, dtype, flags, false).bytes);
        }
        nao::set_sm_limit(0);
        if (total > plain) plain = total;
    }
    *bytes = plain;
    return NAO_OK;
}

// phase bit 0: factor S, reduce, tridiagonalise, D&C (eigenvalues in dE; everything the back-transformation needs stays in
// dwork);  phase bit 1: back-transform the nvec lowest eigenvectors and form C.  A phase-2 call must follow a phase-1 call
// with the same arguments and an untouched workspace.
static int geneig_impl(int n, int batch, int dtype, unsigned flags, int nvec, const void *dH, long ldh, long strideH, void *dS,
                       long lds, long strideS, double *dE, void *dC, long ldc, long strideC, void *dwork,
                       size_t work_bytes, int *d_info, void *cuda_stream, int phase = 3, cudaEvent_t h_ready = nullptr) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    const bool nc = flags & NAO_NC_BLOCK_S;
    if (nc && (dtype != NAO_COMPLEX || (n & 1))) return -4;
    const int nS = nc ? n / 2 : n;
    if (!dH) return -5;
    if (ldh < n) return -6;
    if (batch > 1 && strideH < ldh * (long)n) return -7;
    if (!dS) return -8;
    if (lds < nS) return -9;
    const bool shared_S = (strideS == 0);
    if (!shared_S && batch > 1 && strideS < lds * (long)nS) return -10;
    if (!dE) return -11;
    if (!dC) return -12;
    if (ldc < n) return -13;
    if (batch > 1 && strideC < ldc * (long)n) return -14;
    if (!dwork) return -15;
    GePlan p = ge_plan(n, batch, dtype, flags, shared_S);
    if (work_bytes < p.bytes) return NAO_ERR_WORKSPACE;
    if (!d_info) return -17;
    if (phase != 0) if (int rcb = bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char *w = (char *)dwork;
    const size_t es = esize(dtype);
    void *W = w + p.W, *A = w + p.A, *X = w + p.X;
    const long sW = (long)nS * nS, sAX = (long)n * n;
    int rc;
    const void *Wm = W;
    const long sWm = shared_S ? 0 : sW;
    const bool lowdin = flags & NAO_LOWDIN;
    const int wmask = lowdin ? MASK_NONE : MASK_LOWER;        // the Cholesky route's W = L^{-1} is lower triangular
    if (phase & 1) {
    NAO_CUDA_CHECK(cudaMemsetAsync(d_info, 0, sizeof(int) * batch, st));

    // 1. factor (or unpack) S
    prof_mark(0, st);
    if (lowdin) {
        // the paper's route: S = U s U^H, W = s^{-1/2} U^H (dense); dS keeps W for the later SCF steps
        if (!(flags & NAO_S_FACTORED)) {
            if ((rc = herm_fill(p.sdtype, nS, dS, lds, strideS, X, nS, sW, p.nitemsS, st))) return rc;
            if ((rc = heev(p.sdtype, nS, p.nitemsS, flags, X, nS, sW, dE, A, nS, sW, w + p.heev, d_info, st))) return rc;
            if ((rc = lowdin_w(p.sdtype, nS, p.nitemsS, A, nS, sW, dE, g_lowdin_rel, W, nS, sW, d_info, st))) return rc;
            if ((rc = copy_matrix(p.sdtype, nS, nS, W, nS, sW, dS, lds, strideS, p.nitemsS, 0, st))) return rc;
        } else {
            if ((rc = copy_matrix(p.sdtype, nS, nS, dS, lds, strideS, W, nS, sW, p.nitemsS, 0, st))) return rc;
        }
    } else if (!(flags & NAO_S_FACTORED)) {
        // with a shared S the (single) status goes to d_info[0]
        if ((rc = potrf_trtri(p.sdtype, nS, p.nitemsS, dS, lds, strideS, W, nS, sW, X, nS, sW, d_info, st, A, (size_t)batch * n * n * es))) return rc;
        if ((rc = pack_linv(p.sdtype, nS, dS, lds, strideS, W, nS, sW, p.nitemsS, st))) return rc;
    } else {
        if ((rc = unpack_linv(p.sdtype, nS, dS, lds, strideS, W, nS, sW, p.nitemsS, st))) return rc;
    }
    prof_mark(1, st);
    // nao_solve_host: H arrives on another stream while S is factored
    if (h_ready) NAO_CUDA_CHECK(cudaStreamWaitEvent(st, h_ready, 0));
    }
    if (!nc) {
        if (phase & 1) {
        // 2. A = W H W^H : full Hermitian copy of H, X = W A (triangular W), A = X W^H (lower tiles)
        if ((rc = herm_fill(dtype, n, dH, ldh, strideH, A, n, sAX, batch, st))) return rc;
        {
            GemmDesc g = gemm_desc(OP_N, OP_N, n, n, n, 1.0, Wm, n, A, n, 0.0, X, n);
            g.sA = sWm; g.sB = sAX; g.sC = sAX; g.maskA = wmask;
            if ((rc = gemm_launch(dtype, g, batch, st))) return rc;
        }
        {
            GemmDesc g = gemm_desc(OP_N, OP_C, n, n, n, 1.0, X, n, Wm, n, 0.0, A, n);
            g.sA = sAX; g.sB = sWm; g.sC = sAX; g.maskB = wmask; g.cmode = 1;
            if ((rc = gemm_launch(dtype, g, batch, st))) return rc;
        }
        if (lowdin && (rc = lowdin_shift(dtype, n, nS, batch, A, n, sAX, Wm, p.sdtype, nS, sWm, NAO_PRUNED_LEVEL, st))) return rc;
        // 3. standard problem; eigenvectors into X
        if ((rc = heev(dtype, n, batch, flags, A, n, sAX, dE, X, n, sAX, w + p.heev, d_info, st, nvec, (phase & 2) ? 3 : 1))) return rc;
        }
        if (!(phase & 2)) return NAO_OK;
        if (!(phase & 1))
            if ((rc = heev(dtype, n, batch, flags, A, n, sAX, dE, X, n, sAX, w + p.heev, d_info, st, nvec, 2))) return rc;
        // 4. C = W^H Z
        GemmDesc g = gemm_desc(OP_C, OP_N, n, nvec, n, 1.0, Wm, n, X, n, 0.0, dC, ldc);
        g.sA = sWm; g.sB = sAX; g.sC = strideC; g.maskA = wmask;
        if ((rc = gemm_launch(dtype, g, batch, st))) return rc;
    } else {
        // Noncollinear: W_NC = diag(W, W) with W REAL (Eq. 25-27).  A complex matrix multiplied from the RIGHT by a real one is
        // a real GEMM on its interleaved (re, im) rows -- half the DMMA work of a complex product -- so both congruences are
        // arranged as right-multiplications:
        //   2. Y = H W_NC^T ;  A = W_NC H W_NC^T = (Y^H) W_NC^T          3. heev          4. C^H = Z^H W_NC
        // Real view of a complex (ld) matrix: double pointer, leading dimension 2 ld, row 2i / 2i+1 = re / im of row i.
        double *Ar = (double *)A, *Xr = (double *)X;
        const double *Wr = (const double *)W;
        if (phase & 1) {
        if ((rc = herm_fill(dtype, n, dH, ldh, strideH, A, n, sAX, batch, st))) return rc;
        for (int bj = 0; bj < 2; ++bj) {           // Y(:, block bj) = H(:, block bj) W^T
            const long off = 2 * (long)bj * nS * n;
            GemmDesc g = gemm_desc(OP_N, OP_T, 2 * n, nS, nS, 1.0, Ar + off, 2L * n, Wr, nS, 0.0, Xr + off, 2L * n);
            g.sA = 2 * sAX; g.sB = sWm; g.sC = 2 * sAX; g.maskB = wmask;
            if ((rc = gemm_launch(NAO_REAL, g, batch, st))) return rc;
        }
        if ((rc = conj_transpose(n, n, (const cplx *)X, n, sAX, (cplx *)A, n, sAX, batch, st))) return rc;       // A <- Y^H
        for (int bi = 0; bi < 2; ++bi)
            for (int bj = 0; bj <= bi; ++bj) {     // block (bi, bj) of (Y^H) W_NC^T, lower block triangle, into X
                const long off = 2 * ((long)bi * nS + (long)bj * nS * n);
                GemmDesc g = gemm_desc(OP_N, OP_T, 2 * nS, nS, nS, 1.0, Ar + off, 2L * n, Wr, nS, 0.0, Xr + off, 2L * n);
                g.sA = 2 * sAX; g.sB = sWm; g.sC = 2 * sAX; g.maskB = wmask; g.cmode = (bi == bj) ? 2 : 0;
                if ((rc = gemm_launch(NAO_REAL, g, batch, st))) return rc;
            }
        if ((rc = copy_matrix(dtype, n, n, X, n, sAX, A, n, sAX, batch, 1, st))) return rc;                      // lower triangle
        if (lowdin && (rc = lowdin_shift(dtype, n, nS, batch, A, n, sAX, Wm, p.sdtype, nS, sWm, NAO_PRUNED_LEVEL, st))) return rc;
        // 3. standard problem; eigenvectors into X
        if ((rc = heev(dtype, n, batch, flags, A, n, sAX, dE, X, n, sAX, w + p.heev, d_info, st, nvec, (phase & 2) ? 3 : 1))) return rc;
        }
        if (!(phase & 2)) return NAO_OK;
        if (!(phase & 1))
            if ((rc = heev(dtype, n, batch, flags, A, n, sAX, dE, X, n, sAX, w + p.heev, d_info, st, nvec, 2))) return rc;
        // 4. C = W_NC^T Z through C^H = Z^H W_NC  (Z^H in A as an nvec x n matrix, C^H in X)
        if ((rc = conj_transpose(n, nvec, (const cplx *)X, n, sAX, (cplx *)A, nvec, sAX, batch, st))) return rc;
        for (int bj = 0; bj < 2; ++bj) {
            const long off = 2 * (long)bj * nS * nvec;
            GemmDesc g = gemm_desc(OP_N, OP_N, 2 * nvec, nS, nS, 1.0, Ar + off, 2L * nvec, Wr, nS, 0.0, Xr + off, 2L * nvec);
            g.sA = 2 * sAX; g.sB = sWm; g.sC = 2 * sAX; g.maskB = wmask;
            if ((rc = gemm_launch(NAO_REAL, g, batch, st))) return rc;
        }
        if ((rc = conj_transpose(nvec, n, (const cplx *)X, nvec, sAX, (cplx *)dC, ldc, strideC, batch, st))) return rc;
    }
    prof_mark(8, st);
    // partial spectrum: the columns that were not back-transformed read as zero
    if (nvec < n)
        for (int b = 0; b < batch; ++b)
            if (ldc == n) {
                if ((rc = set_zero((char *)dC + ((size_t)b * strideC + (size_t)nvec * ldc) * es, (size_t)(n - nvec) * n * es, st))) return rc;
            } else {
                for (int j = nvec; j < n; ++j)
                    if ((rc = set_zero((char *)dC + ((size_t)b * strideC + (size_t)j * ldc) * es, (size_t)n * es, st))) return rc;
            }
    return NAO_OK;
}

// Concurrent mid-size solves (the paper's observation that several k-points sharing a GPU fill the gaps
// of one another): the batch is cut into `groups` contiguous groups, each of which runs the whole
// chain on its own internal stream (forked from and joined back into the caller's stream) with its own slice of the
// workspace.  The cooperative kernels of a group are sized for 1/groups of the SMs so that the groups are co-resident.
static int geneig_grouped(int n, int batch, int dtype, unsigned flags, int nvec, const void *dH, long ldh, long strideH, void *dS,
                          long lds, long strideS, double *dE, void *dC, long ldc, long strideC, void *dwork,
                          size_t work_bytes, int *d_info, void *cuda_stream) {
    using namespace nao;
    int groups = (n >= 1 && batch >= 1) ? stream_groups(flags, batch) : 1;
    flags &= ~NAO_STREAM_GROUPS_MASK;
    // one shared S that still has to be factored is written by every group: run the batch as one group
    if (strideS == 0 && !(flags & NAO_S_FACTORED)) groups = 1;
    if (groups <= 1)
        return geneig_impl(n, batch, dtype, flags, nvec, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, dwork, work_bytes,
                           d_info, cuda_stream);
    // argument check of the whole call first (phase 0: no launch)
    int rc = geneig_impl(n, batch, dtype, flags, nvec, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, dwork, (size_t)-1,
                         d_info, cuda_stream, 0);
    if (rc) return rc;
    if ((rc = bind_device())) return rc;
    static SideSet ss = {};
    if ((rc = side_set_init(ss, 8, 9, false))) return rc;
    cudaStream_t *side = ss.stream;
    const cudaEvent_t ev_fork = ss.event[8], *ev_join = ss.event;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t es = esize(dtype), esS = (flags & NAO_NC_BLOCK_S) ? 8 : es;
    set_sm_limit(sm_count() / groups);
    prof_suspend(true);                   // launches go to internal streams: the phase / kernel timers record nothing
    size_t off = 0;
    for (int g = 0; g < groups && rc == NAO_OK; ++g) {
        const int b0 = (int)((long)batch * g / groups), b1 = (int)((long)batch * (g + 1) / groups);
        off += align_up(ge_plan(n, b1 - b0, dtype, flags, strideS == 0).bytes);
    }
    if (off > work_bytes) { set_sm_limit(0); prof_suspend(false); return NAO_ERR_WORKSPACE; }
    if (cudaEventRecord(ev_fork, st) != cudaSuccess) { set_sm_limit(0); prof_suspend(false); return NAO_ERR_CUDA; }
    off = 0;
    int forked = 0;                        // groups whose internal stream has been given work
    for (int g = 0; g < groups; ++g) {
        const int b0 = (int)((long)batch * g / groups), b1 = (int)((long)batch * (g + 1) / groups), nb = b1 - b0;
        const size_t need = ge_plan(n, nb, dtype, flags, strideS == 0).bytes;
        if (cudaStreamWaitEvent(side[g], ev_fork, 0) != cudaSuccess) { rc = NAO_ERR_CUDA; break; }
        forked = g + 1;
        rc = geneig_impl(n, nb, dtype, flags, nvec, (const char *)dH + (size_t)b0 * strideH * es, ldh, strideH,
                         (char *)dS + (size_t)b0 * strideS * esS, lds, strideS, dE + (size_t)b0 * n,
                         (char *)dC + (size_t)b0 * strideC * es, ldc, strideC, (char *)dwork + off, need, d_info + b0, side[g]);
        if (rc) break;
        off += align_up(need);
        if (cudaEventRecord(ev_join[g], side[g]) != cudaSuccess || cudaStreamWaitEvent(st, ev_join[g], 0) != cudaSuccess) {
            rc = NAO_ERR_CUDA; break;
        }
    }
    set_sm_limit(0);
    prof_suspend(false);
    // error exit: whatever the groups already enqueued still runs against the caller's buffers -- order the caller's stream
    // behind all of it (on the success path every group was joined above)
    if (rc)
        for (int g = 0; g < forked; ++g)
            if (cudaEventRecord(ev_join[g], side[g]) == cudaSuccess) cudaStreamWaitEvent(st, ev_join[g], 0);
    return rc;
}

NAO_EXPORT int nao_geneig(int n, int batch, int dtype, unsigned flags, const void *dH, long ldh, long strideH, void *dS,
                          long lds, long strideS, double *dE, void *dC, long ldc, long strideC, void *dwork,
                          size_t work_bytes, int *d_info, void *cuda_stream) {
    return geneig_grouped(n, batch, dtype, flags, n, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, dwork, work_bytes,
                          d_info, cuda_stream);
}

NAO_EXPORT int nao_geneig_partial(int n, int batch, int dtype, unsigned flags, int n_vec, const void *dH, long ldh, long strideH,
                                  void *dS, long lds, long strideS, double *dE, void *dC, long ldc, long strideC, void *dwork,
                                  size_t work_bytes, int *d_info, void *cuda_stream) {
    if (n < 1) return -1;
    if (n_vec < 1 || n_vec > n) return -5;
    int rc = geneig_grouped(n, batch, dtype, flags, n_vec, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, dwork,
                            work_bytes, d_info, cuda_stream);
    return (rc <= -5) ? rc - 1 : rc;          // argument positions after n_vec are shifted by one
}

// ---------------------------------------------------------------------------------------------------------------------
// nao_scf_step: the whole hot path of one SCF step in one call -- eigenvalues, Fermi level, then only the eigenvectors the
// density matrix reads are back-transformed (count taken from the step's own occupations), then D.
// ---------------------------------------------------------------------------------------------------------------------
extern "C" int nao_fermi_workspace(int n, int batch, size_t *bytes);
extern "C" int nao_density_workspace(int n, int batch, int dtype, size_t *bytes);
extern "C" int nao_occupied_count(int n, int batch, const double *dF, double threshold, int *h_count, void *cuda_stream);
extern "C" int nao_density_matrix(int n, int batch, int dtype, const void *dC, long ldc, long strideC, const double *dF, void *dD,
                                  long ldd, long strideD, void *dwork, size_t work_bytes, void *cuda_stream);

// The fused step back-transforms only the occupied vectors, which favours the two-stage reduction for complex matrices as
// well; below order 1536 the one-stage path stays ahead (measured times of both: BASELINE.md section 5).
static unsigned scf_step_flags(int n, unsigned flags) {
    flags &= ~NAO_STREAM_GROUPS_MASK;          // the fused step runs as one group
    if (!(flags & (NAO_TRD_ONE_STAGE | NAO_TRD_TWO_STAGE)) && n >= nao::TWO_STAGE_MIN_N_REAL) flags |= NAO_TRD_TWO_STAGE;
    return flags;
}

// Host checks of the occupation arguments shared by nao_fermi_mu, nao_scf_step and nao_solve_host (made before any launch):
// every weight positive (else -arg_weight), 0 < n_electrons < sum_b w_b n and kT > 0 (else NAO_ERR_ELECTRONS).
int nao::check_occupation_args(int n, int batch, const double *h_weight, double n_electrons, double kT, int arg_weight) {
    if (!h_weight) return -arg_weight;
    double wsum = 0.0;
    for (int b = 0; b < batch; ++b) { if (!(h_weight[b] > 0.0)) return -arg_weight; wsum += h_weight[b] * n; }
    if (!(n_electrons > 0.0) || !(n_electrons < wsum) || !(kT > 0.0)) return NAO_ERR_ELECTRONS;
    return NAO_OK;
}

// argument positions of nao_geneig -> positions of nao_scf_step (negative return codes of the shared implementation)
static int scf_step_argpos(int rc) {
    switch (rc) {
        case -11: return -14;   // dE
        case -12: return -17;   // dC
        case -13: return -18;   // ldc
        case -14: return -19;   // strideC
        case -15: return -24;   // dwork
        case -17: return -26;   // d_info
        default: return rc;     // 1..10 coincide; positive codes pass through
    }
}

static int scf_step_workspace_raw(int n, int batch, int dtype, unsigned flags, size_t *bytes) {
    size_t g = 0, f = 0, d = 0;
    int rc;
    if ((rc = nao_geneig_workspace(n, batch, dtype, flags, &g))) return rc;
    if ((rc = nao_fermi_workspace(n, batch, &f))) return rc;
    if ((rc = nao_density_workspace(n, batch, dtype, &d))) return rc;
    *bytes = nao::align_up(g) + nao::align_up(f) + nao::align_up(d);
    return NAO_OK;
}

NAO_EXPORT int nao_scf_step_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes) {
    // covers both the flags as given (nao_solve_host: full solve) and the fused step's own choice of reduction
    size_t a = 0, b = 0;
    int rc = scf_step_workspace_raw(n, batch, dtype, flags, &a);
    if (rc) return rc;
    if ((rc = scf_step_workspace_raw(n, batch, dtype, scf_step_flags(n, flags), &b))) return rc;
    *bytes = a > b ? a : b;
    return NAO_OK;
}

NAO_EXPORT int nao_scf_step(int n, int batch, int dtype, unsigned flags, const void *dH, long ldh, long strideH, void *dS,
                            long lds, long strideS, const double *h_weight, double n_electrons, double kT, double *dE,
                            double *h_mu, double *dF, void *dC, long ldc, long strideC, void *dD, long ldd, long strideD,
                            int *h_nvec, void *dwork, size_t work_bytes, int *d_info, void *cuda_stream) {
    using namespace nao;
    flags = scf_step_flags(n, flags);
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (int rc0 = check_occupation_args(n, batch, h_weight, n_electrons, kT, 11)) return rc0;
    if (!h_mu) return -15;
    if (!dF) return -16;
    if (!dD) return -20;
    if (ldd < n) return -21;
    if (batch > 1 && strideD < ldd * (long)n) return -22;
    size_t g = 0, f = 0, d = 0, total = 0;
    int rc;
    if ((rc = nao_scf_step_workspace(n, batch, dtype, flags, &total))) return rc;
    if (work_bytes < total) return NAO_ERR_WORKSPACE;
    nao_geneig_workspace(n, batch, dtype, flags, &g); nao_fermi_workspace(n, batch, &f); nao_density_workspace(n, batch, dtype, &d);
    char *wg = (char *)dwork, *wf = wg + align_up(g), *wd = wf + align_up(f);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // eigenvalues (phase 1); argument errors of the shared implementation are renumbered to this signature
    rc = geneig_impl(n, batch, dtype, flags, n, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, wg, g, d_info, cuda_stream, 1);
    if (rc) return scf_step_argpos(rc);
    if ((rc = fermi_mu(n, batch, dE, h_weight, n_electrons, kT, h_mu, dF, wf, st))) return rc;
    int cnt = 0;
    if ((rc = nao_occupied_count(n, batch, dF, 1e-17, &cnt, cuda_stream))) return rc;
    int nvec = cnt + (cnt / 50 > 8 ? cnt / 50 : 8);          // margin: 2 %, at least 8 states (all of them have f < 1e-17)
    if (nvec > n) nvec = n;
    if (nvec < 1) nvec = 1;
    if (h_nvec) *h_nvec = nvec;
    rc = geneig_impl(n, batch, dtype, flags, nvec, dH, ldh, strideH, dS, lds, strideS, dE, dC, ldc, strideC, wg, g, d_info, cuda_stream, 2);
    if (rc) return rc;
    return nao_density_matrix(n, batch, dtype, dC, ldc, strideC, dF, dD, ldd, strideD, wd, d, cuda_stream);
}

// ---------------------------------------------------------------------------------------------------------------------
// nao_solve_host: the whole step with HOST inputs and outputs (nao.h).  H travels on an internal copy stream while S is
// factored on the caller's stream; D goes back item by item behind the density-matrix GEMM of the next item.
// ---------------------------------------------------------------------------------------------------------------------
namespace nao {
struct HostPlan { size_t H, S, E, F, C, D, info, work, wbytes, bytes; int nS, nitemsS; size_t esS; };
static int host_plan(int n, int batch, int dtype, unsigned flags, int shared_S, HostPlan &p) {
    size_t off = 0;
    auto take = [&](size_t b) { size_t o = off; off += align_up(b); return o; };
    const bool nc = flags & NAO_NC_BLOCK_S;
    const size_t es = esize(dtype);
    p.nS = nc ? n / 2 : n; p.esS = nc ? 8 : es; p.nitemsS = shared_S ? 1 : batch;
    p.H = take((size_t)batch * n * n * es);
    p.S = take((size_t)p.nitemsS * p.nS * p.nS * p.esS);
    p.E = take((size_t)batch * n * 8); p.F = take((size_t)batch * n * 8);
    p.C = take((size_t)batch * n * n * es); p.D = take((size_t)batch * n * n * es);
    p.info = take((size_t)batch * sizeof(int));
    int rc = nao_scf_step_workspace(n, batch, dtype, flags, &p.wbytes);
    if (rc) return rc;
    p.work = take(p.wbytes);
    p.bytes = off;
    return NAO_OK;
}
}  // namespace nao

NAO_EXPORT int nao_solve_host_workspace(int n, int batch, int dtype, unsigned flags, int shared_S, size_t *bytes) {
    if (!bytes) return -6;
    nao::HostPlan p;
    int rc = nao::host_plan(n, batch, dtype, flags, shared_S, p);
    if (rc) return rc;
    *bytes = p.bytes;
    return NAO_OK;
}

NAO_EXPORT int nao_solve_host(int n, int batch, int dtype, unsigned flags, const void *hH, const void *hS, int shared_S,
                              const double *h_weight, double n_electrons, double kT, double *hE, double *h_mu, void *hD,
                              int *h_info, void *dwork, size_t work_bytes, void *cuda_stream) {
    using namespace nao;
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -3;
    if ((flags & NAO_NC_BLOCK_S) && (dtype != NAO_COMPLEX || (n & 1))) return -4;
    if (flags & NAO_S_FACTORED) return -4;              // the factor lives in the device scratch: not kept between calls
    flags &= ~NAO_STREAM_GROUPS_MASK;
    if (!hH) return -5;
    if (!hS) return -6;
    if (int rc0 = check_occupation_args(n, batch, h_weight, n_electrons, kT, 8)) return rc0;
    if (!hE) return -11;
    if (!h_mu) return -12;
    if (!hD) return -13;
    if (!h_info) return -14;
    if (!dwork) return -15;
    HostPlan p;
    int rc = host_plan(n, batch, dtype, flags, shared_S, p);
    if (rc) return rc;
    if (work_bytes < p.bytes) return NAO_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = bind_device())) return rc;
    static SideSet ss = {};
    if ((rc = side_set_init(ss, 1, 5, false))) return rc;
    const cudaStream_t cs = ss.stream[0];
    const cudaEvent_t ev_start = ss.event[0], ev_h = ss.event[1], ev_d = ss.event[2], ev_end = ss.event[3];
    SideJoin join(cs, st, ss.event[4]);        // error exits: the caller's stream still ends behind the copy stream
    char *w = (char *)dwork;
    const size_t es = esize(dtype);
    const size_t item = (size_t)n * n * es;
    void *dH = w + p.H, *dS = w + p.S, *dC = w + p.C, *dD = w + p.D;
    double *dE = (double *)(w + p.E), *dF = (double *)(w + p.F);
    int *d_info = (int *)(w + p.info);
    // the copy stream starts behind whatever the caller's stream still does with the scratch
    NAO_CUDA_CHECK(cudaEventRecord(ev_start, st));
    NAO_CUDA_CHECK(cudaStreamWaitEvent(cs, ev_start, 0));
    join.arm();
    NAO_CUDA_CHECK(cudaMemcpyAsync(dS, hS, (size_t)p.nitemsS * p.nS * p.nS * p.esS, cudaMemcpyHostToDevice, st));
    NAO_CUDA_CHECK(cudaMemcpyAsync(dH, hH, (size_t)batch * item, cudaMemcpyHostToDevice, cs));
    NAO_CUDA_CHECK(cudaEventRecord(ev_h, cs));
    size_t g = 0, f = 0, d = 0;
    nao_geneig_workspace(n, batch, dtype, flags, &g); nao_fermi_workspace(n, batch, &f); nao_density_workspace(n, batch, dtype, &d);
    char *wg = w + p.work, *wf = wg + align_up(g), *wd = wf + align_up(f);
    rc = geneig_impl(n, batch, dtype, flags, n, dH, n, (long)n * n, dS, p.nS, shared_S ? 0 : (long)p.nS * p.nS, dE, dC, n, (long)n * n,
                     wg, g, d_info, cuda_stream, 3, ev_h);
    if (rc) return rc;
    if ((rc = fermi_mu(n, batch, dE, h_weight, n_electrons, kT, h_mu, dF, wf, st))) return rc;
    for (int b = 0; b < batch; ++b) {
        rc = nao_density_matrix(n, 1, dtype, (char *)dC + b * item, n, (long)n * n, dF + (size_t)b * n, (char *)dD + b * item, n,
                                (long)n * n, wd, d, cuda_stream);
        if (rc) return rc;
        NAO_CUDA_CHECK(cudaEventRecord(ev_d, st));
        NAO_CUDA_CHECK(cudaStreamWaitEvent(cs, ev_d, 0));
        NAO_CUDA_CHECK(cudaMemcpyAsync((char *)hD + b * item, (char *)dD + b * item, item, cudaMemcpyDeviceToHost, cs));
    }
    NAO_CUDA_CHECK(cudaMemcpyAsync(hE, dE, (size_t)batch * n * 8, cudaMemcpyDeviceToHost, st));
    NAO_CUDA_CHECK(cudaMemcpyAsync(h_info, d_info, (size_t)batch * sizeof(int), cudaMemcpyDeviceToHost, st));
    // the caller's stream finishes behind the last copy: synchronising it is enough
    NAO_CUDA_CHECK(cudaEventRecord(ev_end, cs));
    NAO_CUDA_CHECK(cudaStreamWaitEvent(st, ev_end, 0));
    return NAO_OK;
}

NAO_EXPORT int nao_set_lowdin_threshold(double rel) {
    if (!(rel >= 0.0 && rel < 1.0)) return -1;
    nao::g_lowdin_rel = rel;
    return NAO_OK;
}
