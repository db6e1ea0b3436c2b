// nao_internal.cuh -- shared declarations of the sm_100a kernels behind include/nao.h.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "../../include/nao.h"

#define NAO_EXPORT extern "C" __attribute__((visibility("default")))

namespace nao {

typedef double2 cplx;   // interleaved complex FP64 (x = re, y = im)

// ---------------------------------------------------------------------------------------------------------
// launch bookkeeping
// ---------------------------------------------------------------------------------------------------------
extern long g_launch_count;          // host-side count of kernel launches (nao_launch_count)
// SMs the cooperative (grid-barrier) kernels of the current call may occupy: the device's SM count, or less while a
// stream group of nao_geneig (NAO_STREAM_GROUPS_*) is being enqueued, so that the groups' cooperative kernels are
// co-resident on disjoint SMs instead of waiting for one another.
int sm_count();
void set_sm_limit(int limit);        // 0 = no limit
// The library's process-wide state belongs to one device (include/nao.h).  bind_device(): records the current device on the
// first call, afterwards NAO_ERR_CUDA when another device is current -- called by every entry point after its host-side
// argument checks and before its first launch.  device_sms(): SM count of that device (cached).
int bind_device();
int device_sms();
// Internal streams and events of one call site, created together: all of them exist afterwards, or none (ready stays false).
struct SideSet {
    enum { MAX_STREAMS = 8, MAX_EVENTS = 10 };
    cudaStream_t stream[MAX_STREAMS]; cudaEvent_t event[MAX_EVENTS]; bool ready;
};
int side_set_init(SideSet &s, int nstreams, int nevents, bool high_priority);
// Scope guard of a function that forks work onto an internal stream: once armed, leaving the scope -- by ANY return, error
// exits included -- orders the caller's stream behind everything enqueued on the internal stream so far, so that no kernel
// is still running against the caller's buffers on a stream the caller cannot see.
struct SideJoin {
    cudaStream_t side, st; cudaEvent_t ev; bool armed;
    SideJoin(cudaStream_t side_, cudaStream_t st_, cudaEvent_t ev_) : side(side_), st(st_), ev(ev_), armed(false) {}
    void arm() { armed = true; }
    ~SideJoin() { if (armed && cudaEventRecord(ev, side) == cudaSuccess) cudaStreamWaitEvent(st, ev, 0); }
};
#define NAO_LAUNCHED() (++::nao::g_launch_count)

#define NAO_CUDA_CHECK(expr)                                        \
    do {                                                            \
        cudaError_t e__ = (expr);                                   \
        if (e__ != cudaSuccess) return NAO_ERR_CUDA;                \
    } while (0)

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
static inline int ceil_div(int a, int b) { return (a + b - 1) / b; }
static inline size_t esize(int dtype) { return dtype == NAO_COMPLEX ? 16 : 8; }

// bump allocator over the caller's workspace
struct Arena {
    char *base; size_t cap; size_t off;
    Arena(void *p, size_t c) : base((char *)p), cap(c), off(0) {}
    void *take(size_t bytes) {
        size_t o = off; off += align_up(bytes);
        return (off <= cap) ? (void *)(base + o) : nullptr;
    }
    template <class T> T *get(size_t count) { return (T *)take(count * sizeof(T)); }
};

// ---------------------------------------------------------------------------------------------------------
// DMMA GEMM (gemm.cu)
// ---------------------------------------------------------------------------------------------------------
enum { OP_N = 0, OP_T = 1, OP_C = 2 };
// triangular masks on the STORED operand, coordinates (r, c):  keep the element iff (r - c + off) REL 0
enum { MASK_NONE = 0, MASK_LOWER = 1 /* >= */, MASK_SLOWER = 2 /* > */, MASK_UPPER = 3 /* <= */, MASK_SUPPER = 4 /* < */ };

struct GemmDesc {
    const void *A; const void *B; void *C;
    long lda, ldb, ldc;
    long sA, sB, sC;          // batch strides (elements)
    int m, n, k;              // product dimensions: C (m x n) = op(A) (m x k) * op(B) (k x n)
    int opA, opB;
    int maskA, offA, maskB, offB;
    int cmode;                // 0 full; 1 = skip tiles entirely above the diagonal of C; 2 = the same for a complex matrix
                              // addressed as a real one with interleaved (re, im) rows (row 2i, 2i+1 <-> complex row i)
    int conjC;                // unused (reserved)
    double alpha, beta;
    const double *scaleK;     // optional: op(A)[:,k] is multiplied by scaleK[k]
    long sScale;              // batch stride of scaleK
    int ksplit;               // > 1: the k range is cut into ksplit slices, slice s writes C + s * sSplit (grid.y = batch * ksplit)
    long sSplit;
};

static inline GemmDesc gemm_desc(int opA, int opB, int m, int n, int k, double alpha, const void *A, long lda,
                                 const void *B, long ldb, double beta, void *C, long ldc) {
    GemmDesc d;
    d.A = A; d.B = B; d.C = C; d.lda = lda; d.ldb = ldb; d.ldc = ldc; d.sA = d.sB = d.sC = 0;
    d.m = m; d.n = n; d.k = k; d.opA = opA; d.opB = opB; d.maskA = d.maskB = MASK_NONE; d.offA = d.offB = 0;
    d.cmode = 0; d.conjC = 0; d.alpha = alpha; d.beta = beta; d.scaleK = nullptr; d.sScale = 0; d.ksplit = 1; d.sSplit = 0;
    return d;
}

// Split-K factor that fills the last wave: the GEMM core runs one CTA per SM (255 registers), so `tiles * ks` CTAs take
// ceil(tiles * ks / nsm) rounds; the factor (<= ksmax) with the best fill, a small penalty per extra slice, is returned.
static inline int fill_ksplit(long tiles, int nsm, int ksmax) {
    int best_ks = 1; double best = 0.0;
    for (int ks = 1; ks <= (ksmax < 1 ? 1 : ksmax); ++ks) {
        const double waves = (double)tiles * ks / nsm;
        const double rounds = (double)(long)(waves + 0.999999), eff = waves / rounds - 0.004 * (ks - 1);
        if (eff > best + 1e-9) { best = eff; best_ks = ks; }
    }
    return best_ks;
}

// One problem described on the host (passed by value), `batch` items via the strides in the descriptor.
int gemm_launch(int dtype, const GemmDesc &d, int batch, cudaStream_t st);
// `ngroups` problems described by descriptors in DEVICE memory (their m,n,k may have been written by a kernel);
// max_m/max_n bound the grid.  Each group runs `batch` items.  opA/opB/scale (shared by every descriptor) select the
// kernel instantiation.
// Split-K product for short-and-wide outputs (m, n small, k long): `ksplit` slices write partial products into
// `partial` (batch * ksplit * m * n elements), then C <- alpha * (sum of slices, fixed order) + beta * C.
int gemm_splitk(int dtype, const GemmDesc &d, int batch, int ksplit, void *partial, cudaStream_t st);
int gemm_launch_grouped(int dtype, const GemmDesc *d_descs, int ngroups, int max_m, int max_n, int batch, int opA,
                        int opB, bool scale, cudaStream_t st);

// ---------------------------------------------------------------------------------------------------------
// element-wise helpers (util.cu)
// ---------------------------------------------------------------------------------------------------------
// B <- A for the m x n block (both column-major); uplo: 0 all, 1 lower only (i >= j), 2 strict upper only
int copy_matrix(int dtype, int m, int n, const void *A, long lda, long sA, void *B, long ldb, long sB, int batch,
                int uplo, cudaStream_t st);
// B (full) <- Hermitian completion of the lower triangle of A (B may equal A: in-place mirror)
int herm_fill(int dtype, int n, const void *A, long lda, long sA, void *B, long ldb, long sB, int batch,
              cudaStream_t st);
int set_zero(void *p, size_t bytes, cudaStream_t st);
// real n x n (ldq) -> complex n x n (ldz)
int real_to_complex(int m, int n, const double *Q, long ldq, long sQ, cplx *Z, long ldz, long sZ, int batch,
                    cudaStream_t st);
// B (n x m) <- A^H, complex
int conj_transpose(int m, int n, const cplx *A, long lda, long sA, cplx *B, long ldb, long sB, int batch, cudaStream_t st);
// lowdin.cu: W = s^{-1/2} U^H with pruning of s_i <= rel * s_max; diagonal shift of the pruned directions of the reduced matrix
int lowdin_w(int dtype, int n, int batch, const void *U, long ldu, long sU, const double *s, double rel, void *W, long ldw,
             long sW, int *d_info, cudaStream_t st);
int lowdin_shift(int dtype, int n, int nS, int batch, void *A, long lda, long sA, const void *W, int wdtype, long ldw, long sW,
                 double big, cudaStream_t st);
// Linv (n x n lower, explicit zeros above, diagonal = 1/L_ii) from the packed factor in S (see nao.h)
int unpack_linv(int dtype, int n, const void *S, long lds, long sS, void *W, long ldw, long sW, int batch,
                cudaStream_t st);
int pack_linv(int dtype, int n, void *S, long lds, long sS, const void *W, long ldw, long sW, int batch,
              cudaStream_t st);

// ---------------------------------------------------------------------------------------------------------
// phases
// ---------------------------------------------------------------------------------------------------------
// chol.cu: S -> L (in S lower), W <- L^{-1}; T = n*n scratch.  info[b] = 0 or failing pivot (1-based)
int potrf_trtri(int dtype, int n, int batch, void *S, long lds, long sS, void *W, long ldw, long sW, void *T,
                long ldt, long sT, int *d_info, cudaStream_t st, void *scratch = nullptr, size_t scratch_bytes = 0);

// trd1.cu: one-stage Householder tridiagonalisation of the lower triangle of A (n x n); reflectors left below the
// first sub-diagonal of A (LAPACK xHETRD lower convention), d[n], e[n-1] real, tau[n-1].
size_t hetrd_workspace(int dtype, int n, int batch);
int hetrd(int dtype, int n, int batch, void *A, long lda, long sA, double *d, double *e, void *tau, void *work,
          cudaStream_t st);
// Z <- Q_house * Z where Q_house = H_0 H_1 ... H_{n-2} from hetrd (Z n x ncols)
size_t ormtr_workspace(int dtype, int n, int batch);
// shift = 1: reflectors of hetrd (v_j = A[j+1:, j]);  shift = b: reflectors of he2hb (v_j = A[j+b:, j])
int ormtr(int dtype, int n, int ncols, int batch, int shift, const void *A, long lda, long sA, const void *tau, void *Z,
          long ldz, long sZ, void *work, cudaStream_t st);
// ormtr.cu helpers shared with trd2.cu: explicit V block and the T factor from G = V^H V and tau
int build_v(int dtype, int n, int jb, int kb, int shift, const void *A, long lda, long sA, void *V, long ldv, long sV, int batch,
            cudaStream_t st);
int larft(int dtype, int kb, const void *G, long ldg, long sG, const void *tau, long sTau, void *Tm, long sT, int batch,
          cudaStream_t st);   // Tm is kb x kb dense (ld = kb), kb <= 128

// two-stage tridiagonalisation (trd2.cu, trd2_chase.cu, trd2_back.cu), bandwidth TRD2_B
static const int TRD2_B = 64;
// dense -> band: band in the lower part of A (0 <= i-j <= b), reflectors below it (v_j = A[j+b:, j], unit implicit), tau[n]
size_t he2hb_workspace(int dtype, int n, int batch);
bool he2hb_supported(int dtype, int n, int batch);
int he2hb(int dtype, int n, int batch, void *A, long lda, long sA, void *tau, void *work, cudaStream_t st);
// band -> tridiagonal by bulge chasing: reads the band from A, writes d[n], e[n] (real), reflectors V2 (n x n, ldv),
// tau2 (hb2st_nk(n) x n)
size_t hb2st_workspace(int dtype, int n, int batch);
int hb2st_nk(int n);
int hb2st(int dtype, int n, int batch, const void *A, long lda, long sA, double *d, double *e, void *V2, long ldv, long sV2,
          void *tau2, void *work, cudaStream_t st);
// Z <- Q2 Z (Z n x ncols) with the reflectors of hb2st
size_t q2_workspace(int dtype, int n, int batch);
int q2_apply(int dtype, int n, int ncols, int batch, const void *V2, long ldv, long sV2, const void *tau2, void *Z, long ldz,
             long sZ, void *work, cudaStream_t st);

// stedc.cu
size_t stedc_workspace(int n, int batch);
// nvec: eigenvectors wanted (the nvec lowest); phase 1 = eigenvalues, 2 = eigenvectors (continues a phase-1 call), 3 = both
int stedc(int n, int batch, double *d, double *e, double *evals, double *Q, long ldq, long sQ, void *work,
          int *d_info, cudaStream_t st, int nvec = -1, int phase = 3);

// api.cu: phase-boundary event (no-op unless nao_profile_enable(1))
void prof_mark(int idx, cudaStream_t st);
// on: nothing is recorded until prof_suspend(false) (used around a call that runs as stream groups)
void prof_suspend(bool on);
// per-launch timers: slot 0 = hetrd_panel_kernel (work = algorithmic HBM bytes), slot 1 = gemm_kernel (work = flops)
int prof_kernel_begin(int slot, double work, cudaStream_t st);
void prof_kernel_end(int slot, int k, cudaStream_t st);
// grouped GEMM launches: executed flops = per_mnk * sum over the device descriptors of m n k (counted by a kernel)
void prof_grouped_flops(const GemmDesc *d_descs, int ngroups, double per_mnk, cudaStream_t st);

// fermi.cu / density
int fermi_mu(int n, int batch, const double *dE, const double *h_weight, double n_electrons, double kT, double *h_mu,
             double *dF, void *dwork, cudaStream_t st);
// geneig.cu: host checks of (weights, n_electrons, kT); -arg_weight, NAO_ERR_ELECTRONS or NAO_OK
int check_occupation_args(int n, int batch, const double *h_weight, double n_electrons, double kT, int arg_weight);

}  // namespace nao
