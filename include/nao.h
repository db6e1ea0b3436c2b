/*
 * nao.h -- C-ABI boundary of the B200-native (sm_100a) generalized eigensolver + density-matrix library.
 *
 * The path (paper = /root/reference/PAPER.md, arxiv/paper_2606_09058):
 *   nao_geneig          H C = S C diag(e)              Eq. 5, per k-point Eq. 11,
 *                                                      noncollinear 2N x 2N form Eq. 21/25-27 (PAPER.md:113-115,
 *                                                      175-179); the paper's "Part 2" (section 3.1,
 *                                                      PAPER.md:157-163) / "Part 3" (section 3.2)
 *   nao_fermi_mu        sum g w_k f((e-mu)/kT) = N_e   Fermi-Dirac occupation (after Eq. 3); the
 *                                                      paper's "Part 3"/"Part 4"
 *   nao_density_matrix  D = C diag(f) C^H              Eq. 8 / Eq. 23; the paper's
 *                                                      "Part 4"/"Part 5"
 *
 * Conventions common to every entry point
 *   - All matrix/vector pointers are DEVICE pointers unless the name starts with h_ (host).
 *   - Matrices are column-major with a leading dimension in ELEMENTS (LAPACK convention); element (i,j) of item b
 *     is at  base + b*stride + j*ld + i.  dtype NAO_REAL = double, NAO_COMPLEX = interleaved (re,im) doubles.
 *   - The library allocates NO device memory: the caller owns every buffer, the workspace and the stream.
 *     `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work is enqueued on
 *     that stream and the call returns; the only calls that synchronise it are the ones that hand a host scalar
 *     back: nao_fermi_mu (*h_mu), nao_occupied_count (*h_count), and therefore nao_scf_step and nao_solve_host
 *     (stated at each).  nao_geneig, nao_geneig_partial, nao_heev, nao_stedc, nao_density_matrix, nao_fold_density
 *     never block the host (the divide-and-conquer tree is built by a kernel, not copied from the host).
 *   - Process-wide state: the library keeps per-process settings and caches (nao_set_lowdin_threshold, the profiler,
 *     kernel attributes, SM count, the internal side streams and events of nao_solve_host, of the stream groups and of the
 *     dense-to-band look-ahead, pinned result words) bound to the FIRST device it
 *     is used on.  Use it from one host thread at a time and on one device per process (one process per GPU is the
 *     deployment model); the Python binding rejects tensors on any other device.
 *   - Return value: NAO_OK (0); -i if argument number i (1-based) is invalid (checked on the host before any
 *     launch); a positive NAO_ERR_* code for run-time failures.  Numerical outcomes are reported per batch item
 *     in d_info (device int[batch]).
 *   - There is no CPU fallback anywhere: every step runs in CUDA kernels of this library.
 */
#ifndef NAO_H
#define NAO_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* dtype */
#define NAO_REAL 0
#define NAO_COMPLEX 1

/* flags for nao_geneig / nao_geneig_workspace */
#define NAO_S_FACTORED 1u      /* dS already holds the factor written by an earlier nao_geneig call on the same S
                                  (S and V = its orthogonaliser do not change during the SCF loop) */
#define NAO_NC_BLOCK_S 2u      /* noncollinear fast path: n = 2N, dtype = NAO_COMPLEX, basis spin-major [alpha;beta]
                                  (Eq. 25-27); dS is the N x N REAL overlap (S_NC = diag(S,S)) */
/* Without either of the next two flags the library picks the reduction: two-stage for real matrices of order >= 1536,
   one-stage otherwise (measured crossover on B200, reading T1). */
#define NAO_TRD_ONE_STAGE 4u   /* force the one-stage (HEMV-based, HBM-bound) Householder tridiagonalisation */
#define NAO_TRD_TWO_STAGE 8u   /* force the two-stage (dense->band->tridiagonal) reduction */
#define NAO_LOWDIN 16u         /* orthogonalise by the paper's own route: S = U s U^H with this
                                  library's eigensolver, V = U s^{-1/2}, H' = V^H H V, C = V C'.  Same e, mu, D as the
                                  default Cholesky route.  dS is overwritten by the DENSE matrix V^H = s^{-1/2} U^H (all of
                                  it, not just a triangle); NAO_S_FACTORED | NAO_LOWDIN reuses it.  Directions with
                                  s_i <= rel * s_max (rel set by nao_set_lowdin_threshold, default 0 = none) are pruned:
                                  their levels come out as NAO_PRUNED_LEVEL at the top of the spectrum with zero vectors,
                                  so that mu and D are those of the pruned basis.  With rel = 0 a non-positive eigenvalue
                                  of S sets d_info = (order of S) + 2. */
#define NAO_PRUNED_LEVEL 1.0e4 /* Hartree; eigenvalue reported for a pruned direction */
/* Concurrent mid-size solves: nao_geneig / nao_geneig_partial cut the batch into
   2, 4 or 8 contiguous groups that run the whole chain on internal streams, forked from and joined back into cuda_stream,
   each with its own slice of the workspace (nao_geneig_workspace accounts for it when given the same flags) and with its
   grid-barrier kernels sized for its share of the SMs.  Same results as the single batched call.  Ignored (one group) when
   the batch is smaller than the group count, when one shared S (strideS = 0) still has to be factored, and by
   nao_scf_step / nao_solve_host.  Without these flags every kernel of the chain is launched once for the whole batch --
   on B200 that is the faster arrangement for config 1 (f3). */
#define NAO_STREAM_GROUPS_2 32u
#define NAO_STREAM_GROUPS_4 64u
#define NAO_STREAM_GROUPS_8 96u
#define NAO_STREAM_GROUPS_MASK 96u

/* return codes */
#define NAO_OK 0
#define NAO_ERR_WORKSPACE 1    /* work_bytes smaller than nao_geneig_workspace / nao_density_workspace reports */
#define NAO_ERR_CUDA 2         /* a CUDA runtime call or kernel launch failed */
#define NAO_ERR_ELECTRONS 3    /* nao_fermi_mu: n_electrons outside (0, sum of weights * n) or kT <= 0 */
#define NAO_ERR_UNSUPPORTED 4  /* combination of arguments not implemented */
#define NAO_ERR_STATIC_LIMIT 5 /* nao_fermi_mu_static: n * batch exceeds NAO_FERMI_STATIC_MAX_STATES */

/* Relative pruning threshold of the NAO_LOWDIN route, 0 <= rel < 1 (process-wide, read when S is decomposed). */
int nao_set_lowdin_threshold(double rel);

/* Bytes of device workspace nao_geneig needs for (n, batch, dtype, flags).  Host-only, no launch. */
int nao_geneig_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes);

/*
 * Generalized Hermitian-definite eigenproblem, all eigenpairs, batched over (spin, k) items.
 *   1 n        order of H (2N with NAO_NC_BLOCK_S), n >= 1
 *   2 batch    number of independent (H,S) items, >= 1
 *   3 dtype    NAO_REAL or NAO_COMPLEX
 *   4 flags    OR of NAO_* flags above
 *   5 dH,ldh,strideH   in : Hermitian H; ONLY the lower triangle (i >= j) is referenced.  Not modified.
 *   8 dS,lds,strideS   in : Hermitian positive definite S, lower triangle referenced (with NAO_NC_BLOCK_S:
 *                           real, order n/2).  strideS == 0: ONE overlap matrix shared by all batch items (the spin
 *                           channels of a collinear calculation share S): it is factored once and d_info[0] carries
 *                           its status.
 *                      out: lower triangle = Cholesky factor L (S = L L^H); strict upper triangle = strict upper
 *                           triangle of L^{-H} (kept so that a later call with NAO_S_FACTORED skips both the
 *                           factorisation and the inversion).  With NAO_S_FACTORED: read only.
 *  11 dE       out: batch*n eigenvalues, ascending within each item (item b at dE + b*n)
 *  12 dC,ldc,strideC   out: eigenvectors as columns, normalised so that C^H S C = I.  Phases/signs and the basis
 *                           inside degenerate clusters are unspecified (compare e, mu, f, D, not C).
 *  15 dwork,work_bytes  device scratch of at least nao_geneig_workspace() bytes, 256-byte aligned
 *  17 d_info   out: device int[batch]; 0 = ok; j in 1..n: leading minor j of S not positive definite (LAPACK
 *                   potrf convention; the item's e and C are then undefined); n+1 = the tridiagonal
 *                   divide-and-conquer secular solver failed to converge.
 *  18 cuda_stream
 */
int nao_geneig(int n, int batch, int dtype, unsigned flags,
               const void *dH, long ldh, long strideH,
               void *dS, long lds, long strideS,
               double *dE,
               void *dC, long ldc, long strideC,
               void *dwork, size_t work_bytes, int *d_info, void *cuda_stream);

/*
 * Partial-spectrum variant (the paper notes that only the occupied quarter to half of the spectrum is
 * needed and that its cuSOLVER route cannot exploit this).  Identical to nao_geneig except that only the
 * eigenvectors of the n_vec LOWEST eigenvalues are back-transformed: all n eigenvalues are still written to dE, columns
 * 0..n_vec-1 of every item of dC are written, columns n_vec.. are set to zero.  The density matrix built from these
 * vectors equals the one of the full solve as long as every state with f >= 1e-17 lies below n_vec -- check with
 * nao_occupied_count after nao_fermi_mu (an SCF loop takes n_vec from the previous step plus a margin).
 * Combine with NAO_TRD_TWO_STAGE: with few vectors the second back-transformation of the two-stage reduction is cheap and
 * that path is the faster one at configs 2 and 3 (measured times: BASELINE.md section 5).
 *   1..4 as nao_geneig;  5 n_vec in 1..n;  the remaining arguments as nao_geneig arguments 5..18.
 * Negative return values count the arguments of THIS signature.
 */
int nao_geneig_partial(int n, int batch, int dtype, unsigned flags, int n_vec,
                       const void *dH, long ldh, long strideH,
                       void *dS, long lds, long strideS,
                       double *dE,
                       void *dC, long ldc, long strideC,
                       void *dwork, size_t work_bytes, int *d_info, void *cuda_stream);

/*
 * One SCF step of the hot path in one call (the paper's Parts 2-4 / 3-5): eigenvalues of the
 * pencil, Fermi level and occupations, back-transformation of ONLY the eigenvectors whose occupation is >= 1e-17 (their
 * number, plus a margin of 2 %, is returned in *h_nvec), D = C diag(f) C^H.  dE, *h_mu, dF and dD equal the results of
 * nao_geneig + nao_fermi_mu + nao_density_matrix; dC holds the first *h_nvec eigenvectors, its other columns are zero.
 * Arguments as in those three calls (h_weight, h_mu, h_nvec are HOST pointers); dwork needs nao_scf_step_workspace bytes.
 * The call synchronises the stream twice (Fermi level, vector count).
 * Without NAO_TRD_ONE_STAGE / NAO_TRD_TWO_STAGE the fused step takes the two-stage reduction from order 1536 on for real AND
 * complex matrices (few vectors are back-transformed, which favours it; measured times: BASELINE.md section 5).
 */
int nao_scf_step_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes);
int nao_scf_step(int n, int batch, int dtype, unsigned flags,
                 const void *dH, long ldh, long strideH, void *dS, long lds, long strideS,
                 const double *h_weight, double n_electrons, double kT,
                 double *dE, double *h_mu, double *dF,
                 void *dC, long ldc, long strideC, void *dD, long ldd, long strideD,
                 int *h_nvec, void *dwork, size_t work_bytes, int *d_info, void *cuda_stream);

/*
 * The same step (nao_geneig, all eigenpairs + nao_fermi_mu + nao_density_matrix) with HOST inputs and outputs: the
 * end-to-end form of the metric.  hH (batch matrices, n x n, column-major, contiguous), hS (batch matrices, or ONE when
 * shared_S != 0; order n/2 and real with NAO_NC_BLOCK_S) are copied to the device scratch, hE (batch*n), hD (batch matrices),
 * h_info (batch ints) and *h_mu are written back.  Pinned host memory makes the copies asynchronous: H travels on an internal
 * copy stream while S is factored on the caller's stream, and D returns item by item behind the density-matrix product of
 * the next item.  The call synchronises the stream once (Fermi level); when it returns the remaining copies are enqueued
 * and the caller's stream is ordered behind them -- synchronise it before reading hE, hD, h_info.
 *   1 n, 2 batch, 3 dtype, 4 flags (NAO_S_FACTORED is rejected: the factor lives in the scratch)
 *   5 hH, 6 hS, 7 shared_S, 8 h_weight (HOST double[batch]), 9 n_electrons, 10 kT
 *  11 hE, 12 h_mu, 13 hD, 14 h_info
 *  15 dwork, work_bytes  device scratch of at least nao_solve_host_workspace() bytes
 *  17 cuda_stream
 * Not re-entrant (one internal copy stream per process).
 */
int nao_solve_host_workspace(int n, int batch, int dtype, unsigned flags, int shared_S, size_t *bytes);
int nao_solve_host(int n, int batch, int dtype, unsigned flags,
                   const void *hH, const void *hS, int shared_S,
                   const double *h_weight, double n_electrons, double kT,
                   double *hE, double *h_mu, void *hD, int *h_info,
                   void *dwork, size_t work_bytes, void *cuda_stream);

/*
 * 1 + the largest level index i (over all batch items) with dF[b*n + i] >= threshold: the number of leading
 * eigenvectors nao_density_matrix reads.  Synchronises the stream to write *h_count (HOST int).
 */
int nao_occupied_count(int n, int batch, const double *dF, double threshold, int *h_count, void *cuda_stream);

/*
 * Fermi level and occupations (reading C5).  States are all (item b, level i) pairs; state weight is
 * h_weight[b] (= spin degeneracy g times k-point weight w_k, reading C4).  Finds the unique mu with
 *     sum_b h_weight[b] * sum_i f_bi = n_electrons,   f_bi = 1/(1 + exp((e_bi - mu)/kT)),
 * solved in particle/hole form so that mu is resolved inside a gap.
 *   1 n, 2 batch
 *   3 dE        in : device, batch*n eigenvalues (any order)
 *   4 h_weight  in : HOST double[batch]
 *   5 n_electrons, 6 kT (Hartree, > 0)
 *   7 h_mu      out: HOST double, the Fermi level (the call synchronises the stream to write it)
 *   8 dF        out: device, batch*n occupations f in [0,1]
 *   9 dwork     device scratch of at least nao_fermi_workspace(n, batch) bytes
 *  10 cuda_stream
 */
int nao_fermi_workspace(int n, int batch, size_t *bytes);
int nao_fermi_mu(int n, int batch, const double *dE, const double *h_weight,
                 double n_electrons, double kT, double *h_mu, double *dF,
                 void *dwork, void *cuda_stream);

/*
 * nao_fermi_mu for callers that cannot supply device scratch and must not cause a device allocation.
 *
 * Who that is: code that runs inside a host program which owns all device memory itself -- an SCF code that carves the
 * whole HBM into its own pool at start-up and forbids any later driver allocation, a plug-in that is only handed its input
 * and output arrays, or a call made from a latency-critical section where cudaMalloc / cudaFree are unacceptable because
 * they take the driver's global lock and synchronise the whole device (stalling the host program's other streams).  Such a
 * caller has no `dwork` to pass either, so this entry point has no workspace argument: it keeps its intermediates (the
 * sorted energies and their weights, the per-item weights, the device copy of mu) in a fixed array that is compiled into
 * the library, and it calls neither cudaMalloc nor cudaFree nor any routine that allocates.
 *
 * Same arguments, same result (mu, dF) and same error codes as nao_fermi_mu, without its argument 9:
 *   1 n, 2 batch, 3 dE, 4 h_weight (HOST), 5 n_electrons, 6 kT, 7 h_mu (HOST, out), 8 dF (out), 9 cuda_stream
 * The caller still owns dE and dF.  Like nao_fermi_mu it synchronises the stream to write *h_mu.
 *
 * Limit: n * batch <= NAO_FERMI_STATIC_MAX_STATES (65536 states: every configuration of BASELINE.json fits, config 4 has
 * 26624).  Anything larger returns NAO_ERR_STATIC_LIMIT before the device is touched; use nao_fermi_mu with your own
 * workspace then.
 * Cost: the array is NAO_FERMI_STATIC_BYTES = 1.5 MiB of device memory on EVERY GPU that loads this library's kernels, held
 * until the process exits, also when this entry point is never called.
 * Sharing: all calls on a device use the same array.  It keeps whatever the last call wrote; that is harmless because a
 * call writes every word before it reads it (nothing relies on zeros).  But two calls that are in flight on the GPU at the
 * same time -- different streams or host threads -- overwrite each other's intermediates: serialise them.
 * Set-up: the first call made with a given device current looks up the array's address on that device (one
 * cudaGetSymbolAddress; the library remembers it per device ordinal, 64 at most).  Make that first call outside any
 * stream capture.
 */
#define NAO_FERMI_STATIC_MAX_STATES 65536
#define NAO_FERMI_STATIC_BYTES (3 * NAO_FERMI_STATIC_MAX_STATES * 8 + 256)
int nao_fermi_mu_static(int n, int batch, const double *dE, const double *h_weight,
                        double n_electrons, double kT, double *h_mu, double *dF, void *cuda_stream);

/*
 * Density matrix D_b = C_b diag(f_b) C_b^H per batch item, full Hermitian matrix written (both triangles).
 * Columns after the last one with |f| >= 1e-17 are skipped (their contribution is < 1e-17 * |C|^2, reading C6).
 *   1 n, 2 batch, 3 dtype
 *   4 dC,ldc,strideC  in : eigenvectors (columns)
 *   7 dF              in : device, batch*n weights (occupations f in [0,1]; any real values are allowed, e.g. the f*e of
 *                          nao_energy_weights gives the energy-weighted density matrix)
 *   8 dD,ldd,strideD  out
 *  11 dwork, work_bytes  device scratch of at least nao_density_workspace() bytes
 *  13 cuda_stream
 */
int nao_density_workspace(int n, int batch, int dtype, size_t *bytes);
int nao_density_matrix(int n, int batch, int dtype,
                       const void *dC, long ldc, long strideC,
                       const double *dF,
                       void *dD, long ldd, long strideD,
                       void *dwork, size_t work_bytes, void *cuda_stream);

/*
 * The step after the hot path (the paper's un-offloaded Part 4/5).
 *
 * nao_energy_weights: dFE[b*n + i] = dF[b*n + i] * dE[b*n + i] (device arrays of batch*n doubles).  Passing dFE as the
 * weights of nao_density_matrix gives the energy-weighted density matrix C diag(f e) C^H.
 *
 * nao_fold_density: real-space density matrix from its k-space images, the inverse of the Bloch sum of Eq. 12
 * (sign convention DESIGN.md reading C8):
 *     D(R_r) = sum_k h_w[k] * exp(-i k.R_r) * D(k),      r = 0 .. nR-1
 *   1 n, 2 nk (k-points), 3 nR (lattice vectors)
 *   4 out_dtype         NAO_COMPLEX: D(R) complex; NAO_REAL: only Re D(R) is formed and stored as doubles (D(R) is real
 *                       when the k set is inversion symmetric, D(-k) = conj D(k))
 *   5 dDk,ldd,strideD   in : device, nk complex n x n matrices, column-major
 *   8 h_k               in : HOST double[3 nk], Cartesian k (1/bohr)
 *   9 h_w               in : HOST double[nk], k-point weights
 *  10 h_R               in : HOST double[3 nR], Cartesian lattice vectors (bohr)
 *  11 dDR,lddr,strideDR out: device, nR matrices of out_dtype, column-major
 *  14 dwork, work_bytes device scratch of at least nao_fold_workspace(nk, nR) bytes
 *  16 cuda_stream
 * The host arrays are copied on entry and may be reused when the call returns.  Errors: -i for argument i, positive
 * codes as for the other calls.
 */
int nao_energy_weights(int n, int batch, const double *dE, const double *dF, double *dFE, void *cuda_stream);
int nao_fold_workspace(int nk, int nR, size_t *bytes);
int nao_fold_density(int n, int nk, int nR, int out_dtype,
                     const void *dDk, long ldd, long strideD,
                     const double *h_k, const double *h_w, const double *h_R,
                     void *dDR, long lddr, long strideDR,
                     void *dwork, size_t work_bytes, void *cuda_stream);

/* Human-readable text for a return code (static storage). */
const char *nao_status_string(int status);

/* Library version string, e.g. "nao-b200 0.1 (sm_100a)". */
const char *nao_version(void);

/*
 * Number of kernel launches this process has issued through the library since load (host counter, all entry
 * points).  bench.py uses it for its "gpu_launches" field.
 */
long nao_launch_count(void);

/*
 * Optional phase timing of nao_geneig: when enabled, CUDA events are recorded on the caller's stream at the phase
 * boundaries (potrf_trtri, reduce, tridiagonalise, stedc, back_transform, C = W^H Z).  nao_profile_read waits for the
 * events of the LAST nao_geneig call and writes the phase durations in milliseconds; returns the number written.
 */
/* Measured FP64 tensor-pipe peak of the device: a register-resident DMMA.8x8x4 loop on every SM (no memory traffic), in
 * TFLOP/s.  The roofline denominator of the GEMM-class kernels is checked against it. */
int nao_dmma_peak(double *h_tflops, void *cuda_stream);

/* Calls that run their batch as stream groups (NAO_STREAM_GROUPS_*) record nothing: their launches are on internal streams. */
int nao_profile_enable(int on);
int nao_profile_read(double *h_ms, int max_phases);
const char *nao_profile_phase_name(int i);
/*
 * Per-kernel-class timers (profiling enabled only): events bracket each launch of the class on the caller's stream.
 * slot 0 = hetrd_panel_kernel (HBM-bound; *h_work = algorithmic bytes), slot 1 = reserved.  Sums since the last
 * nao_profile_enable call: total milliseconds, total algorithmic work, number of launches.
 */
int nao_profile_kernel(int slot, double *h_ms, double *h_work, int *h_launches);
const char *nao_profile_kernel_name(int slot);
/* Per-launch durations (ms) of the launches recorded in `slot`, in launch order; returns the number written. */
int nao_profile_kernel_launches(int slot, double *h_ms, int max_launches);

/* ---- building blocks exported for tests and per-kernel measurement (same pointer/stream conventions) ---- */

/*
 * C <- alpha * op(A) * op(B) + beta * C on the FP64 tensor cores (DMMA), batched with strides.
 * op codes: 0 = N, 1 = T (transpose), 2 = C (conjugate transpose).  m,n,k are the dimensions of the product.
 * uplo_c: 0 = full C, 1 = only tiles touching the lower triangle are computed/written.
 */
int nao_gemm(int dtype, int opA, int opB, int m, int n, int k, double alpha,
             const void *dA, long lda, long strideA, const void *dB, long ldb, long strideB,
             double beta, void *dC, long ldc, long strideC, int batch, int uplo_c, void *cuda_stream);

/*
 * Cholesky factor and its inverse: dS (lower referenced) -> lower = L, strict upper = strict upper of L^{-H};
 * dLinv (n x n, ld n) <- L^{-1} (lower, zeros above).  dtmp: n*n elements of scratch per item.  d_info as in
 * nao_geneig.
 */
int nao_potrf_trtri(int n, int batch, int dtype, void *dS, long lds, long strideS,
                    void *dLinv, void *dtmp, int *d_info, void *cuda_stream);

/*
 * Hermitian eigen-decomposition A = Z diag(e) Z^H of a standard problem (lower triangle of dA referenced,
 * dA destroyed): tridiagonalisation, tridiagonal divide-and-conquer, back-transformation.
 * Workspace: nao_heev_workspace bytes.
 */
int nao_heev_workspace(int n, int batch, int dtype, unsigned flags, size_t *bytes);
int nao_heev(int n, int batch, int dtype, unsigned flags, void *dA, long lda, long strideA,
             double *dE, void *dZ, long ldz, long strideZ, void *dwork, size_t work_bytes, int *d_info,
             void *cuda_stream);

/*
 * Symmetric tridiagonal eigen-decomposition T = Q diag(e) Q^T by divide and conquer (real, all eigenpairs).
 * dD[n], dEoff[n-1] per item (item stride n) are destroyed; dE ascending; dQ n x n (ld ldq).
 */
int nao_stedc_workspace(int n, int batch, size_t *bytes);
int nao_stedc(int n, int batch, double *dD, double *dEoff, double *dE, double *dQ, long ldq, long strideQ,
              void *dwork, size_t work_bytes, int *d_info, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* NAO_H */
