// trd2.cu -- stage 1 of the two-stage tridiagonalisation: dense -> band (north_star "dense-to-band
// uses GEMM-rich panels on FP64 DMMA").  Lower storage, bandwidth b = TRD2_B.
//
// For every panel (b columns j0..j0+b-1, rows j0+b..n-1, m = n - j0 - b):
//   1. panel QR  P = Q R, Q = H_0 ... H_{b-1} = I - V T V^H        (panel_qr_kernel: one cooperative launch)
//   2. X = A22 V T ;  W = X - 1/2 V (T^H (V^H X))                    (DMMA GEMMs; A22 read through triangular masks)
//   3. A22 <- A22 - W V^H - V W^H  (lower tiles only)                (one rank-2b DMMA GEMM)
// R stays in the upper triangle of the panel (those are the band entries b + r - c <= b), V below its diagonal with
// the unit implicit: reflector of matrix column j has its unit at row j + b -- the layout ormtr(shift = b) applies.
//
// panel_qr_kernel: the G CTAs of an item hold their rows of the panel in shared memory for the whole panel and meet
// at ONE grid barrier per column.  The classical two reductions per column (norm, then v^H A) are fused: with x the
// column below the diagonal BEFORE the reflector is formed, CTAs publish sigma_c = x^H P[j+1:, c] (c >= j) and the
// owner of the diagonal row publishes rho_c = P[j, c]; then ||x||^2 = sigma_j and
//   v = [1; scale x],  v^H P[j:, c] = rho_c + conj(scale) sigma_c
// so tau, v and the update of the trailing columns follow without a second reduction; the sigma's of column j+1 are
// accumulated in the same pass that applies H_j.  Partials are summed in a fixed order (bit-reproducible).
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>

namespace nao {

static const int QR_NT = 256;
static const int QR_NW = QR_NT / 32;

template <class T> struct QrArgs {
    T *A; long lda, sA;          // full matrix (per item stride sA)
    T *tau; long sTau;           // tau[j0 + c]
    T *part;                     // per item: 2 x G x b   (double-buffered partial sigma)
    T *rowb;                     // per item: 2 x b       (double-buffered rho)
    unsigned *bar;               // per item
    int n, j0, G, chunk;
};

template <class T>
__global__ void __launch_bounds__(QR_NT, 1) panel_qr_kernel(QrArgs<T> p) {
    typedef Ops<T> O;
    constexpr int b = TRD2_B;
    const int G = p.G, item = blockIdx.x / G, g = blockIdx.x % G;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = p.n - p.j0 - b;                         // panel rows
    const int kk = min(m - 1, b);                         // reflectors
    T *P = p.A + (long)item * p.sA + (p.j0 + b) + (long)p.j0 * p.lda;      // panel (m x b), ld = lda
    T *tau = p.tau + (long)item * p.sTau + p.j0;
    T *part = p.part + (long)item * 2 * G * b;
    T *rowb = p.rowb + (long)item * 2 * b;
    unsigned *bar = p.bar + item;
    unsigned bar_ord = 0;
    const int chunk = p.chunk, CHP = chunk | 1;
    const int r0 = g * chunk, r1 = min(m, r0 + chunk);    // own rows (panel-local)
    const int nown = max(0, r1 - r0);

    extern __shared__ __align__(16) unsigned char qr_smem[];
    T *sP = (T *)qr_smem;                                 // [b][CHP]
    T *s_x = sP + (size_t)b * CHP;                        // [chunk] new column j+1
    __shared__ T s_red[4][b];
    __shared__ T s_sig[b], s_rho[b], s_z[b];
    __shared__ T s_tau, s_scale;
    __shared__ double s_beta;

    for (int e = tid; e < nown * b; e += QR_NT) {
        const int c = e / nown, r = e % nown;
        sP[c * CHP + r] = P[(r0 + r) + (long)c * p.lda];
    }
    __syncthreads();

    // partial sigma of column j over own rows r > j, columns c >= j: warp per column
    auto publish = [&](int j) {
        T *pp = part + ((long)(j & 1) * G + g) * b;
        for (int c = j + warp; c < b; c += QR_NW) {
            T s = O::zero();
            for (int r = max(r0, j + 1) - r0 + lane; r < nown; r += 32) s = O::add(s, O::conj_mul(sP[j * CHP + r], sP[c * CHP + r]));
            s = warp_sum(s);
            if (lane == 0) pp[c] = s;
        }
        if (j >= r0 && j < r1)
            for (int c = j + tid; c < b; c += QR_NT) rowb[(j & 1) * b + c] = sP[c * CHP + (j - r0)];
    };
    if (kk > 0) publish(0);

    for (int j = 0; j < kk; ++j) {
        group_barrier(bar, G, ++bar_ord);
        // ---- reduce sigma (fixed order), fetch rho
        {
            const int c = tid & (b - 1), q = tid >> 6;
            T s = O::zero();
            if (c >= j) {
                // all partials of a batch are requested before the first add: one L2 round trip per 20 CTAs x 4 quarters
                const T *pp = part + (long)(j & 1) * G * b + c;
                for (int g0 = q; g0 < G; g0 += 80) {
                    T bt[20];
#pragma unroll
                    for (int u = 0; u < 20; ++u) {
                        const int gg = g0 + 4 * u;
                        bt[u] = gg < G ? ldcg(pp + (long)gg * b) : O::zero();
                    }
#pragma unroll
                    for (int u = 0; u < 20; ++u) s = O::add(s, bt[u]);
                }
            }
            s_red[q][c] = s;
            if (q == 0 && c >= j) s_rho[c] = ldcg(rowb + (j & 1) * b + c);
        }
        __syncthreads();
        if (tid < b) s_sig[tid] = O::add(O::add(s_red[0][tid], s_red[1][tid]), O::add(s_red[2][tid], s_red[3][tid]));
        __syncthreads();
        if (tid < b) {
            // xLARFG from (alpha = rho_j, ||x||^2 = sigma_j), redundantly per thread
            const double xn2 = O::real(s_sig[j]);
            const T alpha = s_rho[j];
            const double ar = O::real(alpha), ai = O::imag(alpha);
            T tauj, scale; double beta;
            if (xn2 == 0.0 && ai == 0.0) { tauj = O::zero(); scale = O::zero(); beta = ar; }
            else {
                const double nrm = sqrt(ar * ar + ai * ai + xn2);
                beta = ar >= 0.0 ? -nrm : nrm;
                if (O::is_complex) {
                    cplx t = make_double2((beta - ar) / beta, -ai / beta);
                    const double dr = ar - beta, di = ai, den = dr * dr + di * di;
                    cplx sc = make_double2(dr / den, -di / den);
                    tauj = *(T *)&t; scale = *(T *)&sc;
                } else {
                    tauj = O::from_real((beta - ar) / beta); scale = O::from_real(1.0 / (ar - beta));
                }
            }
            if (tid > j) s_z[tid] = O::add(s_rho[tid], O::conj_mul(scale, s_sig[tid]));
            if (tid == j) {
                s_tau = tauj; s_scale = scale; s_beta = beta;
                if (g == 0) tau[j] = tauj;
            }
        }
        __syncthreads();
        const T ctau = O::conj(s_tau), scale = s_scale;
        // ---- phase a: v into column j; column j+1 brought up to date (s_x); diagonal row (owner)
        const int lo = max(r0, j + 1) - r0;
        const bool nextcol = (j + 1 < b);
        const T zn = nextcol ? s_z[j + 1] : O::zero();
        for (int r = lo + tid; r < nown; r += QR_NT) {
            const T v = O::mul(scale, sP[j * CHP + r]);
            sP[j * CHP + r] = v;
            if (nextcol) {
                const T x = O::sub(sP[(j + 1) * CHP + r], O::mul(O::mul(ctau, zn), v));
                sP[(j + 1) * CHP + r] = x;
                s_x[r] = x;
            }
        }
        if (j >= r0 && j < r1) {
            for (int c = j + tid; c < b; c += QR_NT) {
                if (c == j) sP[c * CHP + (j - r0)] = O::from_real(s_beta);
                else sP[c * CHP + (j - r0)] = O::sub(sP[c * CHP + (j - r0)], O::mul(ctau, s_z[c]));
            }
        }
        __syncthreads();
        // ---- phase b: apply H_j^H to columns c > j+1, accumulate sigma of column j+1 for c >= j+1
        {
            const bool pub = (j + 1 < kk);
            T *pp = part + ((long)((j + 1) & 1) * G + g) * b;
            const int lo2 = max(r0, j + 2) - r0;            // rows that enter the next sigma
            for (int c = j + 1 + warp; c < b; c += QR_NW) {
                T s = O::zero();
                if (c == j + 1) {
                    if (pub) for (int r = lo2 + lane; r < nown; r += 32) s = O::add(s, O::conj_mul(s_x[r], s_x[r]));
                } else {
                    const T f = O::mul(ctau, s_z[c]);
                    for (int r = lo + lane; r < nown; r += 32) {
                        const T a = O::sub(sP[c * CHP + r], O::mul(f, sP[j * CHP + r]));
                        sP[c * CHP + r] = a;
                        if (r >= lo2) s = O::add(s, O::conj_mul(s_x[r], a));
                    }
                }
                if (pub) {
                    s = warp_sum(s);
                    if (lane == 0) pp[c] = s;
                }
            }
            __syncthreads();
            if (pub && j + 1 >= r0 && j + 1 < r1)
                for (int c = j + 1 + tid; c < b; c += QR_NT) rowb[((j + 1) & 1) * b + c] = sP[c * CHP + (j + 1 - r0)];
        }
    }
    if (g == 0) for (int c = max(kk, 0) + tid; c < b; c += QR_NT) tau[c] = O::zero();
    __syncthreads();
    for (int e = tid; e < nown * b; e += QR_NT) {
        const int c = e / nown, r = e % nown;
        P[(r0 + r) + (long)c * p.lda] = sP[c * CHP + r];
    }
}

// ----------------------------------------------------------------------------------------------------------------
// Small b x b algebra of a panel, one CTA per item:  T from (G = V^H V, tau) by the xLARFT recurrence,
// M = T^H S0 T with S0 = V^H X, and the stacked coefficient matrix  B2 = [T ; -1/2 M]  (2b x b) so that
//   W = X T - 1/2 V M = [X | V] B2   is one GEMM.      GS = [S0 | G] (b x 2b, ld b).
// ----------------------------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) he2hb_small_kernel(const T *GS, long sGS, const T *tau, long sTau, T *B2, long sB2) {
    typedef Ops<T> O;
    constexpr int b = TRD2_B, LD = b + 1;
    extern __shared__ __align__(16) unsigned char sm_raw[];
    T *sG = (T *)sm_raw;            // G, later S0
    T *sT = sG + b * LD;            // T (dense, zeros below the diagonal)
    T *sX = sT + b * LD;            // S0 T
    __shared__ T s_tau[b];
    GS += (long)blockIdx.x * sGS; tau += (long)blockIdx.x * sTau; B2 += (long)blockIdx.x * sB2;
    const int tid = threadIdx.x;
    for (int e = tid; e < b * b; e += 256) {
        const int i = e % b, j = e / b;
        sG[i * LD + j] = GS[(long)(b + j) * b + i];        // G(i,j), row-major in shared memory
        sT[i * LD + j] = O::zero();
    }
    if (tid < b) s_tau[tid] = tau[tid];
    __syncthreads();
    // T = U^{-1} with U = diag(1/tau) + striu(G)  (T^{-1} + T^{-H} = V^H V): column j of T by back substitution,
    //   T(j,j) = tau_j,   T(i,j) = -tau_i sum_{k=i+1..j} G(i,k) T(k,j)   (i = j-1 .. 0),
    // which needs no division (tau_i = 0, H_i = I, gives a zero row and column) and -- unlike the column-by-column xLARFT
    // recurrence -- no block barrier: the 64 columns are independent, 4 adjacent lanes share the k-sum of one column.
    {
        const int j = tid >> 2, part = tid & 3;
        if (part == 0) sT[j * LD + j] = s_tau[j];
        __syncwarp();
        const int jtop = (tid | 31) >> 2;                  // last column of this warp: warp-uniform trip count
        for (int i = jtop - 1; i >= 0; --i) {
            T acc = O::zero();
            if (i < j)
                for (int k = i + 1 + part; k <= j; k += 4) acc = O::fma(sG[i * LD + k], sT[k * LD + j], acc);
            double *a = (double *)&acc;
#pragma unroll
            for (int w = 0; w < (int)(sizeof(T) / 8); ++w) {
                a[w] += __shfl_xor_sync(0xffffffffu, a[w], 1);
                a[w] += __shfl_xor_sync(0xffffffffu, a[w], 2);
            }
            if (part == 0 && i < j) sT[i * LD + j] = O::sub(O::zero(), O::mul(s_tau[i], acc));
            __syncwarp();
        }
    }
    __syncthreads();
    for (int e = tid; e < b * b; e += 256) {
        const int i = e % b, j = e / b;
        sG[i * LD + j] = GS[(long)j * b + i];              // S0(i,j)
        B2[i + (long)j * 2 * b] = sT[i * LD + j];          // rows 0..b-1 of B2 = T
    }
    __syncthreads();
    for (int e = tid; e < b * b; e += 256) {               // sX = S0 T : sX(i,j) = sum_{k<=j} S0(i,k) T(k,j)
        const int j = e % b, i = e / b;
        T acc = O::zero();
        for (int k = 0; k <= j; ++k) acc = O::fma(sG[i * LD + k], sT[k * LD + j], acc);
        sX[i * LD + j] = acc;
    }
    __syncthreads();
    for (int e = tid; e < b * b; e += 256) {               // M(i,j) = sum_{k<=i} conj(T(k,i)) sX(k,j)
        const int j = e % b, i = e / b;
        T acc = O::zero();
        for (int k = 0; k <= i; ++k) acc = O::add(acc, O::conj_mul(sT[k * LD + i], sX[k * LD + j]));
        B2[(b + i) + (long)j * 2 * b] = O::scale(acc, -0.5);
    }
}

// ----------------------------------------------------------------------------------------------------------------
// he2hb driver
// ----------------------------------------------------------------------------------------------------------------
struct He2hbWork {
    void *P4, *GS, *B2, *part, *rowb, *splitk; unsigned *bar;
    int Gq, chunk, ipl, ksX, ksS; size_t smem, bytes;
};
static int trd2_num_sms() { return sm_count(); }
static He2hbWork he2hb_plan(int dtype, int n, int batch, void *work) {
    He2hbWork w; const size_t es = esize(dtype); const int b = TRD2_B;
    const int nsm = trd2_num_sms();
    const int m0 = std::max(1, n - b);
    // rows of the panel a CTA can keep in shared memory (b columns), leaving room for the static arrays
    const int cap = (int)((200 * 1024) / ((size_t)(b + 1) * es)) - 2;
    const int Gneed = ceil_div(m0, cap);
    w.ipl = std::max(1, std::min(batch, nsm / std::max(1, Gneed)));      // items per cooperative launch
    w.Gq = std::max(1, std::min(nsm / w.ipl, ceil_div(m0, 32)));
    w.chunk = ceil_div(m0, w.Gq);
    w.smem = ((size_t)b * (w.chunk | 1) + w.chunk) * es;
    // split-K factors: X = A22 V (m x b, k = m) fills ~3 CTAs per SM-slot; the b x 2b product one slice per SM
    w.ksX = 16;          // upper bound (sizes the scratch); the factor is chosen per panel to fill the last wave of CTAs
    w.ksS = std::max(1, std::min(std::min(nsm / std::max(1, batch), ceil_div(n, 256)), 64));
    Arena ar(work, (size_t)-1);
    w.P4 = ar.take((size_t)batch * n * 4 * b * es);            // [X | V | W | V], ld n, rows indexed globally
    w.GS = ar.take((size_t)batch * 2 * b * b * es);
    w.B2 = ar.take((size_t)batch * 2 * b * b * es);
    w.part = ar.take((size_t)batch * 2 * w.Gq * b * es);
    w.rowb = ar.take((size_t)batch * 2 * b * es);
    w.splitk = ar.take((size_t)batch * std::max((size_t)w.ksX * n * b, (size_t)w.ksS * 2 * b * b) * es);
    w.bar = (unsigned *)ar.take((size_t)batch * (ceil_div(n, b) + 1) * 4);
    w.bytes = ar.off;
    return w;
}
size_t he2hb_workspace(int dtype, int n, int batch) { return he2hb_plan(dtype, n, batch, nullptr).bytes; }
bool he2hb_supported(int dtype, int n, int batch) {
    He2hbWork w = he2hb_plan(dtype, n, batch, nullptr);
    return n > TRD2_B + 1 && w.smem <= 210 * 1024 && w.Gq * w.ipl <= trd2_num_sms();
}

template <class T>
static int he2hb_impl(int dtype, int n, int batch, T *A, long lda, long sA, T *tau, void *work, cudaStream_t st) {
    const int b = TRD2_B;
    He2hbWork w = he2hb_plan(dtype, n, batch, work);
    const size_t small_smem = (size_t)3 * b * (b + 1) * sizeof(T);
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(panel_qr_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024));
        NAO_CUDA_CHECK(cudaFuncSetAttribute(he2hb_small_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem));
        attr = true;
    }
    const int npanels = ceil_div(n, b) + 1;
    NAO_CUDA_CHECK(cudaMemsetAsync(w.bar, 0, (size_t)batch * npanels * 4, st));
    NAO_CUDA_CHECK(cudaMemsetAsync(tau, 0, (size_t)batch * n * sizeof(T), st));
    T *P4 = (T *)w.P4;
    const long sP4 = (long)n * 4 * b, sGS = (long)2 * b * b;
    T *Xb = P4, *Vb = P4 + (long)n * b, *Wb = P4 + (long)n * 2 * b, *Vb2 = P4 + (long)n * 3 * b;
    // Look-ahead: the panel QR is a chain of 64 grid barriers (latency, ~5 us per column) and needs few SMs; the rank-2b
    // update of the trailing matrix is a large GEMM.  The update of panel p is therefore split: the 64 columns that form
    // panel p+1 first, then -- on an internal side stream, on as few CTAs as hold the panel in shared memory -- the QR of
    // panel p+1 WHILE the rest of the update runs on the caller's stream (its CTAs fill the SMs the QR leaves free).
    // Disabled while a stream group limits the SMs (the groups overlap one another instead).
    static SideSet ss = {};
    const bool lookahead = sm_count() >= device_sms() && n >= 1024;
    if (lookahead) if (int rc = side_set_init(ss, 1, 4, true)) return rc;   // high priority: the QR's CTAs take freed SMs first
    const cudaStream_t side = ss.stream[0];
    const cudaEvent_t ev_cols = ss.event[0], ev_side = ss.event[1], ev_qr = ss.event[2];
    SideJoin join(side, st, ss.event[3]);      // armed at the first fork: every exit path rejoins the side stream
    const int cap_rows = (int)((200 * 1024) / ((size_t)(b + 1) * sizeof(T))) - 2;       // panel rows one CTA can hold
    auto launch_qr = [&](int j0, int panel, cudaStream_t qs, bool few_ctas) -> int {
        const int m = n - j0 - b;
        for (int b0 = 0; b0 < batch; b0 += w.ipl) {
            const int nit = std::min(w.ipl, batch - b0);
            QrArgs<T> a;
            a.A = A + (long)b0 * sA; a.lda = lda; a.sA = sA; a.tau = tau + (long)b0 * n; a.sTau = n;
            a.part = (T *)w.part + (long)b0 * 2 * w.Gq * b; a.rowb = (T *)w.rowb + (long)b0 * 2 * b;
            a.bar = w.bar + (size_t)panel * batch + b0;
            a.n = n; a.j0 = j0;
            a.G = std::max(1, std::min(w.Gq, ceil_div(m, 32)));
            // (measured at config 2, dense->band in ms: 8 CTAs per item 92.2, 16: 88.9, 24: 87.9, 37: 86.2, all 74: 89.5; no look-ahead 96.4)
            if (few_ctas) a.G = std::max(1, std::min(a.G, std::max(ceil_div(m, cap_rows), 32)));
            a.chunk = ceil_div(m, a.G);
            const size_t smem = ((size_t)b * (a.chunk | 1) + a.chunk) * sizeof(T);
            void *args[] = {&a};
            NAO_CUDA_CHECK(cudaLaunchCooperativeKernel((void *)panel_qr_kernel<T>, dim3(nit * a.G), dim3(QR_NT), args, smem, qs));
            NAO_LAUNCHED();
        }
        return NAO_OK;
    };
    int panel = 0;
    bool qr_done_ahead = false;            // the QR of the current panel was issued by the previous iteration
    for (int j0 = 0; n - j0 - b > 1; j0 += b, ++panel) {
        const int m = n - j0 - b, jr = j0 + b;      // panel rows start at global row jr
        // 1. panel QR (cooperative), items in groups of ipl
        if (!qr_done_ahead) { if (int rc = launch_qr(j0, panel, st, false)) return rc; }
        else NAO_CUDA_CHECK(cudaStreamWaitEvent(st, ev_qr, 0));
        qr_done_ahead = false;
        // 2. explicit V (m x b, zeros above the unit diagonal) at rows jr.. of both V blocks
        if (int rc = build_v(dtype, n, j0, b, b, A, lda, sA, Vb + jr, n, sP4, batch, st)) return rc;
        if (int rc = copy_matrix(dtype, m, b, Vb + jr, n, sP4, Vb2 + jr, n, sP4, batch, 0, st)) return rc;
        // 3. X = A22 V : lower triangle as stored + strictly lower triangle transposed
        T *A22 = A + jr + (long)jr * lda;
        const int ksx = fill_ksplit((long)ceil_div(m, 128) * batch, sm_count(), std::min(w.ksX, ceil_div(m, 512)));
        GemmDesc x1 = gemm_desc(OP_N, OP_N, m, b, m, 1.0, A22, lda, Vb + jr, n, 0.0, Xb + jr, n);
        x1.sA = sA; x1.sB = sP4; x1.sC = sP4; x1.maskA = MASK_LOWER;
        if (int rc = gemm_splitk(dtype, x1, batch, ksx, w.splitk, st)) return rc;
        GemmDesc x2 = gemm_desc(OP_C, OP_N, m, b, m, 1.0, A22, lda, Vb + jr, n, 1.0, Xb + jr, n);
        x2.sA = sA; x2.sB = sP4; x2.sC = sP4; x2.maskA = MASK_SLOWER;
        if (int rc = gemm_splitk(dtype, x2, batch, ksx, w.splitk, st)) return rc;
        // 4. [S0 | G] = V^H [X | V] ; B2 = [T ; -1/2 T^H S0 T] ; W = [X | V] B2
        GemmDesc gs = gemm_desc(OP_C, OP_N, b, 2 * b, m, 1.0, Vb + jr, n, Xb + jr, n, 0.0, w.GS, b);
        gs.sA = sP4; gs.sB = sP4; gs.sC = sGS;
        if (int rc = gemm_splitk(dtype, gs, batch, std::min(w.ksS, ceil_div(m, 256)), w.splitk, st)) return rc;
        he2hb_small_kernel<T><<<batch, 256, small_smem, st>>>((const T *)w.GS, sGS, tau + j0, n, (T *)w.B2, sGS);
        NAO_LAUNCHED();
        GemmDesc w1 = gemm_desc(OP_N, OP_N, m, b, 2 * b, 1.0, Xb + jr, n, w.B2, 2 * b, 0.0, Wb + jr, n);
        w1.sA = sP4; w1.sB = sGS; w1.sC = sP4;
        if (int rc = gemm_launch(dtype, w1, batch, st)) return rc;
        // 5. A22 -= V W^H + W V^H = [V W] [W V]^H, lower tiles
        const bool next_panel = (n - (j0 + b) - b > 1);
        if (lookahead && next_panel && m - b >= 512) {
            // 5a. the b columns of the next panel (rows jr.. : its diagonal block and everything below)
            GemmDesc ua = gemm_desc(OP_N, OP_C, m, b, 2 * b, -1.0, Vb + jr, n, Wb + jr, n, 1.0, A22, lda);
            ua.sA = sP4; ua.sB = sP4; ua.sC = sA;        // (cmode 0: one tile column starting at the diagonal, no tile is skipped)
            if (int rc = gemm_launch(dtype, ua, batch, st)) return rc;
            NAO_CUDA_CHECK(cudaEventRecord(ev_cols, st));
            NAO_CUDA_CHECK(cudaStreamWaitEvent(side, ev_cols, 0));
            join.arm();
            NAO_CUDA_CHECK(cudaEventRecord(ev_side, side));
            // QR of panel p+1 on the (high-priority) side stream; the big update is held back until the side stream has got
            // past its wait, so that the QR's CTAs are placed first and the update fills the SMs they leave free
            if (int rc = launch_qr(j0 + b, panel + 1, side, true)) return rc;
            NAO_CUDA_CHECK(cudaEventRecord(ev_qr, side));
            qr_done_ahead = true;
            NAO_CUDA_CHECK(cudaStreamWaitEvent(st, ev_side, 0));
            // 5b. the rest of the trailing matrix
            GemmDesc ub = gemm_desc(OP_N, OP_C, m - b, m - b, 2 * b, -1.0, Vb + jr + b, n, Wb + jr + b, n, 1.0,
                                    A22 + b + (long)b * lda, lda);
            ub.sA = sP4; ub.sB = sP4; ub.sC = sA; ub.cmode = 1;
            if (int rc = gemm_launch(dtype, ub, batch, st)) return rc;
        } else {
            GemmDesc u = gemm_desc(OP_N, OP_C, m, m, 2 * b, -1.0, Vb + jr, n, Wb + jr, n, 1.0, A22, lda);
            u.sA = sP4; u.sB = sP4; u.sC = sA; u.cmode = 1;
            if (int rc = gemm_launch(dtype, u, batch, st)) return rc;
        }
    }
    if (qr_done_ahead) NAO_CUDA_CHECK(cudaStreamWaitEvent(st, ev_qr, 0));
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int he2hb(int dtype, int n, int batch, void *A, long lda, long sA, void *tau, void *work, cudaStream_t st) {
    return dtype == NAO_COMPLEX ? he2hb_impl<cplx>(dtype, n, batch, (cplx *)A, lda, sA, (cplx *)tau, work, st)
                                : he2hb_impl<double>(dtype, n, batch, (double *)A, lda, sA, (double *)tau, work, st);
}

}  // namespace nao
