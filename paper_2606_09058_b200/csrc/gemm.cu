// gemm.cu -- FP64 tensor-core (DMMA) GEMM core for sm_100a.
//
// Every GEMM-class phase of the path (Cholesky trailing update, L^{-1} H L^{-H}, rank-2k updates of the
// tridiagonalisation, divide-and-conquer merges, block-reflector back-transformation, C = L^{-H} Z and the
// density matrix D = C f C^H) runs through this one kernel.
//
// sm_100a has no FP64 kind in tcgen05.mma; the FP64 tensor path is warp-level mma.sync.m8n8k4 (SASS DMMA.8x8x4),
// fed from registers.  One DMMA per warp is 512 flop and occupies the FP64 pipe for ~16 issue slots, so the
// instruction-issue and shared-memory load rates are far from limiting; what matters is (i) a CTA tile large
// enough that L2->SM traffic stays small (128x128 real: 8 B/clk/SM), (ii) a multi-stage cp.async pipeline so the
// DMMA pipe never waits, (iii) conflict-free 64/128-bit fragment loads (padding chosen per layout below).
//
// Complex products use real-arithmetic DMMAs on the (re, im) planes of interleaved operands:
//   Cr += Ar*Br + (-Ai)*Bi ;  Ci += Ar*Bi + Ai*Br        (4 real DMMAs per complex tile product).
//
// Features: op(A), op(B) in {N, T, C}; real alpha/beta; triangular masks on either stored operand (elements
// outside the triangle read as zero and the k-range is clipped, so TRMM/SYRK-shaped products skip the empty
// half); "lower tiles only" output; optional scaling of op(A)'s k-th column by s[k] (Fermi weights);
// strided batches and grouped launches whose descriptors (incl. m,n,k) live in device memory.
#include "nao_internal.cuh"
#include "scalar.cuh"

namespace nao {

long g_launch_count = 0;

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ double negate(double x) { return -x; }

__device__ __forceinline__ bool mask_keep(int mask, int off, int r, int c) {
    int t = r - c + off;
    return mask == MASK_NONE || (mask == MASK_LOWER && t >= 0) || (mask == MASK_SLOWER && t > 0) ||
           (mask == MASK_UPPER && t <= 0) || (mask == MASK_SUPPER && t < 0);
}
// clip [kb, ke) given the mask on an operand whose other index spans [x0, x1]; k_is_col: stored (r,c) = (x,k)
__device__ __forceinline__ void mask_krange(int mask, int off, bool k_is_col, int x0, int x1, int &kb, int &ke) {
    if (mask == MASK_NONE) return;
    bool lower = (mask == MASK_LOWER || mask == MASK_SLOWER);
    if (k_is_col) {            // keep x - k + off >= 0 (lower) / <= 0 (upper)
        if (lower) ke = min(ke, x1 + off + 1); else kb = max(kb, x0 + off);
    } else {                   // (r,c) = (k,x): keep k - x + off >= 0 / <= 0
        if (lower) kb = max(kb, x0 - off); else ke = min(ke, x1 - off + 1);
    }
}

// NARROW: 128 x 64 tile for real products whose output has at most 64 columns (tall-skinny panels of he2hb)
template <bool CPLX, bool NARROW = false> struct Cfg;
template <> struct Cfg<false, true> {
    typedef double T;
    static const int BM = 128, BN = 64, BK = 16, WM = 32, WN = 32, STAGES = 4, PADX = 4, PADK = 4;
};
template <> struct Cfg<false, false> {
    typedef double T;
    static const int BM = 128, BN = 128, BK = 16, WM = 32, WN = 64, STAGES = 4, PADX = 4, PADK = 4;
};
template <> struct Cfg<true, false> {
    typedef cplx T;
    static const int BM = 128, BN = 64, BK = 16, WM = 32, WN = 32, STAGES = 4, PADX = 2, PADK = 2;
};
static const int GEMM_THREADS = 256;

template <int BX, int BK, int PADX, int PADK> struct TileSize {
    static const int XC = BK * (BX + PADX), KC = BX * (BK + PADK);
    static const int value = XC > KC ? XC : KC;
};

// Load one BX x BK tile of op(P) into shared memory.
//   xcontig: stored element (x,k) at P[x + k*ld]  -> smem [k][x], else stored at P[k + x*ld] -> smem [x][k].
template <bool CPLX, int BX, int BK, int PADX, int PADK>
__device__ __forceinline__ void load_tile(typename Cfg<CPLX>::T *s, const typename Cfg<CPLX>::T *P, long ld,
                                          bool xcontig, int x0, int X, int k0, int kb, int ke, int mask, int off,
                                          bool k_is_col) {
    const int tid = threadIdx.x;
    if (xcontig) {
#pragma unroll
        for (int it = 0; it < BX * BK / GEMM_THREADS; ++it) {
            int e = tid + it * GEMM_THREADS;
            int x = e % BX, k = e / BX;
            int gx = x0 + x, gk = k0 + k;
            bool p = gx < X && gk >= kb && gk < ke && (k_is_col ? mask_keep(mask, off, gx, gk) : mask_keep(mask, off, gk, gx));
            const typename Cfg<CPLX>::T *src = p ? P + gx + (long)gk * ld : P;
            if constexpr (CPLX) cp_async16(s + k * (BX + PADX) + x, src, p); else cp_async8(s + k * (BX + PADX) + x, src, p);
        }
    } else {
#pragma unroll
        for (int it = 0; it < BX * BK / GEMM_THREADS; ++it) {
            int e = tid + it * GEMM_THREADS;
            int k = e % BK, x = e / BK;
            int gx = x0 + x, gk = k0 + k;
            bool p = gx < X && gk >= kb && gk < ke && (k_is_col ? mask_keep(mask, off, gx, gk) : mask_keep(mask, off, gk, gx));
            const typename Cfg<CPLX>::T *src = p ? P + gk + (long)gx * ld : P;
            if constexpr (CPLX) cp_async16(s + x * (BK + PADK) + k, src, p); else cp_async8(s + x * (BK + PADK) + k, src, p);
        }
    }
}

// is the whole stored rectangle rows [r0,r1] x cols [c0,c1] kept by the mask?
__device__ __forceinline__ bool mask_all_kept(int mask, int off, int r0, int r1, int c0, int c1) {
    switch (mask) {
        case MASK_NONE: return true;
        case MASK_LOWER: return r0 - c1 + off >= 0;
        case MASK_SLOWER: return r0 - c1 + off > 0;
        case MASK_UPPER: return r1 - c0 + off <= 0;
        default: return r1 - c0 + off < 0;
    }
}

// Fast tile loader: 16-byte cp.async, one running global pointer per thread, compile-time shared-memory offsets.
// Used for k-tiles that lie entirely inside the operand (no edge, no mask boundary, aligned); everything else goes
// through load_tile.  The NCH chunks of a thread are issued in 4 parts so that the copies interleave with the DMMAs.
template <bool CPLX, int BX, int BK, int PADX, int PADK, bool XC, bool AL16> struct FastLoad {
    typedef typename Cfg<CPLX>::T T;
    static const int VEC = (CPLX || !AL16) ? 1 : 2;            // elements per chunk (16 bytes; 8 bytes for misaligned real operands)
    static const int NCH = BX * BK / (VEC * GEMM_THREADS);     // chunks per thread per tile
    static const int P = XC ? BX / VEC : BK / VEC;             // chunks along the contiguous direction
    static const int STEP = GEMM_THREADS / P;                  // other-index distance between a thread's chunks
    const T *g;            // chunk 0 of the current k-tile
    long cstride;          // elements between consecutive chunks of this thread (STEP * ld)
    long kadv;             // elements per k-tile
    int soff;              // shared-memory offset of chunk 0
    __device__ __forceinline__ void init(const T *Pm, long ld, int x0, int k0) {
        const int tid = threadIdx.x;
        const int c = (tid % P) * VEC, o = tid / P;
        if (XC) { g = Pm + (x0 + c) + (long)(k0 + o) * ld; soff = o * (BX + PADX) + c; kadv = (long)BK * ld; }
        else { g = Pm + (k0 + c) + (long)(x0 + o) * ld; soff = o * (BK + PADK) + c; kadv = BK; }
        cstride = (long)STEP * ld;
    }
    template <int PART> __device__ __forceinline__ void issue(T *s) const {
        constexpr int SSTR = XC ? STEP * (BX + PADX) : STEP * (BK + PADK);
        constexpr int c0 = PART * NCH / 4, c1 = (PART + 1) * NCH / 4;
#pragma unroll
        for (int c = c0; c < c1; ++c) {
            if constexpr (CPLX || AL16) cp_async16(s + soff + c * SSTR, g + c * cstride, true);
            else cp_async8(s + soff + c * SSTR, g + c * cstride, true);
        }
    }
    __device__ __forceinline__ void advance() { g += kadv; }
};

template <bool CPLX, bool AXC, bool BXC, bool SCALE, bool NARROW, bool AL16>
__global__ void __launch_bounds__(GEMM_THREADS, 1)
gemm_kernel(const GemmDesc hd, const GemmDesc *__restrict__ dd) {
    typedef Cfg<CPLX, NARROW> G;
    typedef typename G::T T;
    constexpr int BM = G::BM, BN = G::BN, BK = G::BK, WM = G::WM, WN = G::WN, ST = G::STAGES;
    constexpr int MI = WM / 8, NI = WN / 8;
    constexpr int ASZ = TileSize<BM, BK, G::PADX, G::PADK>::value;
    constexpr int BSZ = TileSize<BN, BK, G::PADX, G::PADK>::value;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *sA = (T *)smem_raw;
    T *sB = sA + ST * ASZ;
    double *sS = (double *)(sB + ST * BSZ);     // ST * BK scale factors

    const GemmDesc d = dd ? dd[blockIdx.z] : hd;
    const int M = d.m, N = d.n, K = d.k;
    if (M <= 0 || N <= 0) return;
    const int tiles_m = (M + BM - 1) / BM, tiles_n = (N + BN - 1) / BN;
    if ((int)blockIdx.x >= tiles_m * tiles_n) return;
    // supertile raster: CTAs that run together cover GS tile rows x a few tile columns, so that the A and B panels
    // they share stay in L2 (a plain column-of-tiles order re-reads A once per tile column)
    constexpr int GS = 8;
    const int bid = blockIdx.x, gsize = GS * tiles_n, gid = bid / gsize, first_m = gid * GS;
    const int gsz = min(tiles_m - first_m, GS);
    const int tm = first_m + (bid % gsize) % gsz, tn = (bid % gsize) / gsz;
    const int m0 = tm * BM, n0 = tn * BN;
    const int cmode = d.cmode;
    if (cmode == 1 && n0 > m0 + BM - 1) return;
    if (cmode == 2 && n0 > (m0 + BM - 1) / 2) return;

    const int ks = d.ksplit > 1 ? d.ksplit : 1;
    const long b = blockIdx.y / ks;
    const int slice = blockIdx.y % ks;
    const T *A = (const T *)d.A + b * d.sA;
    const T *B = (const T *)d.B + b * d.sB;
    const long lda = d.lda, ldb = d.ldb, ldc = d.ldc;
    T *C = (T *)d.C + b * d.sC + (long)slice * d.sSplit;
    const double *scaleK = SCALE ? d.scaleK + b * d.sScale : nullptr;
    const int maskA = d.maskA, offA = d.offA, maskB = d.maskB, offB = d.offB;

    // op(A)(i,k): N -> stored (r,c) = (i,k), m-contiguous (AXC);  T/C -> stored (k,i), k-contiguous
    // op(B)(k,j): N -> stored (k,j), k-contiguous;  T/C -> stored (j,k), n-contiguous (BXC)
    const bool conjA = CPLX && d.opA == OP_C, conjB = CPLX && d.opB == OP_C;

    int kb = 0, ke = K;
    mask_krange(maskA, offA, AXC, m0, min(m0 + BM, M) - 1, kb, ke);
    mask_krange(maskB, offB, BXC, n0, min(n0 + BN, N) - 1, kb, ke);
    kb = max(kb, 0); ke = min(ke, K);
    if (ks > 1) {
        // slices of the CLIPPED range: every slice of a tile carries the same work also under triangular masks
        const int kb0 = kb / BK * BK;
        const int kchunk = ((max(ke - kb0, 0) + ks - 1) / ks + BK - 1) / BK * BK;
        kb = max(kb, kb0 + slice * kchunk); ke = min(ke, kb0 + (slice + 1) * kchunk);
    }
    const int kt0 = kb / BK;
    const int nkt = ke > kb ? (ke - 1) / BK + 1 - kt0 : 0;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int WARPS_M = BM / WM;
    const int wm = (warp % WARPS_M) * WM, wn = (warp / WARPS_M) * WN;
    const int lr = lane >> 2, lc = lane & 3;

    double acc[MI][NI][CPLX ? 4 : 2];
    const double alpha = d.alpha, beta = d.beta;
    constexpr int a_sx = AXC ? 1 : (BK + G::PADK), a_sk = AXC ? (BM + G::PADX) : 1;
    constexpr int b_sx = BXC ? 1 : (BK + G::PADK), b_sk = BXC ? (BN + G::PADX) : 1;

    // ---- tile loading: fast (interior, aligned) or generic, decided per k-tile, uniformly over the CTA
    FastLoad<CPLX, BM, BK, G::PADX, G::PADK, AXC, AL16> fa;
    FastLoad<CPLX, BN, BK, G::PADX, G::PADK, BXC, AL16> fb;
    fa.init(A, lda, m0, kt0 * BK);
    fb.init(B, ldb, n0, kt0 * BK);
    const bool a_al = CPLX || !AL16 || ((((size_t)A) & 15) == 0 && (lda & 1) == 0 && ((AXC ? m0 : 0) & 1) == 0);
    const bool b_al = CPLX || !AL16 || ((((size_t)B) & 15) == 0 && (ldb & 1) == 0 && ((BXC ? n0 : 0) & 1) == 0);
    const bool a_in = a_al && (m0 + BM <= M), b_in = b_al && (n0 + BN <= N);
    auto a_fast = [&](int k0) -> bool {
        if (!a_in || k0 < kb || k0 + BK > ke) return false;
        return AXC ? mask_all_kept(maskA, offA, m0, m0 + BM - 1, k0, k0 + BK - 1)
                   : mask_all_kept(maskA, offA, k0, k0 + BK - 1, m0, m0 + BM - 1);
    };
    auto b_fast = [&](int k0) -> bool {
        if (!b_in || k0 < kb || k0 + BK > ke) return false;
        return BXC ? mask_all_kept(maskB, offB, n0, n0 + BN - 1, k0, k0 + BK - 1)
                   : mask_all_kept(maskB, offB, k0, k0 + BK - 1, n0, n0 + BN - 1);
    };
    // generic part of the load of k-tile kt_rel (+ the scale factors); returns which operands are left to the fast path
    auto issue_generic = [&](int kt_rel, bool &fa_on, bool &fb_on) {
        fa_on = fb_on = false;
        if (kt_rel < nkt) {
            const int stg = kt_rel % ST;
            const int k0 = (kt0 + kt_rel) * BK;
            fa_on = a_fast(k0); fb_on = b_fast(k0);
            if (!fa_on) load_tile<CPLX, BM, BK, G::PADX, G::PADK>(sA + stg * ASZ, A, lda, AXC, m0, M, k0, kb, ke, maskA, offA, AXC);
            if (!fb_on) load_tile<CPLX, BN, BK, G::PADX, G::PADK>(sB + stg * BSZ, B, ldb, BXC, n0, N, k0, kb, ke, maskB, offB, BXC);
            if (SCALE && threadIdx.x < BK) {
                const int gk = k0 + threadIdx.x;
                const bool p = gk < ke;
                cp_async8(sS + stg * BK + threadIdx.x, p ? scaleK + gk : scaleK, p);
            }
        }
    };

    for (int s = 0; s < ST - 1; ++s) {
        bool fa_on, fb_on;
        issue_generic(s, fa_on, fb_on);
        T *as = sA + (s % ST) * ASZ, *bs = sB + (s % ST) * BSZ;
        if (fa_on) { fa.template issue<0>(as); fa.template issue<1>(as); fa.template issue<2>(as); fa.template issue<3>(as); }
        if (fb_on) { fb.template issue<0>(bs); fb.template issue<1>(bs); fb.template issue<2>(bs); fb.template issue<3>(bs); }
        fa.advance(); fb.advance();
        cp_async_commit();
    }

    // (after the first tiles have been requested, so that the loads of C overlap the pipeline fill)
    // beta != 0: the accumulators start from (beta/alpha) C, loaded while the first tiles are in flight, so that the
    // epilogue is store-only (for alpha = +-1, beta = 1 -- every update on the path -- this is exact)
    const bool preload = (beta != 0.0 && alpha != 0.0);
    if (preload) {
        const double r = beta / alpha;
#pragma unroll
        for (int i = 0; i < MI; ++i) {
            const int gi = m0 + wm + i * 8 + lr;
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int gj = n0 + wn + j * 8 + 2 * lc + q;
                    T v;
                    if constexpr (CPLX) v = make_double2(0.0, 0.0); else v = 0.0;
                    if (gi < M && gj < N) v = C[gi + (long)gj * ldc];
                    if constexpr (CPLX) { acc[i][j][q] = r * v.x; acc[i][j][2 + q] = r * v.y; } else acc[i][j][q] = r * v;
                }
        }
    } else {
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
                for (int q = 0; q < (CPLX ? 4 : 2); ++q) acc[i][j][q] = 0.0;
    }

    for (int kt = 0; kt < nkt; ++kt) {
        cp_async_wait<ST - 2>();
        __syncthreads();
        bool fa_on, fb_on;
        issue_generic(kt + ST - 1, fa_on, fb_on);
        T *as_n = sA + ((kt + ST - 1) % ST) * ASZ, *bs_n = sB + ((kt + ST - 1) % ST) * BSZ;
        const T *a_s = sA + (kt % ST) * ASZ;
        const T *b_s = sB + (kt % ST) * BSZ;
        const double *s_s = sS + (kt % ST) * BK;
        const T *a_p = a_s + (wm + lr) * a_sx + lc * a_sk;
        const T *b_p = b_s + (wn + lr) * b_sx + lc * b_sk;
#pragma unroll
        for (int kq = 0; kq < BK / 4; ++kq) {
            const int kk = kq * 4;
            // one quarter of the next tile's copies per k-step
            if (fa_on) {
                if (kq == 0) fa.template issue<0>(as_n); else if (kq == 1) fa.template issue<1>(as_n);
                else if (kq == 2) fa.template issue<2>(as_n); else fa.template issue<3>(as_n);
            }
            if (fb_on) {
                if (kq == 0) fb.template issue<0>(bs_n); else if (kq == 1) fb.template issue<1>(bs_n);
                else if (kq == 2) fb.template issue<2>(bs_n); else fb.template issue<3>(bs_n);
            }
            if constexpr (!CPLX) {
                double af[MI], bf[NI];
#pragma unroll
                for (int i = 0; i < MI; ++i) af[i] = a_p[i * 8 * a_sx + kk * a_sk];
#pragma unroll
                for (int j = 0; j < NI; ++j) bf[j] = b_p[j * 8 * b_sx + kk * b_sk];
                if constexpr (SCALE) {
                    const double sc = s_s[kk + lc];
#pragma unroll
                    for (int i = 0; i < MI; ++i) af[i] *= sc;
                }
#pragma unroll
                for (int i = 0; i < MI; ++i)
#pragma unroll
                    for (int j = 0; j < NI; ++j) dmma(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
            } else {
                double ar[MI], ai[MI], nai[MI], br[NI], bi[NI];
#pragma unroll
                for (int i = 0; i < MI; ++i) {
                    const cplx v = a_p[i * 8 * a_sx + kk * a_sk];
                    ar[i] = v.x; ai[i] = conjA ? -v.y : v.y;
                }
#pragma unroll
                for (int j = 0; j < NI; ++j) {
                    const cplx v = b_p[j * 8 * b_sx + kk * b_sk];
                    br[j] = v.x; bi[j] = conjB ? -v.y : v.y;
                }
                if constexpr (SCALE) {
                    const double sc = s_s[kk + lc];
#pragma unroll
                    for (int i = 0; i < MI; ++i) { ar[i] *= sc; ai[i] *= sc; }
                }
#pragma unroll
                for (int i = 0; i < MI; ++i) nai[i] = -ai[i];
#pragma unroll
                for (int i = 0; i < MI; ++i)
#pragma unroll
                    for (int j = 0; j < NI; ++j) {
                        dmma(acc[i][j][0], acc[i][j][1], ar[i], br[j]);
                        dmma(acc[i][j][0], acc[i][j][1], nai[i], bi[j]);
                        dmma(acc[i][j][2], acc[i][j][3], ar[i], bi[j]);
                        dmma(acc[i][j][2], acc[i][j][3], ai[i], br[j]);
                    }
            }
        }
        fa.advance(); fb.advance();
        cp_async_commit();
    }
    cp_async_wait<0>();

    // epilogue: lane holds C[row = lr][cols 2*lc, 2*lc+1] of each 8x8 block
#pragma unroll
    for (int i = 0; i < MI; ++i) {
        const int gi = m0 + wm + i * 8 + lr;
        if (gi >= M) continue;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const int gj = n0 + wn + j * 8 + 2 * lc + q;
                if (gj >= N) continue;
                T *p = C + gi + (long)gj * ldc;
                if constexpr (!CPLX) {
                    double v = alpha * acc[i][j][q];
                    if (beta != 0.0 && !preload) v += beta * *p;
                    *p = v;
                } else {
                    cplx v; v.x = alpha * acc[i][j][q]; v.y = alpha * acc[i][j][2 + q];
                    if (beta != 0.0 && !preload) { const cplx o = *p; v.x += beta * o.x; v.y += beta * o.y; }
                    *p = v;
                }
            }
        }
    }
}

template <bool CPLX, bool NARROW> static size_t gemm_smem_bytes() {
    typedef Cfg<CPLX, NARROW> G;
    size_t a = TileSize<G::BM, G::BK, G::PADX, G::PADK>::value, b = TileSize<G::BN, G::BK, G::PADX, G::PADK>::value;
    return G::STAGES * (a + b) * sizeof(typename G::T) + G::STAGES * G::BK * sizeof(double);
}

template <bool CPLX, bool AXC, bool BXC, bool SCALE, bool NARROW, bool AL16>
static int launch_variant2(const GemmDesc *hd, const GemmDesc *dd, int ngroups, int max_m, int max_n, int batch,
                           cudaStream_t st) {
    typedef Cfg<CPLX, NARROW> G;
    static bool attr_set = false;
    size_t smem = gemm_smem_bytes<CPLX, NARROW>();
    if (!attr_set) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(gemm_kernel<CPLX, AXC, BXC, SCALE, NARROW, AL16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    long tiles = (long)ceil_div(max_m, G::BM) * ceil_div(max_n, G::BN);
    dim3 grid((unsigned)tiles, (unsigned)batch, (unsigned)ngroups);
    GemmDesc dummy = hd ? *hd : gemm_desc(0, 0, 0, 0, 0, 0, nullptr, 0, nullptr, 0, 0, nullptr, 0);
    const double flops = hd ? (CPLX ? 8.0 : 2.0) * hd->m * (double)hd->n * hd->k * (hd->cmode != 0 ? 0.5 : 1.0) *
                                  (hd->maskA != MASK_NONE || hd->maskB != MASK_NONE ? 0.5 : 1.0) * batch /
                                  (hd->ksplit > 1 ? hd->ksplit : 1)
                            : 0.0;
    if (!hd) prof_grouped_flops(dd, ngroups, (CPLX ? 8.0 : 2.0) * batch, st);
    const int pk = prof_kernel_begin(1, flops, st);
    gemm_kernel<CPLX, AXC, BXC, SCALE, NARROW, AL16><<<grid, GEMM_THREADS, smem, st>>>(dummy, dd);
    prof_kernel_end(1, pk, st);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

// Real operands that are not 16-byte aligned (odd row offsets such as Z + jb + 1, odd leading dimensions) take the
// instantiation whose fast loader copies 8 bytes at a time; device-side descriptors keep the 16-byte variant, which checks
// the alignment per CTA and falls back to the generic loader.
template <bool CPLX, bool AXC, bool BXC, bool SCALE, bool NARROW>
static int launch_variant(const GemmDesc *hd, const GemmDesc *dd, int ngroups, int max_m, int max_n, int batch,
                          cudaStream_t st) {
    if constexpr (!CPLX && !SCALE) {
        if (hd) {
            const bool al = (((size_t)hd->A | (size_t)hd->B) & 15) == 0 && ((hd->lda | hd->ldb | hd->sA | hd->sB) & 1) == 0;
            if (!al) return launch_variant2<CPLX, AXC, BXC, SCALE, NARROW, false>(hd, dd, ngroups, max_m, max_n, batch, st);
        }
    }
    return launch_variant2<CPLX, AXC, BXC, SCALE, NARROW, true>(hd, dd, ngroups, max_m, max_n, batch, st);
}

// the operand layouts (and the presence of scale factors) select the kernel instantiation; for grouped launches every
// descriptor must share them
template <bool CPLX>
static int launch_impl(const GemmDesc *hd, const GemmDesc *dd, int ngroups, int max_m, int max_n, int batch, int opA,
                       int opB, bool scale, cudaStream_t st) {
    if (max_m <= 0 || max_n <= 0 || batch <= 0 || ngroups <= 0) return NAO_OK;
    const bool axc = (opA == OP_N), bxc = (opB != OP_N);
    if (scale) {
        if (!(axc && bxc)) return NAO_ERR_UNSUPPORTED;
        return launch_variant<CPLX, true, true, true, false>(hd, dd, ngroups, max_m, max_n, batch, st);
    }
    if constexpr (!CPLX) {
        if (max_n <= Cfg<false, true>::BN) {
            if (axc) return bxc ? launch_variant<false, true, true, false, true>(hd, dd, ngroups, max_m, max_n, batch, st)
                                : launch_variant<false, true, false, false, true>(hd, dd, ngroups, max_m, max_n, batch, st);
            return bxc ? launch_variant<false, false, true, false, true>(hd, dd, ngroups, max_m, max_n, batch, st)
                       : launch_variant<false, false, false, false, true>(hd, dd, ngroups, max_m, max_n, batch, st);
        }
    }
    if (axc) return bxc ? launch_variant<CPLX, true, true, false, false>(hd, dd, ngroups, max_m, max_n, batch, st)
                        : launch_variant<CPLX, true, false, false, false>(hd, dd, ngroups, max_m, max_n, batch, st);
    return bxc ? launch_variant<CPLX, false, true, false, false>(hd, dd, ngroups, max_m, max_n, batch, st)
               : launch_variant<CPLX, false, false, false, false>(hd, dd, ngroups, max_m, max_n, batch, st);
}

int gemm_launch(int dtype, const GemmDesc &d, int batch, cudaStream_t st) {
    if (d.m <= 0 || d.n <= 0) return NAO_OK;
    const int by = batch * (d.ksplit > 1 ? d.ksplit : 1);
    return dtype == NAO_COMPLEX ? launch_impl<true>(&d, nullptr, 1, d.m, d.n, by, d.opA, d.opB, d.scaleK != nullptr, st)
                                : launch_impl<false>(&d, nullptr, 1, d.m, d.n, by, d.opA, d.opB, d.scaleK != nullptr, st);
}

template <class T>
__global__ void splitk_reduce_kernel(int m, int n, int ks, const T *P, T *C, long ldc, long sC, double alpha, double beta) {
    const long b = blockIdx.z;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    P += b * (long)ks * m * n; C += b * sC;
    for (int j = blockIdx.y; j < n; j += gridDim.y) {
        double sr = 0.0, si = 0.0;
        for (int s = 0; s < ks; ++s) {
            const T v = P[((long)s * n + j) * m + i];
            if constexpr (sizeof(T) == 16) { sr += v.x; si += v.y; } else { sr += v; }
        }
        T *c = C + i + (long)j * ldc;
        if constexpr (sizeof(T) == 16) {
            cplx o = make_double2(alpha * sr, alpha * si);
            if (beta != 0.0) { o.x += beta * c->x; o.y += beta * c->y; }
            *c = o;
        } else {
            double o = alpha * sr;
            if (beta != 0.0) o += beta * *c;
            *c = o;
        }
    }
}

int gemm_splitk(int dtype, const GemmDesc &d0, int batch, int ksplit, void *partial, cudaStream_t st) {
    if (d0.m <= 0 || d0.n <= 0 || batch <= 0) return NAO_OK;
    if (ksplit <= 1) return gemm_launch(dtype, d0, batch, st);
    GemmDesc d = d0;
    d.C = partial; d.ldc = d0.m; d.sC = (long)ksplit * d0.m * d0.n; d.sSplit = (long)d0.m * d0.n; d.ksplit = ksplit;
    d.alpha = 1.0; d.beta = 0.0; d.cmode = 0;
    if (int rc = gemm_launch(dtype, d, batch, st)) return rc;
    dim3 grid((unsigned)ceil_div(d0.m, 128), (unsigned)(d0.n < 4096 ? d0.n : 4096), (unsigned)batch);
    if (dtype == NAO_COMPLEX)
        splitk_reduce_kernel<cplx><<<grid, 128, 0, st>>>(d0.m, d0.n, ksplit, (const cplx *)partial, (cplx *)d0.C, d0.ldc, d0.sC, d0.alpha, d0.beta);
    else
        splitk_reduce_kernel<double><<<grid, 128, 0, st>>>(d0.m, d0.n, ksplit, (const double *)partial, (double *)d0.C, d0.ldc, d0.sC, d0.alpha, d0.beta);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}
int gemm_launch_grouped(int dtype, const GemmDesc *dd, int ngroups, int max_m, int max_n, int batch, int opA, int opB,
                        bool scale, cudaStream_t st) {
    return dtype == NAO_COMPLEX ? launch_impl<true>(nullptr, dd, ngroups, max_m, max_n, batch, opA, opB, scale, st)
                                : launch_impl<false>(nullptr, dd, ngroups, max_m, max_n, batch, opA, opB, scale, st);
}

}  // namespace nao

NAO_EXPORT int nao_gemm(int dtype, int opA, int opB, int m, int n, int k, double alpha, const void *dA, long lda,
                        long strideA, const void *dB, long ldb, long strideB, double beta, void *dC, long ldc,
                        long strideC, int batch, int uplo_c, void *cuda_stream) {
    using namespace nao;
    if (dtype != NAO_REAL && dtype != NAO_COMPLEX) return -1;
    if (opA < 0 || opA > 2) return -2;
    if (opB < 0 || opB > 2) return -3;
    if (m < 0) return -4;
    if (n < 0) return -5;
    if (k < 0) return -6;
    if (!dA && m > 0 && k > 0) return -8;
    if (!dB && n > 0 && k > 0) return -11;
    if (!dC && m > 0 && n > 0) return -15;
    if (batch < 0) return -18;
    GemmDesc d = gemm_desc(opA, opB, m, n, k, alpha, dA, lda, dB, ldb, beta, dC, ldc);
    d.sA = strideA; d.sB = strideB; d.sC = strideC; d.cmode = uplo_c ? 1 : 0;
    if (int rcb = nao::bind_device()) return rcb;
    return gemm_launch(dtype, d, batch, (cudaStream_t)cuda_stream);
}
