// trd2_back.cu -- back-transformation of the bulge-chasing stage: Z <- Q2 Z ("stage 2 then
// stage 1, blocked Householder GEMMs").
//
// Q2 = prod_s prod_k H_{s,k} (sweeps s ascending, steps k ascending; reflector (s,k) acts on rows s+1+kb .. s+(k+1)b).
// Reflectors are grouped in "diamonds": S-block I = sweeps s0 .. s0+NBK-1 (s0 = I*NBK) and step k give the group
//   G(I,k) = H_{s0,k} H_{s0+1,k} ... = I - V T V^H,   V = (b + NBK - 1) x NBK parallelogram (rows s0+1+kb ..).
// Reflectors of different steps of one sweep commute, and (s,k) overlaps (s',k+1) only for s' < s, so Q2 Z is obtained
// by applying the groups with I DESCENDING and, inside an S-block, k ASCENDING (checked against the sweep-by-sweep
// product in tests).  Columns of Z are independent.
//
// B200 design (round 2):
//   q2_pack_kernel   one CTA per diamond: T by the xLARFT recurrence, then the diamond is written as ONE contiguous,
//                    padded block [V (ci-major) | V (row-major, real only) | T (row-major)] in exactly the
//                    shared-memory layout the apply kernel reads, so that it arrives with a single 1-D TMA copy.
//   q2_apply_kernel  every WARP owns 8 or 16 columns of Z and keeps its 96-row window of them in REGISTERS, in the
//                    accumulator layout of mma.sync.m8n8k4 (lane = (column, row pair)).  The three products of a diamond
//                    are chained in registers in transposed form,
//                        W^T = Z_w^T conj(V),   W2^T = W^T T^T,   Z_w^T -= W2^T V^T,
//                    the accumulator fragments of one product being the A fragments of the next: the contraction index of
//                    a DMMA may be enumerated in any order, so k-step "even"/"odd" of an 8-row tile contracts over the rows
//                    2q / 2q+1 a lane already holds.  Only V and T are read from shared memory (B fragments, one 16-byte
//                    load feeds two k-steps): a third of the shared-memory traffic of a formulation that keeps Z, W and W2
//                    there, no block-wide barrier in the loop.  A producer warp streams the packed diamonds with
//                    cp.async.bulk (TMA) into a two-stage ring guarded by full/empty mbarriers; the 64 rows of Z that
//                    enter the window at the next step are prefetched with cp.async into a per-warp staging area; the 64
//                    rows that leave are stored from registers.
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>

namespace nao {

static const int Q2_NBK = 32;                 // sweeps per diamond
static const int Q2_LW = 96;                  // window rows (>= TRD2_B + Q2_NBK - 1), 12 tiles of 8
static const int Q2_NT = Q2_LW / 8;

// Packed diamond (elements of T).  Leading dimensions make every fragment load conflict free:
//   real:    16-byte loads of (k, k+1) pairs, quarter-warp = 2 rows x 4 pairs  ->  ld = 8 mod 16
//   complex: 16-byte loads of one element, quarter-warp = 2 rows x 4 elements 2 apart -> ld odd (1 mod 8)
template <class T> struct Q2P;
template <> struct Q2P<double> {
    static const int LDV = 104, LDVT = 40, LDT = 40, OFF_VT = Q2_NBK * 104, OFF_T = OFF_VT + Q2_LW * 40, BLK = OFF_T + Q2_NBK * 40;
    static const int CW = 16, LDS = 72;       // widest warp slab (columns), staging leading dimension (64 rows + pad)
};
template <> struct Q2P<cplx> {
    static const int LDV = 97, LDVT = 0, LDT = 33, OFF_VT = 0, OFF_T = Q2_NBK * 97, BLK = OFF_T + Q2_NBK * 33;
    static const int CW = 8, LDS = 65;
};

__host__ __device__ inline int q2_nwin(int n, int s0) {      // windows of the S-block starting at sweep s0
    return s0 + 1 <= n - 1 ? (n - 2 - s0) / TRD2_B + 1 : 0;
}
__host__ __device__ inline long q2_ngroups(int n) {
    long t = 0;
    for (int s0 = 0; s0 < n - 1; s0 += Q2_NBK) t += q2_nwin(n, s0);
    return t;
}

// ---------------------------------------------------------------------------------------------------------------------
// pack: V parallelogram of diamond (I, k) -> shared memory, T, packed block
// ---------------------------------------------------------------------------------------------------------------------
template <class T>
__global__ void __launch_bounds__(256) q2_pack_kernel(int n, const T *V2, long ldv, long sV2, const T *tau2, long sTau2,
                                                      T *Pk, long sPk) {
    typedef Ops<T> O;
    typedef Q2P<T> L;
    constexpr int NBK = Q2_NBK, b = TRD2_B, LW = Q2_LW;
    const int I = blockIdx.x, k = blockIdx.y, item = blockIdx.z;
    const int s0 = I * NBK;
    if (k >= q2_nwin(n, s0)) return;
    const int ns = min(NBK, n - 1 - s0);
    V2 += (long)item * sV2; tau2 += (long)item * sTau2; Pk += (long)item * sPk;
    long goff = 0;
    for (int s = 0; s < s0; s += NBK) goff += q2_nwin(n, s);
    T *out = Pk + (goff + k) * L::BLK;

    extern __shared__ __align__(16) unsigned char q2p_smem[];
    T *sV = (T *)q2p_smem;                    // [NBK][LDV]
    __shared__ T sG[NBK][NBK + 1], sT[NBK][NBK + 1], s_tau[NBK];
    const int tid = threadIdx.x;
    const int w0 = s0 + 1 + k * b;
    for (int e = tid; e < NBK * L::LDV; e += 256) {
        const int r = e % L::LDV, ci = e / L::LDV;
        const int s = s0 + ci, gr = w0 + r;
        T v = O::zero();
        if (r < LW && ci < ns && gr >= s + 1 + k * b && gr <= min(s + (k + 1) * b, n - 1)) v = V2[gr + (long)s * ldv];
        sV[e] = v;
    }
    if (tid < NBK) s_tau[tid] = tid < ns ? tau2[(long)k * n + s0 + tid] : O::zero();
    for (int e = tid; e < NBK * NBK; e += 256) sT[e / NBK][e % NBK] = O::zero();
    __syncthreads();
    // G = V^H V (upper part is what the recurrence reads)
    for (int e = tid; e < NBK * NBK; e += 256) {
        const int i = e % NBK, j = e / NBK;
        T s = O::zero();
        if (i < j) for (int r = 0; r < LW; ++r) s = O::add(s, O::conj_mul(sV[i * L::LDV + r], sV[j * L::LDV + r]));
        sG[i][j] = s;
    }
    __syncthreads();
    // T(i,i) = tau_i ; T(0:i, i) = -tau_i T(0:i,0:i) G(0:i, i)
    for (int i = 0; i < NBK; ++i) {
        if (tid < i) {
            T acc = O::zero();
            for (int c = tid; c < i; ++c) acc = O::fma(sT[tid][c], sG[c][i], acc);
            sT[tid][i] = O::sub(O::zero(), O::mul(s_tau[i], acc));
        }
        if (tid == i) sT[i][i] = s_tau[i];
        __syncthreads();
    }
    for (int e = tid; e < NBK * L::LDV; e += 256) out[e] = sV[e];
    if constexpr (L::LDVT > 0)
        for (int e = tid; e < LW * L::LDVT; e += 256) {
            const int ci = e % L::LDVT, r = e / L::LDVT;
            out[L::OFF_VT + e] = ci < NBK ? sV[ci * L::LDV + r] : O::zero();
        }
    for (int e = tid; e < NBK * L::LDT; e += 256) {
        const int kk = e % L::LDT, i = e / L::LDT;
        out[L::OFF_T + e] = kk < NBK ? sT[i][kk] : O::zero();
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// mbarrier / TMA helpers
// ---------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "Q2_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra Q2_DONE;\n"
        "bra Q2_WAIT;\n"
        "Q2_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one 1-D bulk copy global -> shared (TMA), completion counted in bytes on `bar`
__device__ __forceinline__ void tma_load_1d(void *smem_dst, const void *gsrc, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------------------------------------------------------------
// per-warp window of Z in registers.  Lane (lr = lane >> 2, lc = lane & 3) holds, for every 8-row tile t and column group
// mt, the rows 8t + 2lc and 8t + 2lc + 1 of column 8mt + lr (the C-fragment layout with M = column, N = row).
// ---------------------------------------------------------------------------------------------------------------------
template <class T, int MT> struct Q2Warp;

template <int MT> struct Q2Warp<double, MT> {
    typedef Q2P<double> L;
    double z[Q2_NT][MT][2];

    // rows [8 t0, 8 t1) of the window that starts at global row w0, straight from global memory
    __device__ __forceinline__ void load_global(const double *Z, long ldz, int n, int ncols, int c0, int w0, int t0, int t1, int lr, int lc) {
#pragma unroll
        for (int t = 0; t < Q2_NT; ++t) {
            if (t < t0 || t >= t1) continue;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int c = c0 + 8 * mt + lr, r = w0 + 8 * t + 2 * lc;
                const double *p = Z + (long)c * ldz + r;
                z[t][mt][0] = (c < ncols && r < n) ? p[0] : 0.0;
                z[t][mt][1] = (c < ncols && r + 1 < n) ? p[1] : 0.0;
            }
        }
    }
    // rows [0, nrows) of the window to global memory, tiles [0, t1)
    __device__ __forceinline__ void store_global(double *Z, long ldz, int ncols, int c0, int w0, int t1, int nrows, int lr, int lc) const {
#pragma unroll
        for (int t = 0; t < Q2_NT; ++t) {
            if (t >= t1) continue;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int c = c0 + 8 * mt + lr, rr = 8 * t + 2 * lc;
                double *p = Z + (long)c * ldz + w0 + rr;
                if (c < ncols && rr < nrows) p[0] = z[t][mt][0];
                if (c < ncols && rr + 1 < nrows) p[1] = z[t][mt][1];
            }
        }
    }
    // staging area [column][64 rows] (ld LDS) <- global rows [g0, g0 + 64), asynchronous
    __device__ __forceinline__ void stage_issue(double *stg, const double *Z, long ldz, int n, int ncols, int c0, int g0, int lane) const {
#pragma unroll
        for (int c = 0; c < 8 * MT; ++c) {
            const double *p = Z + (long)(c0 + c) * ldz + g0;
            const bool cok = c0 + c < ncols;
            cp_async8(stg + c * L::LDS + lane, cok && g0 + lane < n ? p + lane : Z, cok && g0 + lane < n);
            cp_async8(stg + c * L::LDS + 32 + lane, cok && g0 + 32 + lane < n ? p + 32 + lane : Z, cok && g0 + 32 + lane < n);
        }
    }
    // slide by 64 rows: tiles 8..11 -> 0..3, tiles 4..11 <- staging
    __device__ __forceinline__ void slide(const double *stg, int lr, int lc) {
#pragma unroll
        for (int t = 0; t < 4; ++t)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) { z[t][mt][0] = z[t + 8][mt][0]; z[t][mt][1] = z[t + 8][mt][1]; }
#pragma unroll
        for (int t = 4; t < Q2_NT; ++t)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const double2 v = *(const double2 *)(stg + (8 * mt + lr) * L::LDS + 8 * (t - 4) + 2 * lc);
                z[t][mt][0] = v.x; z[t][mt][1] = v.y;
            }
    }
    // one diamond: blk = packed [V | Vt | T] in shared memory
    __device__ __forceinline__ void apply(const double *blk, int lr, int lc) {
        const double *sV = blk, *sVt = blk + L::OFF_VT, *sT = blk + L::OFF_T;
        double w[4][MT][2], w2[4][MT][2];
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) { w[j][mt][0] = w[j][mt][1] = 0.0; w2[j][mt][0] = w2[j][mt][1] = 0.0; }
        // B fragments are fetched one step ahead of the DMMAs that use them (explicit double buffering: the compiler places a
        // shared-memory load right in front of its first use otherwise, and two or three warps per scheduler do not cover it)
        // W^T = Z_w^T V : row tile t meets reflector tile j iff j <= t <= j + 8 (parallelogram)
        {
            double2 bc[4], bn[4];
            bc[0] = *(const double2 *)(sV + lr * L::LDV + 2 * lc);
#pragma unroll
            for (int t = 0; t < Q2_NT; ++t) {
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (t + 1 < Q2_NT && j <= t + 1 && t + 1 <= j + 8) bn[j] = *(const double2 *)(sV + (8 * j + lr) * L::LDV + 8 * (t + 1) + 2 * lc);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (j > t || t > j + 8) continue;
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        dmma884(w[j][mt][0], w[j][mt][1], z[t][mt][0], bc[j].x);
                        dmma884(w[j][mt][0], w[j][mt][1], z[t][mt][1], bc[j].y);
                    }
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) bc[j] = bn[j];
            }
        }
        // W2^T = W^T T^T : T upper triangular, T[i][k] != 0 for k >= i
        {
            double2 bt[4][4];
#pragma unroll
            for (int ji = 0; ji < 4; ++ji)
#pragma unroll
                for (int u = ji; u < 4; ++u) bt[ji][u] = *(const double2 *)(sT + (8 * ji + lr) * L::LDT + 8 * u + 2 * lc);
#pragma unroll
            for (int ji = 0; ji < 4; ++ji)
#pragma unroll
                for (int u = ji; u < 4; ++u)
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        dmma884(w2[ji][mt][0], w2[ji][mt][1], w[u][mt][0], bt[ji][u].x);
                        dmma884(w2[ji][mt][0], w2[ji][mt][1], w[u][mt][1], bt[ji][u].y);
                    }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) { w2[j][mt][0] = -w2[j][mt][0]; w2[j][mt][1] = -w2[j][mt][1]; }
        // Z_w^T -= W2^T V^T
        {
            double2 bc[4], bn[4];
            bc[0] = *(const double2 *)(sVt + lr * L::LDVT + 2 * lc);
#pragma unroll
            for (int t = 0; t < Q2_NT; ++t) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (t + 1 < Q2_NT && u <= t + 1 && t + 1 <= u + 8) bn[u] = *(const double2 *)(sVt + (8 * (t + 1) + lr) * L::LDVT + 8 * u + 2 * lc);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (u > t || t > u + 8) continue;
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        dmma884(z[t][mt][0], z[t][mt][1], w2[u][mt][0], bc[u].x);
                        dmma884(z[t][mt][0], z[t][mt][1], w2[u][mt][1], bc[u].y);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) bc[u] = bn[u];
            }
        }
    }
};

template <int MT> struct Q2Warp<cplx, MT> {
    static_assert(MT == 1, "complex warps own 8 columns");
    typedef Q2P<cplx> L;
    double zr[Q2_NT][2], zi[Q2_NT][2];

    __device__ __forceinline__ void load_global(const cplx *Z, long ldz, int n, int ncols, int c0, int w0, int t0, int t1, int lr, int lc) {
#pragma unroll
        for (int t = 0; t < Q2_NT; ++t) {
            if (t < t0 || t >= t1) continue;
            const int c = c0 + lr, r = w0 + 8 * t + 2 * lc;
            const cplx *p = Z + (long)c * ldz + r;
            const cplx a = (c < ncols && r < n) ? p[0] : make_double2(0.0, 0.0);
            const cplx b2 = (c < ncols && r + 1 < n) ? p[1] : make_double2(0.0, 0.0);
            zr[t][0] = a.x; zi[t][0] = a.y; zr[t][1] = b2.x; zi[t][1] = b2.y;
        }
    }
    __device__ __forceinline__ void store_global(cplx *Z, long ldz, int ncols, int c0, int w0, int t1, int nrows, int lr, int lc) const {
#pragma unroll
        for (int t = 0; t < Q2_NT; ++t) {
            if (t >= t1) continue;
            const int c = c0 + lr, rr = 8 * t + 2 * lc;
            cplx *p = Z + (long)c * ldz + w0 + rr;
            if (c < ncols && rr < nrows) p[0] = make_double2(zr[t][0], zi[t][0]);
            if (c < ncols && rr + 1 < nrows) p[1] = make_double2(zr[t][1], zi[t][1]);
        }
    }
    __device__ __forceinline__ void stage_issue(cplx *stg, const cplx *Z, long ldz, int n, int ncols, int c0, int g0, int lane) const {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const cplx *p = Z + (long)(c0 + c) * ldz + g0;
            const bool cok = c0 + c < ncols;
            cp_async16(stg + c * L::LDS + lane, cok && g0 + lane < n ? p + lane : Z, cok && g0 + lane < n);
            cp_async16(stg + c * L::LDS + 32 + lane, cok && g0 + 32 + lane < n ? p + 32 + lane : Z, cok && g0 + 32 + lane < n);
        }
    }
    __device__ __forceinline__ void slide(const cplx *stg, int lr, int lc) {
#pragma unroll
        for (int t = 0; t < 4; ++t) { zr[t][0] = zr[t + 8][0]; zr[t][1] = zr[t + 8][1]; zi[t][0] = zi[t + 8][0]; zi[t][1] = zi[t + 8][1]; }
#pragma unroll
        for (int t = 4; t < Q2_NT; ++t) {
            const cplx *p = stg + lr * L::LDS + 8 * (t - 4) + 2 * lc;
            const cplx a = p[0], b2 = p[1];
            zr[t][0] = a.x; zi[t][0] = a.y; zr[t][1] = b2.x; zi[t][1] = b2.y;
        }
    }
    __device__ __forceinline__ void apply(const cplx *blk, int lr, int lc) {
        const cplx *sV = blk, *sT = blk + L::OFF_T;
        double wr[4][2], wi[4][2], vr[4][2], vi[4][2];
#pragma unroll
        for (int j = 0; j < 4; ++j) { wr[j][0] = wr[j][1] = wi[j][0] = wi[j][1] = 0.0; vr[j][0] = vr[j][1] = vi[j][0] = vi[j][1] = 0.0; }
        // (B fragments one step ahead of their DMMAs, as in the real case)
        // W^T = Z_w^T conj(V):  re += ar br + ai bi,  im += ai br - ar bi
        {
            cplx c0[4], c1[4], n0[4], n1[4];
            { const cplx *bp = sV + lr * L::LDV + 2 * lc; c0[0] = bp[0]; c1[0] = bp[1]; }
#pragma unroll
            for (int t = 0; t < Q2_NT; ++t) {
                const double nr0 = -zr[t][0], nr1 = -zr[t][1];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (t + 1 < Q2_NT && j <= t + 1 && t + 1 <= j + 8) {
                        const cplx *bp = sV + (8 * j + lr) * L::LDV + 8 * (t + 1) + 2 * lc;
                        n0[j] = bp[0]; n1[j] = bp[1];
                    }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    if (j > t || t > j + 8) continue;
                    const cplx b0 = c0[j], b1 = c1[j];
                    dmma884(wr[j][0], wr[j][1], zr[t][0], b0.x); dmma884(wr[j][0], wr[j][1], zi[t][0], b0.y);
                    dmma884(wi[j][0], wi[j][1], zi[t][0], b0.x); dmma884(wi[j][0], wi[j][1], nr0, b0.y);
                    dmma884(wr[j][0], wr[j][1], zr[t][1], b1.x); dmma884(wr[j][0], wr[j][1], zi[t][1], b1.y);
                    dmma884(wi[j][0], wi[j][1], zi[t][1], b1.x); dmma884(wi[j][0], wi[j][1], nr1, b1.y);
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) { c0[j] = n0[j]; c1[j] = n1[j]; }
            }
        }
        // W2^T = W^T T^T:  re += ar br - ai bi,  im += ar bi + ai br
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const double ni0 = -wi[u][0], ni1 = -wi[u][1];
            cplx t0[4], t1[4];
#pragma unroll
            for (int ji = 0; ji <= u; ++ji) {
                const cplx *bp = sT + (8 * ji + lr) * L::LDT + 8 * u + 2 * lc;
                t0[ji] = bp[0]; t1[ji] = bp[1];
            }
#pragma unroll
            for (int ji = 0; ji <= u; ++ji) {
                const cplx b0 = t0[ji], b1 = t1[ji];
                dmma884(vr[ji][0], vr[ji][1], wr[u][0], b0.x); dmma884(vr[ji][0], vr[ji][1], ni0, b0.y);
                dmma884(vi[ji][0], vi[ji][1], wr[u][0], b0.y); dmma884(vi[ji][0], vi[ji][1], wi[u][0], b0.x);
                dmma884(vr[ji][0], vr[ji][1], wr[u][1], b1.x); dmma884(vr[ji][0], vr[ji][1], ni1, b1.y);
                dmma884(vi[ji][0], vi[ji][1], wr[u][1], b1.y); dmma884(vi[ji][0], vi[ji][1], wi[u][1], b1.x);
            }
        }
        // Z_w^T -= W2^T V^T:  re += (-ar) br + ai bi,  im += (-ar) bi + (-ai) br      (V[row 8t + lr][i = 8u + 2lc (+1)])
        {
            double nvr[4][2], nvi[4][2];
#pragma unroll
            for (int u = 0; u < 4; ++u) { nvr[u][0] = -vr[u][0]; nvr[u][1] = -vr[u][1]; nvi[u][0] = -vi[u][0]; nvi[u][1] = -vi[u][1]; }
            cplx c0[4], c1[4], n0[4], n1[4];
            { const cplx *bp = sV + (2 * lc) * L::LDV + lr; c0[0] = bp[0]; c1[0] = bp[L::LDV]; }
#pragma unroll
            for (int t = 0; t < Q2_NT; ++t) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (t + 1 < Q2_NT && u <= t + 1 && t + 1 <= u + 8) {
                        const cplx *bp = sV + (8 * u + 2 * lc) * L::LDV + 8 * (t + 1) + lr;
                        n0[u] = bp[0]; n1[u] = bp[L::LDV];
                    }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (u > t || t > u + 8) continue;
                    const cplx b0 = c0[u], b1 = c1[u];
                    dmma884(zr[t][0], zr[t][1], nvr[u][0], b0.x); dmma884(zr[t][0], zr[t][1], vi[u][0], b0.y);
                    dmma884(zi[t][0], zi[t][1], nvr[u][0], b0.y); dmma884(zi[t][0], zi[t][1], nvi[u][0], b0.x);
                    dmma884(zr[t][0], zr[t][1], nvr[u][1], b1.x); dmma884(zr[t][0], zr[t][1], vi[u][1], b1.y);
                    dmma884(zi[t][0], zi[t][1], nvr[u][1], b1.y); dmma884(zi[t][0], zi[t][1], nvi[u][1], b1.x);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) { c0[u] = n0[u]; c1[u] = n1[u]; }
            }
        }
    }
};

// The per-warp walk through all diamonds for one slab of 8 MT columns starting at column c0.
template <class T, int MT>
__device__ __forceinline__ void q2_consumer(int n, int ncols, T *Z, long ldz, int c0, const T *ring, T *stg,
                                            unsigned long long *full, unsigned long long *empty) {
    typedef Q2P<T> L;
    constexpr int b = TRD2_B, NBK = Q2_NBK;
    const int lane = threadIdx.x & 31, lr = lane >> 2, lc = lane & 3;
    const int nsweeps = n - 1, nS = (nsweeps + NBK - 1) / NBK;
    Q2Warp<T, MT> W;
    unsigned d = 0;                                   // running diamond index (ring stage d & 1, phase (d >> 1) & 1)
    for (int I = nS - 1; I >= 0; --I) {
        const int s0 = I * NBK, ns = min(NBK, nsweeps - s0), nwin = q2_nwin(n, s0);
        for (int k = 0; k < nwin; ++k, ++d) {
            const int w0 = s0 + 1 + k * b;
            const int Lw = min(s0 + ns - 1 + (k + 1) * b, n - 1) - w0 + 1;      // rows of the window the diamond touches
            if (k == 0) {
                __syncwarp();                         // the rows were stored by other lanes of this warp (previous S-block)
                W.load_global(Z, ldz, n, ncols, c0, w0, 0, Q2_NT, lr, lc);
            } else {
                cp_async_wait<0>();
                __syncwarp();
                W.slide(stg, lr, lc);
                __syncwarp();                         // everybody has read the staging area before it is refilled
            }
            if (k + 1 < nwin) W.stage_issue(stg, Z, ldz, n, ncols, c0, w0 + b + NBK, lane);      // rows entering at step k + 1
            cp_async_commit();
            mbar_wait(full + (d & 1), (d >> 1) & 1);
            W.apply(ring + (size_t)(d & 1) * L::BLK, lr, lc);
            __syncwarp();
            // The refill of this ring stage is a write through the async proxy (TMA); the fragment loads above went through
            // the generic proxy.  Without a proxy fence before the release nothing orders the two: with nine warps per CTA
            // (config 3) a refill now and then overtook the last reads of the warp that runs ahead of the others.
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            if (lane == 0) mbar_arrive(empty + (d & 1));
            const bool last = (k + 1 == nwin);
            if (last) {
                W.store_global(Z, ldz, ncols, c0, w0, Q2_NT, Lw, lr, lc);
            } else {
                W.store_global(Z, ldz, ncols, c0, w0, 8, b, lr, lc);
            }
        }
    }
    cp_async_wait<0>();
}

// n2 of the NW consumer warps own 16 columns (real only), the others 8; warp NW is the TMA producer.
// MAXW = most consumer warps (bounds the registers per thread); MT2 = 16-column warps allowed (real only).
template <class T, int MAXW, bool MT2>
__global__ void __launch_bounds__((MAXW + 1) * 32, 1) q2_apply_kernel(int n, int ncols, const T *Pk, long sPk, T *Z, long ldz, long sZ,
                                                                         int NW, int n2) {
    typedef Q2P<T> L;
    constexpr int NBK = Q2_NBK;
    const int item = blockIdx.y;
    Pk += (long)item * sPk; Z += (long)item * sZ;
    extern __shared__ __align__(128) unsigned char q2_smem[];
    T *ring = (T *)q2_smem;                                              // [2][BLK]
    constexpr int CWS = (sizeof(T) == 8 && MT2) ? 16 : 8;                // columns of a warp's staging area
    T *stg_all = ring + 2 * L::BLK;                                      // [NW][CWS * LDS]
    unsigned long long *bars = (unsigned long long *)(stg_all + (size_t)NW * CWS * L::LDS);       // full[2], empty[2]
    unsigned long long *full = bars, *empty = bars + 2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(full, 1); mbar_init(full + 1, 1);
        mbar_init(empty, NW); mbar_init(empty + 1, NW);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    }
    __syncthreads();
    const int cols_cta = 16 * n2 + 8 * (NW - n2);
    const int cta_c0 = blockIdx.x * cols_cta;
    if (warp == NW) {
        // ---- producer: diamonds in application order (I descending, k ascending), two in flight
        if (lane == 0) {
            const int nsweeps = n - 1, nS = (nsweeps + NBK - 1) / NBK;
            long goff = q2_ngroups(n);
            unsigned d = 0;
            for (int I = nS - 1; I >= 0; --I) {
                const int nwin = q2_nwin(n, I * NBK);
                goff -= nwin;
                for (int k = 0; k < nwin; ++k, ++d) {
                    if (d >= 2) mbar_wait(empty + (d & 1), ((d >> 1) - 1) & 1);
                    mbar_expect_tx(full + (d & 1), (unsigned)(L::BLK * sizeof(T)));
                    tma_load_1d(ring + (size_t)(d & 1) * L::BLK, Pk + (goff + k) * L::BLK, (unsigned)(L::BLK * sizeof(T)), full + (d & 1));
                }
            }
        }
        return;
    }
    if (warp > NW) return;
    T *stg = stg_all + (size_t)warp * CWS * L::LDS;
    if constexpr (sizeof(T) == 8 && MT2) {
        if (warp < n2) q2_consumer<T, 2>(n, ncols, Z, ldz, cta_c0 + 16 * warp, ring, stg, full, empty);
        else q2_consumer<T, 1>(n, ncols, Z, ldz, cta_c0 + 16 * n2 + 8 * (warp - n2), ring, stg, full, empty);
    } else {
        q2_consumer<T, 1>(n, ncols, Z, ldz, cta_c0 + 8 * warp, ring, stg, full, empty);
    }
}

size_t q2_workspace(int dtype, int n, int batch) {
    const size_t blk = dtype == NAO_COMPLEX ? (size_t)Q2P<cplx>::BLK * 16 : (size_t)Q2P<double>::BLK * 8;
    return align_up((size_t)batch * q2_ngroups(n) * blk);
}

template <class T>
static int q2_apply_impl(int n, int ncols, int batch, const T *V2, long ldv, long sV2, const T *tau2, T *Z, long ldz, long sZ,
                         void *work, cudaStream_t st) {
    typedef Q2P<T> L;
    if (n < 2 || ncols < 1) return NAO_OK;
    const long ng = q2_ngroups(n), sPk = ng * L::BLK, sTau2 = (long)hb2st_nk(n) * n;
    T *Pk = (T *)work;
    const int nS = ceil_div(n - 1, Q2_NBK), kmax = q2_nwin(n, 0);
    const size_t smem_p = (size_t)Q2_NBK * L::LDV * sizeof(T);
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(q2_pack_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_p));
        attr = true;
    }
    q2_pack_kernel<T><<<dim3(nS, kmax, batch), 256, smem_p, st>>>(n, V2, ldv, sV2, tau2, sTau2, Pk, sPk);
    NAO_LAUNCHED();
    // Columns per CTA: one CTA per SM walks through all diamonds, so the slab width is what gives every SM the same share.
    // Units of 8 columns, spread over the four schedulers of an SM: u units per scheduler as 16-column warps (real) plus at
    // most one 8-column warp each.
    // (sm_count(): under NAO_STREAM_GROUPS_* a group's share of the SMs, so that the groups' kernels run side by side)
    const int nsm = sm_count();
    const long units_sm = std::max(1L, ((long)ceil_div(ncols, 8) * batch + nsm - 1) / nsm);      // 8-column units per SM
    int NW, n2 = 0;
    bool wide = false;                                               // 12 eight-column warps (three per scheduler)
    if (sizeof(T) == 8) {
        const int u = (int)std::min(4L, (units_sm + 3) / 4);          // units per scheduler
        if (units_sm <= 2) { NW = (int)units_sm; n2 = 0; }
        else if (u == 1) { NW = 4; n2 = 0; }
        else if (u == 2) { NW = 4; n2 = 4; }
        else if (u == 3) { NW = 12; n2 = 0; wide = true; }
        else { NW = 8; n2 = 8; }
    } else {
        NW = (int)std::min(9L, units_sm);
    }
    const int cols_cta = 16 * n2 + 8 * (NW - n2);
    const int cws = (sizeof(T) == 8 && !wide) ? 16 : 8;               // staging columns per warp (kernel's CWS)
    const size_t smem = (size_t)2 * L::BLK * sizeof(T) + (size_t)NW * cws * L::LDS * sizeof(T) + 64;
    const dim3 grid(ceil_div(ncols, cols_cta), batch);
    // (kernel instantiations share one function-pointer type: the attribute flag is kept per instantiation, not per lambda)
    auto launch = [&](auto kernel, int maxw, bool &attr_set) -> int {
        if (!attr_set) {
            const size_t smem_max = (size_t)2 * L::BLK * sizeof(T) + (size_t)maxw * cws * L::LDS * sizeof(T) + 64;
            NAO_CUDA_CHECK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
            attr_set = true;
        }
        kernel<<<grid, (NW + 1) * 32, smem, st>>>(n, ncols, Pk, sPk, Z, ldz, sZ, NW, n2);
        return NAO_OK;
    };
    static bool set_wide = false, set_mixed = false, set_cplx = false;
    int rc;
    if constexpr (sizeof(T) == 8) {
        if (wide) rc = launch(q2_apply_kernel<T, 12, false>, 12, set_wide);
        else rc = launch(q2_apply_kernel<T, 8, true>, 8, set_mixed);
    } else {
        rc = launch(q2_apply_kernel<T, 9, false>, 9, set_cplx);
    }
    if (rc) return rc;
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int q2_apply(int dtype, int n, int ncols, int batch, const void *V2, long ldv, long sV2, const void *tau2, void *Z, long ldz,
             long sZ, void *work, cudaStream_t st) {
    return dtype == NAO_COMPLEX
               ? q2_apply_impl<cplx>(n, ncols, batch, (const cplx *)V2, ldv, sV2, (const cplx *)tau2, (cplx *)Z, ldz, sZ, work, st)
               : q2_apply_impl<double>(n, ncols, batch, (const double *)V2, ldv, sV2, (const double *)tau2, (double *)Z, ldz, sZ, work, st);
}

}  // namespace nao
