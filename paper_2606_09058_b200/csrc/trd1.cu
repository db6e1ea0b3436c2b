// trd1.cu -- one-stage Householder tridiagonalisation (SURVEY.md 8a row a3/a4 role, 8d ambiguity M1: this is the
// HBM-bound "BLAS2 half" the paper describes for the one-stage reduction).
//
// Algorithm: LAPACK xHETRD/xLATRD, lower storage, panels of NB columns.  Inside a panel the trailing matrix is NOT
// updated; column j is brought up to date with the panel's (V, W), a reflector is generated, and
//   w = tau (A22 v - V (W^H v) - W (V^H v)) - 1/2 |tau|^2 (v^H A22 v - 2 Re (W^H v)^H (V^H v)) v
// is appended.  After the panel A22 -= V W^H + W V^H runs on the DMMA GEMM core.
//
// B200 design: ONE cooperative persistent kernel per panel.  The G CTAs that work on an item are co-resident and meet
// at a software grid barrier only TWICE per column:
//   phase A: finalise w of the previous column for the CTA's own rows, update column j, partial norm   | barrier
//   phase B: reflector scalars (every CTA, redundantly), v written to A, partial W^H v / V^H v,
//            HEMV of the lower triangle, partial v^H A v                                               | barrier
// The CTA's own rows of the panel's V and W live in shared memory for the whole panel.
//
// HEMV (the HBM-bound part): the lower triangle is cut into units of 64 rows x SW columns (SW = 64 real, 32 complex),
// enumerated strip by strip (column-major), and every WARP owns a contiguous run of units -- the loop has no
// __syncthreads at all.  Within a unit a lane owns 4 rows (q, q+16, q+32, q+48: each half-warp reads 128/256
// contiguous bytes per column) and half of the strip's columns; every element is loaded once (ld.global.cg, next
// batch in flight while the current one is used) and used for both its row and its column contribution:
//   row sums   : complete per unit in registers, halves combined with one shuffle, written to Prow[strip][row]
//   column sums: accumulated in registers over the whole run of units in the strip, reduced across lanes ONCE per
//                run by a 16-lane transpose-reduction and written to Pcol[first row block of the run][column]
// Every cross-CTA reduction goes through such partial buffers summed in a fixed order: results are bit-reproducible
// (no floating-point atomics).
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <cooperative_groups.h>

namespace nao {

static const int TRD_NB = 32;        // panel width
static const int TRD_NT = 256;       // threads per CTA
static const int TRD_NW = TRD_NT / 32;
static const int TRD_TB = 64;        // rows per HEMV unit / block edge
static const int TRD_CH = 96;        // rows of V/W cached in shared memory per CTA
static const int TRD_CHP = TRD_CH + 1;
static const int TRD_PASS = 128;     // rows finalised per pass in phase A


template <class T> struct Hv;
template <> struct Hv<double> { static const int SW = 32, CPT = 16, HS = 2, CB = 4; };   // 64 x 32 units: finer load balance
template <> struct Hv<cplx> { static const int SW = 32, CPT = 16, HS = 2, CB = 2; };

template <class T> struct TrdArgs {
    T *A; long lda, sA;
    double *d, *e; T *tau;           // per item: n each
    T *Wp;                           // per item: n x 4NB (ld n): [V | W | W | V] so that A22 -= [V W][W V]^H is one GEMM
    T *acol;                         // per item: n
    double *pn;                      // per item: G
    T *pt;                           // per item: G x 2NB
    double *pvav;                    // per item: G
    T *Prow, *Pcol;                  // per item: (HS*nblk) x n and nblk x n
    unsigned *bar;                   // per item: one counter for this launch
    int n, j0, nbp, G, nblk;
};

__device__ __forceinline__ double block_sum_d(double v, double *red /* TRD_NW */) {
    v = warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < TRD_NW; ++w) s += red[w];
    __syncthreads();
    return s;
}

// units of the lower triangle of an nbk x nbk block matrix, strip-major: block column J', half h, row block I >= J'
__device__ __forceinline__ int tri_off(int Jp, int nbk) { return Jp * nbk - Jp * (Jp - 1) / 2; }
__device__ __forceinline__ int tri_decode(int t, int nbk) {      // largest J' with tri_off(J') <= t
    const double b = 2.0 * nbk + 1.0;
    int Jp = (int)((b - sqrt(fmax(b * b - 8.0 * (double)t, 0.0))) * 0.5);
    Jp = max(0, min(Jp, nbk - 1));
    while (Jp + 1 < nbk && tri_off(Jp + 1, nbk) <= t) ++Jp;
    while (Jp > 0 && tri_off(Jp, nbk) > t) --Jp;
    return Jp;
}
template <int HS> __device__ __forceinline__ void unit_decode(int u, int nbk, int &Jp, int &h, int &Irel) {
    Jp = tri_decode(u / HS, nbk);
    const int len = nbk - Jp, w = u - HS * tri_off(Jp, nbk);
    h = w / len; Irel = Jp + w % len;
}
__device__ __forceinline__ int units_per_warp(int U, int G) { return (U + G * TRD_NW - 1) / (G * TRD_NW); }

__device__ __forceinline__ double shfl_xor_T(double v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }
__device__ __forceinline__ cplx shfl_xor_T(cplx v, int o) {
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, o), __shfl_xor_sync(0xffffffffu, v.y, o));
}

// Transpose-reduction over the 16 lanes of a half-warp: every lane enters with NV partial sums cs[0..NV) and leaves
// with the complete sums of indices q*(NV/16) + i, i < NV/16, in cs[0..NV/16)  (q = lane & 15).  Fixed tree order.
template <class T, int N, int NV, int XO>
__device__ __forceinline__ void treduce16(T (&cs)[N], int lane) {
    if constexpr (XO >= 1) {
        constexpr int half = NV / 2;
        const bool up = (lane & XO) != 0;
#pragma unroll
        for (int i = 0; i < half; ++i) {
            const T send = up ? cs[i] : cs[i + half];
            const T keep = up ? cs[i + half] : cs[i];
            cs[i] = Ops<T>::add(keep, shfl_xor_T(send, XO));
        }
        treduce16<T, N, half, XO / 2>(cs, lane);
    }
}

// HEMV y = A22 v over this warp's run of units (see the header).  Returns the lane's share of v^H A22 v.
template <class T>
__device__ __forceinline__ double hemv_warp(const T *__restrict__ A, long lda, int n, int j, int nblk, int G, int g,
                                            const T *acol, T scale, T *sx, T *__restrict__ Prow, T *__restrict__ Pcol) {
    typedef Ops<T> O;
    typedef Hv<T> H;
    constexpr int SW = H::SW, CPT = H::CPT, HS = H::HS, CB = H::CB, NBATCH = CPT / CB, CPL = CPT / 16;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, q = lane & 15, hh = lane >> 4;
    const int bmin = (j + 1) / TRD_TB, nbk = nblk - bmin;
    const int U = HS * (nbk * (nbk + 1) / 2);
    const int per = units_per_warp(U, G);
    const int gw = g * TRD_NW + warp;
    const int u0 = min(U, gw * per), u1 = min(U, u0 + per);
    if (u0 >= u1) return 0.0;

    auto vval = [&](int x) -> T {
        if (x < j + 1 || x >= n) return O::zero();
        if (x == j + 1) return O::one();
        return O::mul(ldcg(acol + x), scale);
    };
    auto load = [&](T (&buf)[CB][4], int Jp_, int h_, int Irel_, int b) {
        const int rbase = (bmin + Irel_) * TRD_TB + q;
        const int cbase = (bmin + Jp_) * TRD_TB + h_ * SW + hh * CPT + b * CB;
        const bool diag = (Irel_ == Jp_);
#pragma unroll
        for (int cc = 0; cc < CB; ++cc) {
            const int col = cbase + cc;
            const T *pc = A + (long)col * lda + rbase;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int r = rbase + 16 * k;
                const bool ok = r < n && col < n && (!diag || r >= col);
                T v = O::zero();
                if (ok) v = ldcg(pc + 16 * k);
                buf[cc][k] = v;
            }
        }
    };

    int Jp, h, Irel;
    unit_decode<HS>(u0, nbk, Jp, h, Irel);
    double vav = 0.0;
    T cs[CPT];
    T cur[CB][4], nxt[CB][4];
    int runI = Irel;
    auto strip_begin = [&](int Jp_, int h_) {
        __syncwarp();
        for (int c = lane; c < SW; c += 32) sx[c] = vval((bmin + Jp_) * TRD_TB + h_ * SW + c);
        __syncwarp();
#pragma unroll
        for (int c = 0; c < CPT; ++c) cs[c] = O::zero();
    };
    strip_begin(Jp, h);
    load(cur, Jp, h, Irel, 0);
    // x for the rows of the NEXT unit is fetched (L2) one unit ahead, like the matrix batches
    T xr_n[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) xr_n[k] = vval((bmin + Irel) * TRD_TB + q + 16 * k);

    for (int u = u0; u < u1; ++u) {
        int Jn = Jp, hn = h, In = Irel + 1;
        if (In >= nbk) {
            hn = h + 1;
            if (hn >= HS) { hn = 0; Jn = Jp + 1; }
            In = Jn;
        }
        const bool more = (u + 1 < u1);
        const bool diag = (Irel == Jp);
        const int rbase = (bmin + Irel) * TRD_TB + q;
        const int cb0 = (bmin + Jp) * TRD_TB + h * SW + hh * CPT;
        T xr[4], rs[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) { xr[k] = xr_n[k]; rs[k] = O::zero(); }
        if (more) {
#pragma unroll
            for (int k = 0; k < 4; ++k) xr_n[k] = vval((bmin + In) * TRD_TB + q + 16 * k);
        }
        // Two register buffers used alternately WITHOUT copying between them: a copy "cur = nxt" would have to wait for
        // nxt before the following request is issued, leaving one batch in flight per warp; this way the request for
        // batch b+2 is issued before the first use of batch b+1 (two batches = 8 KB per warp in flight).
        auto consume = [&](T (&buf)[CB][4], int b) {
#pragma unroll
            for (int cc = 0; cc < CB; ++cc) {
                const T xc = sx[hh * CPT + b * CB + cc];
                const int col = cb0 + b * CB + cc;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    T a = buf[cc][k], ac = a;
                    if (diag) {
                        const int r = rbase + 16 * k;
                        if (r == col) a = O::from_real(O::real(a));
                        if (r <= col) ac = O::zero();
                    }
                    rs[k] = O::fma(a, xc, rs[k]);
                    cs[b * CB + cc] = O::add(cs[b * CB + cc], O::conj_mul(ac, xr[k]));
                }
            }
        };
        static_assert(NBATCH % 2 == 0, "ping-pong buffers need an even number of batches per unit");
#pragma unroll
        for (int b = 0; b < NBATCH; b += 2) {
            load(nxt, Jp, h, Irel, b + 1);
            consume(cur, b);
            if (b + 2 < NBATCH) load(cur, Jp, h, Irel, b + 2);
            else if (more) load(cur, Jn, hn, In, 0);
            consume(nxt, b + 1);
        }
        // row sums of this unit: combine the two column halves, lanes 0..15 write 4 x 16 consecutive rows
#pragma unroll
        for (int k = 0; k < 4; ++k) rs[k] = O::add(rs[k], shfl_xor_T(rs[k], 16));
        if (hh == 0) {
            T *pr = Prow + (long)(HS * (bmin + Jp) + h) * n;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int r = rbase + 16 * k;
                if (r < n) { pr[r] = rs[k]; vav += O::real(O::conj_mul(xr[k], rs[k])); }
            }
        }
        if (!more || Jn != Jp || hn != h) {
            // end of this warp's run in the strip: one cross-lane reduction of the column sums
            treduce16<T, CPT, CPT, 8>(cs, lane);
            T *pcl = Pcol + (long)(bmin + runI) * n;
#pragma unroll
            for (int c = 0; c < CPL; ++c) {
                const int col = cb0 + q * CPL + c;
                if (col < n) { pcl[col] = cs[c]; vav += O::real(O::conj_mul(sx[hh * CPT + q * CPL + c], cs[c])); }
            }
            if (more) { strip_begin(Jn, hn); runI = In; }
        }
        Jp = Jn; h = hn; Irel = In;
    }
    return vav;
}

// ---------------------------------------------------------------------------------------------------------------------
// TMA-fed HEMV (n a multiple of 64, 16-byte aligned columns).  The matrix bytes no longer pass through registers on their
// way in: every warp owns a small ring of 4 KB stages in shared memory (64 rows x 8 real / 4 complex columns of a unit),
// filled by 1-D bulk copies (cp.async.bulk, one 64-row column segment per copy, completion counted on an mbarrier) that the
// warp issues for itself TRD_S stages ahead.  The stream of stages is continuous over the columns of the launch: while the
// CTA sits in the reductions and grid barriers of column j+1 the first stages of that column's run are already landing
// (the trailing matrix does not change inside a panel).  Lane l owns rows 2l, 2l+1 (real) / l, l+32 (complex) of a unit and
// all of its columns: row sums complete in registers per unit, column sums accumulate in registers over the warp's run in a
// strip and are reduced across the 32 lanes once per run, exactly the partial-sum layout of hemv_warp (Prow / Pcol).
// ---------------------------------------------------------------------------------------------------------------------
template <class T> struct HvT {
    static const int SC = sizeof(T) == 8 ? 8 : 4;        // columns per stage
    static const int NSUB = 32 / SC;                     // stages per 64 x 32 unit
    static const int STAGE = 64 * SC;                    // elements per stage (4096 bytes)
    static const int S = sizeof(T) == 8 ? 4 : 3;         // stages per warp
};

__device__ __forceinline__ unsigned trd_smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void trd_mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "TRD_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra TRD_DONE;\n"
        "bra TRD_WAIT;\n"
        "TRD_DONE:\n"
        "}\n" ::"r"(trd_smem_u32(bar)), "r"(parity) : "memory");
}

// Position in this warp's stream of stages: column i of the launch, unit u of its run [., u1), sub-stage q.
struct TrdCursor {
    int i, u, u1, q, Jp, h, Irel, bmin, nbk;
};
template <int HS>
__device__ __forceinline__ bool trd_cursor_column(TrdCursor &c, int i, int nbp, int j0, int nblk, int G, int gw) {
    // first column >= i with a non-empty run for this warp; false when the launch has none left
    for (; i < nbp; ++i) {
        const int j = j0 + i;
        c.bmin = (j + 1) / TRD_TB; c.nbk = nblk - c.bmin;
        const int U = HS * (c.nbk * (c.nbk + 1) / 2);
        const int per = units_per_warp(U, G);
        const int u0 = min(U, gw * per);
        c.u1 = min(U, u0 + per);
        if (u0 < c.u1) {
            c.i = i; c.u = u0; c.q = 0;
            unit_decode<HS>(u0, c.nbk, c.Jp, c.h, c.Irel);
            return true;
        }
    }
    c.i = nbp;
    return false;
}
template <int HS, int NSUB>
__device__ __forceinline__ void trd_cursor_next(TrdCursor &c, int nbp, int j0, int nblk, int G, int gw) {
    if (++c.q < NSUB) return;
    c.q = 0;
    if (++c.u < c.u1) {
        if (++c.Irel >= c.nbk) {
            if (++c.h >= HS) { c.h = 0; ++c.Jp; }
            c.Irel = c.Jp;
        }
        return;
    }
    trd_cursor_column<HS>(c, c.i + 1, nbp, j0, nblk, G, gw);
}

template <class T> struct TrdRing {
    T *buf;                          // this warp's S stages
    unsigned long long *full;        // S mbarriers
    unsigned pseq, cseq;             // stages issued / consumed since the start of the launch
    TrdCursor pc;                    // producer cursor
    bool more;                       // the producer cursor still points at a stage of this launch
};

// issue the bulk copies of the stage under the producer cursor into ring slot pseq % S
template <class T>
__device__ __forceinline__ void trd_issue(TrdRing<T> &r, const T *A, long lda, int lane) {
    typedef HvT<T> HT;
    const unsigned slot = r.pseq % HT::S;
    const int col = (r.pc.bmin + r.pc.Jp) * TRD_TB + r.pc.h * 32 + r.pc.q * HT::SC + lane;
    const int rbase = (r.pc.bmin + r.pc.Irel) * TRD_TB;
    const unsigned bar = trd_smem_u32(r.full + slot);
    if (lane == 0) asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(4096u) : "memory");
    __syncwarp();
    if (lane < HT::SC) {
        const T *src = A + (long)col * lda + rbase;
        const unsigned dst = trd_smem_u32(r.buf + (size_t)slot * HT::STAGE + lane * 64);
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(dst), "l"(src),
                     "r"((unsigned)(64 * sizeof(T))), "r"(bar)
                     : "memory");
    }
    ++r.pseq;
}

template <class T>
__device__ __forceinline__ double hemv_warp_tma(TrdRing<T> &ring, const T *__restrict__ A, long lda, int n, int j, int i, int nbp, int j0,
                                                int nblk, int G, int g, const T *acol, T scale, T *sx, T *__restrict__ Prow,
                                                T *__restrict__ Pcol) {
    typedef Ops<T> O;
    typedef Hv<T> H;
    typedef HvT<T> HT;
    constexpr int SW = H::SW, HS = H::HS, SC = HT::SC, NSUB = HT::NSUB;
    static_assert(SW == 32, "a stage stream assumes 32-column strips");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int bmin = (j + 1) / TRD_TB, nbk = nblk - bmin;
    const int U = HS * (nbk * (nbk + 1) / 2);
    const int per = units_per_warp(U, G);
    const int gw = g * TRD_NW + warp;
    const int u0 = min(U, gw * per), u1 = min(U, u0 + per);
    if (u0 >= u1) return 0.0;

    auto vval = [&](int x) -> T {
        if (x < j + 1 || x >= n) return O::zero();
        if (x == j + 1) return O::one();
        return O::mul(ldcg(acol + x), scale);
    };
    // rows of a unit owned by this lane: real 2l, 2l+1; complex l, l+32
    const int ro0 = O::is_complex ? lane : 2 * lane, ro1 = O::is_complex ? lane + 32 : 2 * lane + 1;

    int Jp, h, Irel;
    unit_decode<HS>(u0, nbk, Jp, h, Irel);
    double vav = 0.0;
    T cs[SW];
    int runI = Irel;
    auto strip_begin = [&](int Jp_, int h_) {
        __syncwarp();
        sx[lane] = vval((bmin + Jp_) * TRD_TB + h_ * SW + lane);
        __syncwarp();
#pragma unroll
        for (int c = 0; c < SW; ++c) cs[c] = O::zero();
    };
    strip_begin(Jp, h);
    T xr_n0 = vval((bmin + Irel) * TRD_TB + ro0), xr_n1 = vval((bmin + Irel) * TRD_TB + ro1);

    for (int u = u0; u < u1; ++u) {
        int Jn = Jp, hn = h, In = Irel + 1;
        if (In >= nbk) {
            hn = h + 1;
            if (hn >= HS) { hn = 0; Jn = Jp + 1; }
            In = Jn;
        }
        const bool more = (u + 1 < u1);
        const bool diag = (Irel == Jp);
        const int rbase = (bmin + Irel) * TRD_TB;
        const int cb0 = (bmin + Jp) * TRD_TB + h * SW;
        const T xr0 = xr_n0, xr1 = xr_n1;
        T rs0 = O::zero(), rs1 = O::zero();
        if (more) { xr_n0 = vval((bmin + In) * TRD_TB + ro0); xr_n1 = vval((bmin + In) * TRD_TB + ro1); }
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            const unsigned slot = ring.cseq % HT::S;
            trd_mbar_wait(ring.full + slot, (ring.cseq / HT::S) & 1);
            const T *tile = ring.buf + (size_t)slot * HT::STAGE;
            T a0[SC], a1[SC];
#pragma unroll
            for (int c = 0; c < SC; ++c) {
                if constexpr (O::is_complex) { a0[c] = tile[c * 64 + lane]; a1[c] = tile[c * 64 + 32 + lane]; }
                else { const double2 v = *(const double2 *)(tile + c * 64 + 2 * lane); a0[c] = v.x; a1[c] = v.y; }
            }
            // the slot is free again: refill it with the stage S ahead in the stream (this or a later column)
            __syncwarp();
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            ++ring.cseq;
            if (ring.more) {
                trd_issue<T>(ring, A, lda, lane);
                trd_cursor_next<HS, NSUB>(ring.pc, nbp, j0, nblk, G, gw);
                ring.more = ring.pc.i < nbp;
            }
#pragma unroll
            for (int c = 0; c < SC; ++c) {
                const T xc = sx[q * SC + c];
                T v0 = a0[c], v1 = a1[c], c0 = v0, c1 = v1;
                if (diag) {
                    const int col = cb0 + q * SC + c, r0 = rbase + ro0, r1 = rbase + ro1;
                    if (r0 == col) v0 = O::from_real(O::real(v0));
                    if (r1 == col) v1 = O::from_real(O::real(v1));
                    if (r0 < col) v0 = O::zero();
                    if (r1 < col) v1 = O::zero();
                    c0 = r0 <= col ? O::zero() : v0;
                    c1 = r1 <= col ? O::zero() : v1;
                }
                rs0 = O::fma(v0, xc, rs0);
                rs1 = O::fma(v1, xc, rs1);
                cs[q * SC + c] = O::add(cs[q * SC + c], O::add(O::conj_mul(c0, xr0), O::conj_mul(c1, xr1)));
            }
        }
        // row sums of this unit
        {
            T *pr = Prow + (long)(HS * (bmin + Jp) + h) * n + rbase;
            if constexpr (O::is_complex) { pr[ro0] = rs0; pr[ro1] = rs1; }
            else *(double2 *)(pr + ro0) = make_double2(rs0, rs1);
            vav += O::real(O::conj_mul(xr0, rs0)) + O::real(O::conj_mul(xr1, rs1));
        }
        if (!more || Jn != Jp || hn != h) {
            // end of this warp's run in the strip: transpose-reduction over the 32 lanes, lane l ends with column l
#pragma unroll
            for (int XO = 16, half = 16; XO >= 1; XO >>= 1, half >>= 1) {
                const bool up = (lane & XO) != 0;
#pragma unroll
                for (int c = 0; c < 16; ++c) {
                    if (c < half) {
                        const T send = up ? cs[c] : cs[c + half];
                        const T keep = up ? cs[c + half] : cs[c];
                        cs[c] = O::add(keep, shfl_xor_T(send, XO));
                    }
                }
            }
            Pcol[(long)(bmin + runI) * n + cb0 + lane] = cs[0];
            vav += O::real(O::conj_mul(sx[lane], cs[0]));
            if (more) { strip_begin(Jn, hn); runI = In; }
        }
        Jp = Jn; h = hn; Irel = In;
    }
    return vav;
}

template <class T, bool TMA>
__global__ void __launch_bounds__(TRD_NT, 1) hetrd_panel_kernel(TrdArgs<T> p) {
    typedef Ops<T> O;
    typedef Hv<T> H;
    constexpr int HS = H::HS, SW = H::SW;
    const int G = p.G;
    const int item = blockIdx.x / G, g = blockIdx.x % G;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = p.n, j0 = p.j0, nblk = p.nblk;
    const long lda = p.lda;
    T *A = p.A + (long)item * p.sA;
    double *dd = p.d + (long)item * n, *ee = p.e + (long)item * n;
    T *tauv = p.tau + (long)item * n;
    T *P2 = p.Wp + (long)item * n * 4 * TRD_NB;       // [V | W | W | V], 32 columns each, ld n
    T *Wp = P2 + (long)n * TRD_NB;
    T *acol = p.acol + (long)item * n;
    double *pn = p.pn + (long)item * G;
    T *pt = p.pt + (long)item * G * 2 * TRD_NB;
    double *pvav = p.pvav + (long)item * G;
    T *Prow = p.Prow + (long)item * HS * nblk * n, *Pcol = p.Pcol + (long)item * nblk * n;
    unsigned *bar = p.bar + item;
    unsigned bar_ord = 0;

    const int m = n - j0;
    const int chunk = (m + G - 1) / G;
    const int r0 = j0 + g * chunk, r1 = min(n, r0 + chunk);     // rows owned by this CTA
    const bool cached = chunk <= TRD_CH;

    extern __shared__ __align__(16) unsigned char trd_smem[];
    T *sV = (T *)trd_smem;                       // [NB][CHP]  own rows of V (reflectors of this panel)
    T *sW = sV + TRD_NB * TRD_CHP;               // [NB][CHP]  own rows of W
    T *s_part = sW + TRD_NB * TRD_CHP;           // [NW][PASS]
    T *sx = s_part + TRD_NW * TRD_PASS;          // [NW][SW]
    // TMA variant: per warp a ring of HvT::S stages of 4 KB and their mbarriers
    TrdRing<T> ring;
    if constexpr (TMA) {
        typedef HvT<T> HT;
        T *ring_all = sx + TRD_NW * SW;                                   // 16-byte aligned: every region above is a multiple of 16 bytes
        unsigned long long *bars = (unsigned long long *)(ring_all + (size_t)TRD_NW * HT::S * HT::STAGE);
        if (tid < TRD_NW * HT::S) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(trd_smem_u32(bars + tid)));
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        __syncthreads();
        ring.buf = ring_all + (size_t)warp * HT::S * HT::STAGE;
        ring.full = bars + warp * HT::S;
        ring.pseq = ring.cseq = 0;
        // prologue: the first S stages of this warp's stream (they land while phase A of the first column runs)
        ring.more = trd_cursor_column<HS>(ring.pc, 0, p.nbp, j0, nblk, G, g * TRD_NW + warp);
        for (int s = 0; s < HT::S && ring.more; ++s) {
            trd_issue<T>(ring, A, lda, lane);
            trd_cursor_next<HS, HT::NSUB>(ring.pc, p.nbp, j0, nblk, G, g * TRD_NW + warp);
            ring.more = ring.pc.i < p.nbp;
        }
    }
    __shared__ T s_t[2 * TRD_NB];                // t1 = W^H v at [0,NB), t2 = V^H v at [NB,2NB)
    __shared__ T s_wrow[TRD_NB], s_vrow[TRD_NB];
    __shared__ T s_red4[4][2 * TRD_NB];
    __shared__ T s_tau, s_scale;
    __shared__ double s_alpha, s_vav, s_dred[TRD_NW];

    auto getV = [&](int r, int k) -> T { return cached ? sV[k * TRD_CHP + (r - r0)] : A[r + (long)(j0 + k) * lda]; };
    auto getW = [&](int r, int k) -> T { return cached ? sW[k * TRD_CHP + (r - r0)] : Wp[r + (long)k * n]; };

    for (int i = 0; i <= p.nbp; ++i) {
        const int j = j0 + i;
        const int ra = max(r0, j);                 // first own row still in play
        // =============================== phase A ===============================
        // row j of the panel's V and W (columns < i resp. < i-1): needed by every CTA, fetched first so that the
        // loads overlap the reduction below
        if (tid < i) {
            s_vrow[tid] = ldcg(A + j + (long)(j0 + tid) * lda);
            if (tid < i - 1) s_wrow[tid] = ldcg(Wp + j + (long)tid * n);
        }
        if (i > 0) {
            const int nk = i - 1;
            // (1) reduce the partials of phase B(i-1): t1, t2 (k < i-1) and v^H A v, fixed order
            {
                const int idx = tid & 63, part = tid >> 6;
                const int k = idx < TRD_NB ? idx : idx - TRD_NB;
                T s = O::zero();
                if (k < nk)
                    for (int q0 = part; q0 < G; q0 += 80) {           // 20 loads in flight, summed in a fixed order
                        T bq[20];
#pragma unroll
                        for (int u = 0; u < 20; ++u) bq[u] = (q0 + 4 * u < G) ? ldcg(pt + (long)(q0 + 4 * u) * 2 * TRD_NB + idx) : O::zero();
#pragma unroll
                        for (int u = 0; u < 20; ++u) s = O::add(s, bq[u]);
                    }
                s_red4[part][idx] = s;
                if (warp == 0) {
                    double sv = 0.0, bv[5];
#pragma unroll
                    for (int u = 0; u < 5; ++u) bv[u] = (lane + 32 * u < G) ? ldcg(pvav + lane + 32 * u) : 0.0;
#pragma unroll
                    for (int u = 0; u < 5; ++u) sv += bv[u];
                    for (int qq = lane + 160; qq < G; qq += 32) sv += ldcg(pvav + qq);
                    sv = warp_sum(sv);
                    if (lane == 0) s_vav = sv;
                }
                __syncthreads();
                if (tid < 2 * TRD_NB)
                    s_t[tid] = O::add(O::add(s_red4[0][tid], s_red4[1][tid]), O::add(s_red4[2][tid], s_red4[3][tid]));
                __syncthreads();
                if (warp == 0) {
                    double c = lane < nk ? 2.0 * O::real(O::conj_mul(s_t[lane], s_t[TRD_NB + lane])) : 0.0;
                    c = warp_sum(c);
                    if (lane == 0) s_alpha = -0.5 * O::abs2(s_tau) * (s_vav - c);
                }
                __syncthreads();
            }
            // (2) w_{i-1} for the own rows r >= j and (redundantly, every CTA) for row j
            const int nown = max(0, r1 - ra);
            const bool extra = !(j >= r0 && j < r1);
            const int nloc = nown + (extra ? 1 : 0);
            const int bminp = j / TRD_TB, nbkp = nblk - bminp;           // geometry of the HEMV of column j-1
            const int perp = units_per_warp(HS * (nbkp * (nbkp + 1) / 2), G);
            for (int base = 0; base < nloc; base += TRD_PASS) {
                const int np = min(TRD_PASS, nloc - base);
                {
                    // row sums of the strips: lane <-> 4 rows of the pass, warp <-> strips S = warp, warp + NW, ...;
                    // 4 x 4 independent L2 loads in flight per thread, every row summed in ascending strip order
                    constexpr int NG = TRD_PASS / 32, UB = 8;
                    int rr[NG], se[NG]; T acc[NG];
                    int smax = -1;
#pragma unroll
                    for (int g4 = 0; g4 < NG; ++g4) {
                        const int lp = g4 * 32 + lane, l = base + lp;
                        rr[g4] = l < nown ? ra + l : j;
                        se[g4] = lp < np ? HS * (rr[g4] / TRD_TB) + HS - 1 : -1;
                        smax = max(smax, se[g4]);
                        acc[g4] = O::zero();
                    }
                    for (int S = HS * bminp + warp; S <= smax; S += UB * TRD_NW) {
                        T bq[NG][UB];
#pragma unroll
                        for (int g4 = 0; g4 < NG; ++g4)
#pragma unroll
                            for (int u = 0; u < UB; ++u)
                                bq[g4][u] = (S + u * TRD_NW <= se[g4]) ? ldcg(Prow + (long)(S + u * TRD_NW) * n + rr[g4]) : O::zero();
#pragma unroll
                        for (int g4 = 0; g4 < NG; ++g4)
#pragma unroll
                            for (int u = 0; u < UB; ++u) acc[g4] = O::add(acc[g4], bq[g4][u]);
                    }
#pragma unroll
                    for (int g4 = 0; g4 < NG; ++g4)
                        if (g4 * 32 + lane < np) s_part[warp * TRD_PASS + g4 * 32 + lane] = acc[g4];
                }
                __syncthreads();
                for (int lp = tid; lp < np; lp += TRD_NT) {
                    const int l = base + lp;
                    const bool own = l < nown;
                    const int r = own ? ra + l : j;
                    T y = O::zero();
#pragma unroll
                    for (int w = 0; w < TRD_NW; ++w) y = O::add(y, s_part[w * TRD_PASS + lp]);
                    // column partials: one per run of units in the strip of column r
                    const int Jp = r / TRD_TB - bminp, h = (r % TRD_TB) / SW, len = nbkp - Jp;
                    const int ua = HS * tri_off(Jp, nbkp) + h * len, ub = ua + len;
                    y = O::add(y, ldcg(Pcol + (long)(bminp + Jp) * n + r));
                    for (int kk = ua / perp + 1; kk * perp < ub; ++kk)
                        y = O::add(y, ldcg(Pcol + (long)(bminp + Jp + kk * perp - ua) * n + r));
                    T acc = y;
                    for (int k = 0; k < nk; ++k) {
                        const T v = own ? getV(r, k) : s_vrow[k];          // the extra row is row j
                        const T w = own ? getW(r, k) : s_wrow[k];
                        acc = O::sub(acc, O::add(O::mul(v, s_t[k]), O::mul(w, s_t[TRD_NB + k])));
                    }
                    const T vr = (r == j) ? O::one() : getV(r, i - 1);
                    const T wv = O::add(O::mul(s_tau, acc), O::scale(vr, s_alpha));
                    if (own) {
                        Wp[r + (long)(i - 1) * n] = wv;
                        Wp[r + (long)(TRD_NB + i - 1) * n] = wv;
                        if (cached) sW[(i - 1) * TRD_CHP + (r - r0)] = wv;
                    }
                    if (r == j) s_wrow[i - 1] = wv;
                }
                __syncthreads();
            }
        }
        const bool do_col = (i < p.nbp) || (j == n - 1);
        __syncthreads();
        if (do_col) {
            double nrm = 0.0;
            for (int r = ra + tid; r < r1; r += TRD_NT) {
                T a = A[r + (long)j * lda];
                if (r == j) a = O::from_real(O::real(a));
                for (int k = 0; k < i; ++k)
                    a = O::sub(a, O::add(O::mul_conj(getV(r, k), s_wrow[k]), O::mul_conj(getW(r, k), s_vrow[k])));
                if (r == j) dd[j] = O::real(a);
                else { acol[r] = a; if (r >= j + 2) nrm += O::abs2(a); }
            }
            nrm = block_sum_d(nrm, s_dred);
            if (tid == 0) pn[g] = nrm;
        }
        if (i == p.nbp) break;
        group_barrier(bar, G, ++bar_ord);

        // =============================== phase B ===============================
        if (warp == 0) {
            double s = 0.0, bn[5];
#pragma unroll
            for (int u = 0; u < 5; ++u) bn[u] = (lane + 32 * u < G) ? ldcg(pn + lane + 32 * u) : 0.0;
#pragma unroll
            for (int u = 0; u < 5; ++u) s += bn[u];
            for (int qq = lane + 160; qq < G; qq += 32) s += ldcg(pn + qq);
            s = warp_sum(s);
            if (lane == 0) {
                T alpha0 = ldcg(acol + j + 1);
                double ar = O::real(alpha0), ai = O::imag(alpha0);
                T tau, scale; double beta;
                if (s == 0.0 && ai == 0.0) { tau = O::zero(); scale = O::zero(); beta = ar; }
                else {
                    double nrm = sqrt(ar * ar + ai * ai + s);
                    beta = ar >= 0.0 ? -nrm : nrm;
                    if (O::is_complex) {
                        cplx t = make_double2((beta - ar) / beta, -ai / beta);
                        double dr = ar - beta, di = ai, den = dr * dr + di * di;     // 1/(alpha0 - beta)
                        cplx sc = make_double2(dr / den, -di / den);
                        tau = *(T *)&t; scale = *(T *)&sc;
                    } else {
                        tau = O::from_real((beta - ar) / beta); scale = O::from_real(1.0 / (ar - beta));
                    }
                }
                s_tau = tau; s_scale = scale;
                if (g == 0) { ee[j] = beta; tauv[j] = tau; }
            }
        }
        __syncthreads();
        const T scale = s_scale;
        auto vval = [&](int x) -> T {
            if (x < j + 1 || x >= n) return O::zero();
            if (x == j + 1) return O::one();
            return O::mul(ldcg(acol + x), scale);
        };
        // v into column j of A (own rows) and into the shared-memory panel
        const int rb = max(r0, j + 1);
        for (int r = rb + tid; r < r1; r += TRD_NT) {
            const T v = vval(r);
            A[r + (long)j * lda] = v;
            P2[r + (long)i * n] = v;
            P2[r + (long)(3 * TRD_NB + i) * n] = v;
            if (cached) sV[i * TRD_CHP + (r - r0)] = v;
        }
        __syncthreads();
        // partial t1 = W^H v, t2 = V^H v over the own rows: thread <-> (which, k, quarter of the rows)
        {
            const int idx = tid & 63, part = tid >> 6;
            const int k = idx < TRD_NB ? idx : idx - TRD_NB;
            T s = O::zero();
            if (k < i) {
                if (idx < TRD_NB)
                    for (int r = rb + part; r < r1; r += 4) s = O::add(s, O::conj_mul(getW(r, k), cached ? sV[i * TRD_CHP + (r - r0)] : vval(r)));
                else
                    for (int r = rb + part; r < r1; r += 4) s = O::add(s, O::conj_mul(getV(r, k), cached ? sV[i * TRD_CHP + (r - r0)] : vval(r)));
            }
            s_red4[part][idx] = s;
            __syncthreads();
            if (tid < 2 * TRD_NB)
                pt[(long)g * 2 * TRD_NB + tid] = O::add(O::add(s_red4[0][tid], s_red4[1][tid]), O::add(s_red4[2][tid], s_red4[3][tid]));
        }
        double vav;
        if constexpr (TMA) vav = hemv_warp_tma<T>(ring, A, lda, n, j, i, p.nbp, j0, nblk, G, g, acol, scale, sx + warp * SW, Prow, Pcol);
        else vav = hemv_warp<T>(A, lda, n, j, nblk, G, g, acol, scale, sx + warp * SW, Prow, Pcol);
        vav = block_sum_d(vav, s_dred);
        if (tid == 0) pvav[g] = vav;
        group_barrier(bar, G, ++bar_ord);
    }
}

// workspace layout per call (all items)
struct TrdWork {
    void *Wp, *acol, *pt, *Prow, *Pcol; double *pn, *pvav; unsigned *bar; int G, nblk, items_per_launch; size_t bytes;
};
static int trd_G(int n, int batch, int nsm) {
    int per = nsm / (batch < nsm ? batch : nsm);
    if (per < 1) per = 1;
    int want = ceil_div(n, 64);
    return per < want ? per : want;
}
static int num_sms() { return sm_count(); }
static TrdWork trd_plan(int dtype, int n, int batch, void *work) {
    TrdWork w;
    const size_t es = esize(dtype);
    const int nsm = num_sms();
    w.G = trd_G(n, batch, nsm);
    w.nblk = ceil_div(n, TRD_TB);
    w.items_per_launch = batch < nsm ? batch : nsm;
    const int npanels = ceil_div(n, TRD_NB) + 1;
    Arena ar(work, (size_t)-1);
    w.Wp = ar.take((size_t)batch * n * 4 * TRD_NB * es);
    w.acol = ar.take((size_t)batch * n * es);
    w.pt = ar.take((size_t)batch * w.G * 2 * TRD_NB * es);
    w.Prow = ar.take((size_t)batch * 2 * w.nblk * n * es);          // HS = 2 strips per block column
    w.Pcol = ar.take((size_t)batch * w.nblk * n * es);
    w.pn = (double *)ar.take((size_t)batch * w.G * 8);
    w.pvav = (double *)ar.take((size_t)batch * w.G * 8);
    w.bar = (unsigned *)ar.take((size_t)batch * npanels * 4);
    w.bytes = ar.off;
    return w;
}
size_t hetrd_workspace(int dtype, int n, int batch) { return trd_plan(dtype, n, batch, nullptr).bytes; }

template <class T>
static int hetrd_impl(int dtype, int n, int batch, T *A, long lda, long sA, double *d, double *e, T *tau, void *work,
                      cudaStream_t st) {
    TrdWork w = trd_plan(dtype, n, batch, work);
    const int npanels = ceil_div(n, TRD_NB) + 1;
    const size_t smem_base = (size_t)(2 * TRD_NB * TRD_CHP + TRD_NW * TRD_PASS + TRD_NW * Hv<T>::SW) * sizeof(T);
    const size_t smem_tma = smem_base + (size_t)TRD_NW * HvT<T>::S * (HvT<T>::STAGE * sizeof(T) + 8);
    // the TMA-fed kernel needs whole 64-row units and 16-byte aligned column segments; anything else takes the register-fed one
    // (and pays off from order ~2000 on: for small matrices a warp's run is one or two units and the stage-by-stage latency
    // of the ring shows -- config 1: 22.5 ms against 20.2 ms register-fed; config 2: 289 vs 299 ms; config 3: 776 vs 803 ms)
    const bool tma = n >= 2048 && n % TRD_TB == 0 && ((uintptr_t)A % 16) == 0 && (lda * sizeof(T)) % 16 == 0 && (sA * sizeof(T)) % 16 == 0;
    const size_t smem = tma ? smem_tma : smem_base;
    void *kernel = tma ? (void *)hetrd_panel_kernel<T, true> : (void *)hetrd_panel_kernel<T, false>;
    static bool attr_set = false;
    if (!attr_set) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(hetrd_panel_kernel<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_base));
        NAO_CUDA_CHECK(cudaFuncSetAttribute(hetrd_panel_kernel<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_tma));
        attr_set = true;
    }
    NAO_CUDA_CHECK(cudaMemsetAsync(w.bar, 0, (size_t)batch * npanels * 4, st));
    int panel = 0;
    for (int j0 = 0; j0 == 0 || j0 < n - 1; j0 += TRD_NB, ++panel) {
        const int nbp = max(0, min(TRD_NB, n - 1 - j0));
        for (int b0 = 0; b0 < batch; b0 += w.items_per_launch) {
            const int nb_items = min(w.items_per_launch, batch - b0);
            TrdArgs<T> a;
            a.A = A + (long)b0 * sA; a.lda = lda; a.sA = sA;
            a.d = d + (long)b0 * n; a.e = e + (long)b0 * n; a.tau = tau + (long)b0 * n;
            a.Wp = (T *)w.Wp + (long)b0 * n * 4 * TRD_NB; a.acol = (T *)w.acol + (long)b0 * n;
            a.pn = w.pn + (long)b0 * w.G; a.pt = (T *)w.pt + (long)b0 * w.G * 2 * TRD_NB; a.pvav = w.pvav + (long)b0 * w.G;
            a.Prow = (T *)w.Prow + (long)b0 * Hv<T>::HS * w.nblk * n; a.Pcol = (T *)w.Pcol + (long)b0 * w.nblk * n;
            a.bar = w.bar + (size_t)panel * batch + b0;
            a.n = n; a.j0 = j0; a.nbp = nbp; a.G = w.G; a.nblk = w.nblk;
            // algorithmic bytes of this launch: the lower triangle of the trailing matrix once per column
            double bytes = 0.0;
            for (int i = 0; i < nbp; ++i) { double mm = n - (j0 + i) - 1; bytes += 0.5 * mm * (mm + 1) * sizeof(T); }
            const int pk = prof_kernel_begin(0, bytes * nb_items, st);
            void *args[] = {&a};
            NAO_CUDA_CHECK(cudaLaunchCooperativeKernel(kernel, dim3(nb_items * w.G), dim3(TRD_NT), args, smem, st));
            NAO_LAUNCHED();
            prof_kernel_end(0, pk, st);
        }
        const int jn = j0 + nbp;             // first row/column of the trailing matrix
        if (nbp > 0 && jn < n) {
            const int mt = n - jn;
            const long sP = (long)n * 4 * TRD_NB;
            T *P2 = (T *)w.Wp;
            if (nbp == TRD_NB) {
                // A22 -= [V W] [W V]^H : one rank-64 update, the trailing matrix is read and written once
                GemmDesc g1 = gemm_desc(OP_N, OP_C, mt, mt, 2 * TRD_NB, -1.0, P2 + jn, n, P2 + jn + (long)n * 2 * TRD_NB, n, 1.0,
                                        A + jn + (long)jn * lda, lda);
                g1.sA = sP; g1.sB = sP; g1.sC = sA; g1.cmode = 1;
                if (int rc = gemm_launch(dtype, g1, batch, st)) return rc;
            } else {
                GemmDesc g1 = gemm_desc(OP_N, OP_C, mt, mt, nbp, -1.0, P2 + jn, n, P2 + jn + (long)n * TRD_NB, n, 1.0,
                                        A + jn + (long)jn * lda, lda);
                g1.sA = sP; g1.sB = sP; g1.sC = sA; g1.cmode = 1;
                if (int rc = gemm_launch(dtype, g1, batch, st)) return rc;
                GemmDesc g2 = gemm_desc(OP_N, OP_C, mt, mt, nbp, -1.0, P2 + jn + (long)n * TRD_NB, n, P2 + jn, n, 1.0,
                                        A + jn + (long)jn * lda, lda);
                g2.sA = sP; g2.sB = sP; g2.sC = sA; g2.cmode = 1;
                if (int rc = gemm_launch(dtype, g2, batch, st)) return rc;
            }
        }
        if (n == 1) break;
    }
    return NAO_OK;
}


int hetrd(int dtype, int n, int batch, void *A, long lda, long sA, double *d, double *e, void *tau, void *work,
          cudaStream_t st) {
    return dtype == NAO_COMPLEX ? hetrd_impl<cplx>(dtype, n, batch, (cplx *)A, lda, sA, d, e, (cplx *)tau, work, st)
                                : hetrd_impl<double>(dtype, n, batch, (double *)A, lda, sA, d, e, (double *)tau, work, st);
}
}  // namespace nao
