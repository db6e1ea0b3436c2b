// trd2_chase.cu -- stage 2 of the two-stage tridiagonalisation: band -> real tridiagonal by bulge chasing, staged in
// shared memory (north_star "band-to-tridiagonal uses bulge chasing staged in shared memory").
//
// Band B (lower, bandwidth b = TRD2_B) is kept in HBM/L2 as AB[(i - j) + j * 2b], 0 <= i - j < 2b (the second b rows
// hold the bulge).  Sweep s annihilates column s below the sub-diagonal:
//   step 0   : v = house(B[s+1 : s+b, s]);  D_0 <- H^H D_0 H                         (D_0 = diagonal block of those rows)
//   step k>=1: O = B[R_k, R_{k-1}] <- O H_{k-1};  v_k = house(O[:, 0]);  O[:, 1:] <- H_k^H O[:, 1:];  D_k <- H_k^H D_k H_k
// with R_k = rows s+1+kb .. s+(k+1)b.  One CTA runs a whole sweep, carrying the reflector in shared memory; sweeps are
// pipelined over the co-resident CTAs of a persistent cooperative kernel: sweep s+1 may run step k once sweep s has
// finished step k+1 (progress counters in global memory, release/acquire).  CTA c of an item runs sweeps c, c+P, ...
// in order, so the lowest unfinished sweep can always advance (no deadlock).
//
// Reflector (s, k) is stored for the back-transformation at V2[R_k, s] (unit stored explicitly), tau2[k * n + s].
// Complex case: beta of every reflector is real, so the final sub-diagonal is real; the last sweep (length 1) only
// removes the phase of B[n-1, n-2].
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>
#include <climits>

namespace nao {

static const int CH_NT = 256;


template <class T>
__global__ void band_extract_kernel(int n, const T *A, long lda, long sA, T *AB, long sAB) {
    constexpr int b = TRD2_B, ld = 2 * b;
    A += (long)blockIdx.y * sA; AB += (long)blockIdx.y * sAB;
    const int j = blockIdx.x;
    for (int r = threadIdx.x; r < ld; r += blockDim.x) {
        const int i = j + r;
        T v = Ops<T>::zero();
        if (r <= b && i < n) { v = A[i + (long)j * lda]; if (r == 0) v = Ops<T>::from_real(Ops<T>::real(v)); }
        AB[r + (long)j * ld] = v;
    }
}

template <class T> struct ChaseArgs {
    T *AB; long sAB;             // band, 2b x n per item
    T *V2; long ldv, sV2;        // n x n per item
    T *tau2; long sTau2;         // nk x n per item (tau2[k * n + s])
    double *d, *e;               // n each per item
    int *prog;                   // n per item, zero-initialised
    int n, P;
};

__device__ __forceinline__ int ld_acquire(const int *p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int *p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// xLARFG on x[0..L) held in shared memory (x[0] = alpha); executed by warp 0.  Leaves v in x (x[0] = 1), returns
// (tau, beta) through shared scalars.
template <class T>
__device__ __forceinline__ void house_warp(T *x, int L, T *s_tau, double *s_beta) {
    typedef Ops<T> O;
    const int lane = threadIdx.x & 31;
    double xn2 = 0.0;
    for (int i = 1 + lane; i < L; i += 32) xn2 += O::abs2(x[i]);
    xn2 = warp_sum(xn2);
    const T alpha = x[0];
    const double ar = O::real(alpha), ai = O::imag(alpha);
    T tau, scale; double beta;
    if (xn2 == 0.0 && ai == 0.0) { tau = O::zero(); scale = O::zero(); beta = ar; }
    else {
        const double nrm = sqrt(ar * ar + ai * ai + xn2);
        beta = ar >= 0.0 ? -nrm : nrm;
        if (O::is_complex) {
            cplx t = make_double2((beta - ar) / beta, -ai / beta);
            const double dr = ar - beta, di = ai, den = dr * dr + di * di;
            cplx sc = make_double2(dr / den, -di / den);
            tau = *(T *)&t; scale = *(T *)&sc;
        } else {
            tau = O::from_real((beta - ar) / beta); scale = O::from_real(1.0 / (ar - beta));
        }
    }
    __syncwarp();
    for (int i = 1 + lane; i < L; i += 32) x[i] = O::mul(scale, x[i]);
    if (lane == 0) { x[0] = O::one(); *s_tau = tau; *s_beta = beta; }
}

// PF (real only: two pairs of blocks fit in shared memory): the blocks of step k+1 are requested (cp.async, second buffer)
// while step k is computed.  Only the LAST row of O and of D is written by the predecessor sweep's step k+2; everything
// else of those blocks is final once the predecessor has finished step k+1 -- which the CTA has already waited for at the
// start of step k.  The last row is read after the wait of step k+1, with one short round trip.
template <class T, bool PF>
__global__ void __launch_bounds__(CH_NT, 1) chase_kernel(ChaseArgs<T> p) {
    typedef Ops<T> O;
    constexpr int b = TRD2_B, ld = 2 * b, LDS = b + 1;
    const int P = p.P, item = blockIdx.x / P, c = blockIdx.x % P;
    const int n = p.n, tid = threadIdx.x, warp = tid >> 5;
    T *AB = p.AB + (long)item * p.sAB;
    T *V2 = p.V2 + (long)item * p.sV2;
    T *tau2 = p.tau2 + (long)item * p.sTau2;
    double *dd = p.d + (long)item * n, *ee = p.e + (long)item * n;
    int *prog = p.prog + (long)item * n;

    extern __shared__ __align__(16) unsigned char ch_smem[];
    T *sO = (T *)ch_smem;              // [b][LDS]  off-diagonal block, column-major
    T *sD = sO + b * LDS;              // [b][LDS]  diagonal block (full Hermitian)
    T *sO2 = sD + b * LDS, *sD2 = sO2 + b * LDS;      // PF: the pair of the next step
    __shared__ T s_vp[b], s_vn[b], s_w[b], s_u[b], s_z[b], s_part[4][b], s_part2[4][b];
    __shared__ T s_tau_p, s_tau_n, s_kappa;
    __shared__ double s_beta, s_gamma;

    const int iq = tid & (b - 1), qq = tid >> 6;        // (row or column index, quarter)

    // D <- H^H D H for the L x L block in sD with v = s_vn, tau = s_tau_n  (u = D v, gamma = v^H u,
    // w = tau u - 1/2 |tau|^2 gamma v,  D -= w v^H + v w^H)
    auto two_sided = [&](int L) {
        {   // (block and vector are zero beyond L: full-range loops with compile-time trip counts, two accumulators)
            T s0 = O::zero(), s1 = O::zero();
#pragma unroll
            for (int t = 0; t < b / 8; ++t) {
                const int c0_ = qq + 8 * t, c1_ = c0_ + 4;
                s0 = O::fma(sD[c0_ * LDS + iq], s_vn[c0_], s0);
                s1 = O::fma(sD[c1_ * LDS + iq], s_vn[c1_], s1);
            }
            s_part[qq][iq] = O::add(s0, s1);
        }
        __syncthreads();
        if (warp == 0) {
            // u = D v (two elements per lane) and gamma = v^H u in one go
            const int i0_ = tid, i1_ = tid + 32;
            const T u0 = i0_ < L ? O::add(O::add(s_part[0][i0_], s_part[1][i0_]), O::add(s_part[2][i0_], s_part[3][i0_])) : O::zero();
            const T u1 = i1_ < L ? O::add(O::add(s_part[0][i1_], s_part[1][i1_]), O::add(s_part[2][i1_], s_part[3][i1_])) : O::zero();
            s_w[i0_] = u0; s_w[i1_] = u1;
            double gsum = O::real(O::conj_mul(s_vn[i0_], u0)) + O::real(O::conj_mul(s_vn[i1_], u1));
            gsum = warp_sum(gsum);
            if (tid == 0) s_gamma = gsum;
        }
        __syncthreads();
        {
            const T tau = s_tau_n;
            const double f = -0.5 * O::abs2(tau) * s_gamma;
            T wv = O::zero();
            if (tid < L) wv = O::add(O::mul(tau, s_w[tid]), O::scale(s_vn[tid], f));
            if (tid < b) s_w[tid] = wv;              // every thread rewrites only the element it has just read
        }
        __syncthreads();
        if (iq < L) {
            const T wi = s_w[iq], vi = s_vn[iq];
#pragma unroll
            for (int t = 0; t < b / 4; ++t) {
                const int cc = qq + 4 * t;
                if (cc < L) {
                    T a = sD[cc * LDS + iq];
                    a = O::sub(a, O::add(O::mul_conj(wi, s_vn[cc]), O::mul_conj(vi, s_w[cc])));
                    if (cc == iq) a = O::from_real(O::real(a));
                    sD[cc * LDS + iq] = a;
                }
            }
        }
        __syncthreads();
    };
    // diagonal block rows/cols [g0, g0+L): load (Hermitian completion) / store (lower part)
    // (all loads of a block are issued before the first shared-memory store: one L2 round trip per block)
    auto load_D = [&](int g0, int L) {
        T buf[b * b / CH_NT];
#pragma unroll
        for (int it = 0; it < b * b / CH_NT; ++it) {
            const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
            T v = O::zero();
            if (i < L && cc < L) v = (i >= cc) ? ldcg(AB + (i - cc) + (long)(g0 + cc) * ld) : ldcg(AB + (cc - i) + (long)(g0 + i) * ld);
            buf[it] = v;
        }
#pragma unroll
        for (int it = 0; it < b * b / CH_NT; ++it) {
            const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
            sD[cc * LDS + i] = (i >= cc) ? buf[it] : O::conj(buf[it]);
        }
    };
    auto load_O = [&](int q0, int Lq, int r0, int Lp) {
        T buf[b * b / CH_NT];
#pragma unroll
        for (int it = 0; it < b * b / CH_NT; ++it) {
            const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
            T v = O::zero();
            if (i < Lq && cc < Lp) v = ldcg(AB + (q0 + i - r0 - cc) + (long)(r0 + cc) * ld);
            buf[it] = v;
        }
#pragma unroll
        for (int it = 0; it < b * b / CH_NT; ++it) {
            const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
            sO[cc * LDS + i] = buf[it];
        }
    };
    auto store_D = [&](int g0, int L) {
        for (int e = tid; e < b * b; e += CH_NT) {
            const int i = e & (b - 1), cc = e >> 6;
            if (i < L && cc < L && i >= cc) AB[(i - cc) + (long)(g0 + cc) * ld] = sD[cc * LDS + i];
        }
    };

    // PF: request rows 0..b-2 of the blocks of step k1 of sweep s into (sO2, sD2); D lower part only; zero elsewhere
    auto prefetch = [&](int s, int k1) {
        const int q1 = s + 1 + k1 * b;
        if (q1 > n - 1) return;
        const int Lq1 = min(s + (k1 + 1) * b, n - 1) - q1 + 1, r1 = q1 - b;      // the column block of O has b columns
#pragma unroll
        for (int it = 0; it < b * b / CH_NT; ++it) {
            const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
            const bool po = i < Lq1 && i < b - 1, pd = po && i >= cc;
            cp_async8(sO2 + cc * LDS + i, po ? AB + (q1 + i - r1 - cc) + (long)(r1 + cc) * ld : AB, po);
            cp_async8(sD2 + cc * LDS + i, pd ? AB + (i - cc) + (long)(q1 + cc) * ld : AB, pd);
        }
        cp_async_commit();
    };
    for (int s = c; s < n - 1; s += P) {
        // ------------------------------------------------ step 0
        int r0 = s + 1, Lp = min(s + b, n - 1) - r0 + 1;
        // Column s and the diagonal block are final after the predecessor's step 0 except for their last row (global row
        // s + b), which its step 1 writes: everything else is read as soon as the counter shows 1, the last row after 2.
        const bool late0 = (Lp == b);
        if (s > 0) {
            if (tid == 0) { while (ld_acquire(prog + s - 1) < 1) { } }
            __syncthreads();
        }
        if (tid < b) s_vn[tid] = (tid < Lp && !(late0 && tid == b - 1)) ? ldcg(AB + (1 + tid) + (long)s * ld) : O::zero();
        load_D(r0, late0 ? b - 1 : Lp);
        if (late0) {
            if (s > 0 && tid == 0) { while (ld_acquire(prog + s - 1) < 2) { } }
            __syncthreads();             // (also orders the zero fill of row b-1 above before the late values below)
        }
        if (late0) {
            if (tid < b) {
                const T v = ldcg(AB + (b - 1 - tid) + (long)(r0 + tid) * ld);          // D(b-1, tid)
                sD[tid * LDS + b - 1] = v; sD[(b - 1) * LDS + tid] = O::conj(v);
            } else if (tid == b) s_vn[b - 1] = ldcg(AB + b + (long)s * ld);
        }
        if constexpr (PF) prefetch(s, 1);
        __syncthreads();
        if (warp == 0) house_warp<T>(s_vn, Lp, &s_tau_n, &s_beta);
        __syncthreads();
        if (tid < Lp) {
            V2[(r0 + tid) + (long)s * p.ldv] = s_vn[tid];
            AB[(1 + tid) + (long)s * ld] = tid == 0 ? O::from_real(s_beta) : O::zero();
        }
        if (tid == 0) { tau2[s] = s_tau_n; ee[s] = s_beta; dd[s] = O::real(ldcg(AB + (long)s * ld)); }
        two_sided(Lp);
        store_D(r0, Lp);
        if (tid < b) s_vp[tid] = s_vn[tid];
        if (tid == 0) s_tau_p = s_tau_n;
        __syncthreads();
        if (tid == 0) { __threadfence(); st_release(prog + s, 1); }
        // ------------------------------------------------ steps k >= 1
        for (int k = 1;; ++k) {
            const int q0 = s + 1 + k * b;
            if (q0 > n - 1) break;
            const int Lq = min(s + (k + 1) * b, n - 1) - q0 + 1;
            if (PF && s > 0) {
                if (tid == 0) { while (ld_acquire(prog + s - 1) < k + 2) { } }
                __syncthreads();
            }
            if constexpr (PF) {
                // the prefetched pair becomes current; its last row arrives now (written by the predecessor's latest step)
                cp_async_wait<0>();
                { T *t = sO; sO = sO2; sO2 = t; t = sD; sD = sD2; sD2 = t; }
                T late = O::zero();
                const bool has_late = Lq == b && tid < 2 * b;
                if (has_late) {
                    const int cc = tid & (b - 1);
                    late = tid < b ? ldcg(AB + (q0 + b - 1 - r0 - cc) + (long)(r0 + cc) * ld)
                                   : ldcg(AB + (b - 1 - cc) + (long)(q0 + cc) * ld);
                }
                __syncthreads();                 // everybody's prefetched elements have landed; the old pair is free
                prefetch(s, k + 1);
                // Hermitian completion of D from its lower part (rows <= b-2 now, row/column b-1 below)
#pragma unroll
                for (int it = 0; it < b * b / CH_NT; ++it) {
                    const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
                    if (i < cc && cc < b - 1) sD[cc * LDS + i] = O::conj(sD[i * LDS + cc]);
                }
                if (has_late) {
                    const int cc = tid & (b - 1);
                    if (tid < b) sO[cc * LDS + b - 1] = late;
                    else { sD[cc * LDS + b - 1] = late; sD[(b - 1) * LDS + cc] = O::conj(late); }
                }           // (short last block: row b-1 does not exist; column b-1 of D was zero-filled by the prefetch)
            } else
            {   // No second buffer (complex).  Everything except the last row of the two blocks is final since the predecessor
                // finished step k+1 -- known since the wait of the previous step -- so those loads are issued BEFORE waiting for
                // its step k+2; the last row follows with one short round trip.  All loads of a thread are in flight at once.
                T bo[b * b / CH_NT], bd[b * b / CH_NT];
                const bool lateK = (Lq == b);
#pragma unroll
                for (int it = 0; it < b * b / CH_NT; ++it) {
                    const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
                    T vo = O::zero(), vd = O::zero();
                    if (i < Lq && cc < Lp && !(lateK && i == b - 1)) vo = ldcg(AB + (q0 + i - r0 - cc) + (long)(r0 + cc) * ld);
                    if (i < Lq && cc < Lq && !(lateK && (i == b - 1 || cc == b - 1)))
                        vd = (i >= cc) ? ldcg(AB + (i - cc) + (long)(q0 + cc) * ld) : ldcg(AB + (cc - i) + (long)(q0 + i) * ld);
                    bo[it] = vo; bd[it] = vd;
                }
                if (s > 0) {
                    if (tid == 0) { while (ld_acquire(prog + s - 1) < k + 2) { } }
                    __syncthreads();
                }
                T late = O::zero();
                const bool has_late = lateK && tid < 2 * b;
                if (has_late) {
                    const int cc = tid & (b - 1);
                    late = tid < b ? ldcg(AB + (q0 + b - 1 - r0 - cc) + (long)(r0 + cc) * ld)
                                   : ldcg(AB + (b - 1 - cc) + (long)(q0 + cc) * ld);
                }
#pragma unroll
                for (int it = 0; it < b * b / CH_NT; ++it) {
                    const int e = tid + it * CH_NT, i = e & (b - 1), cc = e >> 6;
                    if (!(lateK && i == b - 1)) sO[cc * LDS + i] = bo[it];
                    if (!(lateK && (i == b - 1 || cc == b - 1))) sD[cc * LDS + i] = (i >= cc) ? bd[it] : O::conj(bd[it]);
                }
                if (has_late) {
                    const int cc = tid & (b - 1);
                    if (tid < b) sO[cc * LDS + b - 1] = late;
                    else { sD[cc * LDS + b - 1] = late; sD[(b - 1) * LDS + cc] = O::conj(late); }
                }
            }
            __syncthreads();
            // Fused form of  O <- H_n^H (O H_p),  D <- H_n^H D H_n  with ONE pass over each block:
            //   w = O v_p ;  x = O[:,0] - tau_p w  -> (v_n, tau_n, beta) ;  kappa = v_n^H w
            //   q = O^H v_n (on the ORIGINAL O) ;  z_c = q_c - tau_p kappa conj(v_p[c])   (= v_n^H (O H_p)[:,c])
            //   O[:,c] <- O[:,c] - tau_p w conj(v_p[c]) - conj(tau_n) v_n z_c  (c >= 1);  O[:,0] <- beta e_0
            //   u = D v_n ; gamma = v_n^H u ; y = tau_n u - 1/2 |tau_n|^2 gamma v_n ;  D <- D - y v_n^H - v_n y^H
            // (1) w partials: thread <-> (row iq, column quarter qq)
            // (the blocks and the vectors are zero beyond Lq / Lp: all loops run over the full block with compile-time trip
            //  counts, two accumulators each)
            {
                T s0 = O::zero(), s1 = O::zero();
#pragma unroll
                for (int t = 0; t < b / 8; ++t) {
                    const int c0_ = qq + 8 * t, c1_ = c0_ + 4;
                    s0 = O::fma(sO[c0_ * LDS + iq], s_vp[c0_], s0);
                    s1 = O::fma(sO[c1_ * LDS + iq], s_vp[c1_], s1);
                }
                s_part[qq][iq] = O::add(s0, s1);
            }
            __syncthreads();
            // (2)+(3) w, x, the reflector (xLARFG) and kappa by warp 0 alone, two elements per lane, reductions in registers
            if (warp == 0) {
                const int i0_ = tid, i1_ = tid + 32;
                const T w0_ = i0_ < Lq ? O::add(O::add(s_part[0][i0_], s_part[1][i0_]), O::add(s_part[2][i0_], s_part[3][i0_])) : O::zero();
                const T w1_ = i1_ < Lq ? O::add(O::add(s_part[0][i1_], s_part[1][i1_]), O::add(s_part[2][i1_], s_part[3][i1_])) : O::zero();
                const T taup = s_tau_p;
                T x0_ = i0_ < Lq ? O::sub(sO[i0_], O::mul(taup, w0_)) : O::zero();      // v_p[0] = 1
                T x1_ = i1_ < Lq ? O::sub(sO[i1_], O::mul(taup, w1_)) : O::zero();
                s_w[i0_] = w0_; s_w[i1_] = w1_;
                double xn2 = (tid == 0 ? 0.0 : O::abs2(x0_)) + O::abs2(x1_);
                xn2 = warp_sum(xn2);
                const double ar = __shfl_sync(0xffffffffu, O::real(x0_), 0), ai = __shfl_sync(0xffffffffu, O::imag(x0_), 0);
                T tau, scale; double beta;
                if (xn2 == 0.0 && ai == 0.0) { tau = O::zero(); scale = O::zero(); beta = ar; }
                else {
                    const double nrm = sqrt(ar * ar + ai * ai + xn2);
                    beta = ar >= 0.0 ? -nrm : nrm;
                    if (O::is_complex) {
                        cplx t = make_double2((beta - ar) / beta, -ai / beta);
                        const double dr = ar - beta, di = ai, den = dr * dr + di * di;
                        cplx sc = make_double2(dr / den, -di / den);
                        tau = *(T *)&t; scale = *(T *)&sc;
                    } else {
                        tau = O::from_real((beta - ar) / beta); scale = O::from_real(1.0 / (ar - beta));
                    }
                }
                x0_ = tid == 0 ? O::one() : O::mul(scale, x0_);
                x1_ = O::mul(scale, x1_);
                s_vn[i0_] = x0_; s_vn[i1_] = x1_;
                T kp = O::add(O::conj_mul(x0_, w0_), O::conj_mul(x1_, w1_));
                kp = warp_sum(kp);
                if (tid == 0) { s_tau_n = tau; s_beta = beta; s_kappa = kp; }
            }
            __syncthreads();
            if (tid < Lq) V2[(q0 + tid) + (long)s * p.ldv] = s_vn[tid];
            if (tid == 0) tau2[(long)k * n + s] = s_tau_n;
            // (4) q partials: thread <-> (column iq, row quarter qq);  u partials: thread <-> (row iq, column quarter qq)
            {
                T qa0 = O::zero(), qa1 = O::zero(), ua0 = O::zero(), ua1 = O::zero();
#pragma unroll
                for (int t = 0; t < b / 8; ++t) {
                    const int i0_ = qq + 8 * t, i1_ = i0_ + 4;
                    qa0 = O::add(qa0, O::conj_mul(s_vn[i0_], sO[iq * LDS + i0_]));
                    qa1 = O::add(qa1, O::conj_mul(s_vn[i1_], sO[iq * LDS + i1_]));
                    ua0 = O::fma(sD[i0_ * LDS + iq], s_vn[i0_], ua0);
                    ua1 = O::fma(sD[i1_ * LDS + iq], s_vn[i1_], ua1);
                }
                s_part[qq][iq] = O::add(qa0, qa1); s_part2[qq][iq] = O::add(ua0, ua1);
            }
            __syncthreads();
            // (5) z (scaled by conj(tau_n)), u, gamma
            if (tid < b) {
                const T q = O::add(O::add(s_part[0][tid], s_part[1][tid]), O::add(s_part[2][tid], s_part[3][tid]));
                const T z = tid < Lp ? O::sub(q, O::mul(O::mul(s_tau_p, s_kappa), O::conj(s_vp[tid]))) : O::zero();
                s_z[tid] = O::mul(O::conj(s_tau_n), z);
                s_u[tid] = tid < Lq ? O::add(O::add(s_part2[0][tid], s_part2[1][tid]), O::add(s_part2[2][tid], s_part2[3][tid])) : O::zero();
            }
            else if (warp == 2) {
                // gamma = v_n^H u straight from the partial sums, beside the threads that form z and u
                double gsum = 0.0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int i = (tid & 31) + 32 * h;
                    const T u = O::add(O::add(s_part2[0][i], s_part2[1][i]), O::add(s_part2[2][i], s_part2[3][i]));
                    if (i < Lq) gsum += O::real(O::conj_mul(s_vn[i], u));
                }
                gsum = warp_sum(gsum);
                if ((tid & 31) == 0) s_gamma = gsum;
            }
            __syncthreads();
            // (6) one pass over O and D: new values go straight to global memory
            {
                const T tau_n = s_tau_n, tau_p = s_tau_p;
                const double f = -0.5 * O::abs2(tau_n) * s_gamma;
                auto yv = [&](int i) -> T { return O::add(O::mul(tau_n, s_u[i]), O::scale(s_vn[i], f)); };
                if (iq < Lq) {
                    const T twi = O::mul(tau_p, s_w[iq]), vni = s_vn[iq], yi = yv(iq);
                    T *po = AB + (q0 + iq - r0 - qq) + (long)(r0 + qq) * ld;     // element (iq, cc) of O; cc -> cc + 4: += 4 (ld - 1)
                    T *pd = AB + (iq - qq) + (long)(q0 + qq) * ld;               // element (iq, cc) of D
#pragma unroll
                    for (int t = 0; t < b / 4; ++t) {
                        const int cc = qq + 4 * t;
                        if (cc < Lp) {
                            T o;
                            if (cc == 0) o = iq == 0 ? O::from_real(s_beta) : O::zero();
                            else o = O::sub(O::sub(sO[cc * LDS + iq], O::mul_conj(twi, s_vp[cc])), O::mul(vni, s_z[cc]));
                            po[(long)t * 4 * (ld - 1)] = o;
                        }
                    }
#pragma unroll
                    for (int t = 0; t < b / 4; ++t) {
                        const int cc = qq + 4 * t;
                        if (cc <= iq) {                                          // lower part is what is stored (iq < Lq)
                            T a = O::sub(sD[cc * LDS + iq], O::add(O::mul_conj(yi, s_vn[cc]), O::mul_conj(vni, yv(cc))));
                            if (cc == iq) a = O::from_real(O::real(a));
                            pd[(long)t * 4 * (ld - 1)] = a;
                        }
                    }
                }
            }
            // publish: the block barrier orders every thread's stores before thread 0, whose fence + release store make
            // them visible to the CTA that acquires the counter (the pattern of a cooperative-groups grid sync)
            __syncthreads();
            if (tid < b) s_vp[tid] = s_vn[tid];
            if (tid == 0) { s_tau_p = s_tau_n; __threadfence(); st_release(prog + s, k + 1); }
            r0 = q0; Lp = Lq;
        }
        __syncthreads();
        if (tid == 0) st_release(prog + s, INT_MAX);
    }
    // the last diagonal entry
    if (c == (n - 1) % P || n == 1) {
        if (n >= 2) { if (tid == 0) { while (ld_acquire(prog + n - 2) < INT_MAX) { } } }
        __syncthreads();
        if (tid == 0) { dd[n - 1] = O::real(ldcg(AB + (long)(n - 1) * ld)); ee[n - 1] = 0.0; }
    }
}

struct ChaseWork { void *AB; int *prog; int P, ipl; size_t bytes; };
static int ch_num_sms() { return sm_count(); }
static ChaseWork chase_plan(int dtype, int n, int batch, void *work) {
    ChaseWork w; const size_t es = esize(dtype);
    const int nsm = ch_num_sms();
    const int want = ceil_div(n, 2 * TRD2_B) + 1;              // sweeps that can be in flight
    w.ipl = std::max(1, std::min(batch, nsm / std::min(want, nsm)));
    w.P = std::max(1, std::min(want, nsm / w.ipl));
    Arena ar(work, (size_t)-1);
    w.AB = ar.take((size_t)batch * 2 * TRD2_B * n * es);
    w.prog = (int *)ar.take((size_t)batch * n * 4);
    w.bytes = ar.off;
    return w;
}
size_t hb2st_workspace(int dtype, int n, int batch) { return chase_plan(dtype, n, batch, nullptr).bytes; }
int hb2st_nk(int n) { return ceil_div(n, TRD2_B) + 1; }

template <class T>
static int hb2st_impl(int dtype, int n, int batch, const T *A, long lda, long sA, double *d, double *e, T *V2, long ldv,
                      long sV2, T *tau2, void *work, cudaStream_t st) {
    constexpr int b = TRD2_B;
    ChaseWork w = chase_plan(dtype, n, batch, work);
    constexpr bool PF = sizeof(T) == 8;          // double-buffered blocks: real only (complex blocks are twice the size)
    const size_t smem = (size_t)(PF ? 4 : 2) * b * (b + 1) * sizeof(T);
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(chase_kernel<T, PF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    const long sAB = (long)2 * b * n, sTau2 = (long)hb2st_nk(n) * n;
    band_extract_kernel<T><<<dim3(n, batch), 128, 0, st>>>(n, A, lda, sA, (T *)w.AB, sAB);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaMemsetAsync(w.prog, 0, (size_t)batch * n * 4, st));
    NAO_CUDA_CHECK(cudaMemsetAsync(V2, 0, (size_t)batch * sV2 * sizeof(T), st));
    NAO_CUDA_CHECK(cudaMemsetAsync(tau2, 0, (size_t)batch * sTau2 * sizeof(T), st));
    for (int b0 = 0; b0 < batch; b0 += w.ipl) {
        const int nit = std::min(w.ipl, batch - b0);
        ChaseArgs<T> a;
        a.AB = (T *)w.AB + (long)b0 * sAB; a.sAB = sAB;
        a.V2 = V2 + (long)b0 * sV2; a.ldv = ldv; a.sV2 = sV2;
        a.tau2 = tau2 + (long)b0 * sTau2; a.sTau2 = sTau2;
        a.d = d + (long)b0 * n; a.e = e + (long)b0 * n; a.prog = w.prog + (long)b0 * n;
        a.n = n; a.P = w.P;
        void *args[] = {&a};
        NAO_CUDA_CHECK(cudaLaunchCooperativeKernel((void *)chase_kernel<T, PF>, dim3(nit * w.P), dim3(CH_NT), args, smem, st));
        NAO_LAUNCHED();
    }
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}


int hb2st(int dtype, int n, int batch, const void *A, long lda, long sA, double *d, double *e, void *V2, long ldv, long sV2,
          void *tau2, void *work, cudaStream_t st) {
    return dtype == NAO_COMPLEX
               ? hb2st_impl<cplx>(dtype, n, batch, (const cplx *)A, lda, sA, d, e, (cplx *)V2, ldv, sV2, (cplx *)tau2, work, st)
               : hb2st_impl<double>(dtype, n, batch, (const double *)A, lda, sA, d, e, (double *)V2, ldv, sV2, (double *)tau2, work, st);
}

}  // namespace nao
