// trd2_back.cu -- back-transformation of the bulge-chasing stage: Z <- Q2 Z ("stage 2 then
// stage 1, blocked Householder GEMMs").
//
// Q2 = prod_s prod_k H_{s,k} (sweeps s ascending, steps k ascending; reflector (s,k) acts on rows s+1+kb .. s+(k+1)b).
// Reflectors are grouped in "diamonds": S-block I = sweeps s0 .. s0+NBK-1 (s0 = I*NBK) and step k give the group
//   G(I,k) = H_{s0,k} H_{s0+1,k} ... = I - V T V^H,   V = (b + NBK - 1) x NBK parallelogram (rows s0+1+kb ..).
// Reflectors of different steps of one sweep commute, and (s,k) overlaps (s',k+1) only for s' < s, so Q2 Z is obtained
// by applying the groups with I DESCENDING and, inside an S-block, k ASCENDING (checked against the sweep-by-sweep
// product in tests).  Columns of Z are independent: each CTA owns NC columns and walks through all groups without any
// inter-CTA synchronisation; the three products per group (W = V^H Z_w, W <- T W, Z_w -= V W) run on FP64 DMMA from
// shared memory.  T factors of all groups are precomputed by q2_tfactor_kernel.
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>

namespace nao {

static const int Q2_NBK = 32;                 // sweeps per diamond
static const int Q2_LW = 96;                  // padded window rows (>= TRD2_B + Q2_NBK - 1)
static const int Q2_NT = 128;
static const int Q2_LDV = 100, Q2_LDW = 36;   // shared-memory leading dimensions (conflict-free fragment loads)
// T: 36 for real (conflict-free A fragments); complex stays at 32 so that two CTAs of 16 columns still fit on an SM
template <class T> struct Q2Ldt { static const int value = sizeof(T) == 8 ? 36 : 32; };

__host__ __device__ inline int q2_nwin(int n, int s0) {      // windows of the S-block starting at sweep s0
    return s0 + 1 <= n - 1 ? (n - 2 - s0) / TRD2_B + 1 : 0;
}
__host__ __device__ inline long q2_ngroups(int n) {
    long t = 0;
    for (int s0 = 0; s0 < n - 1; s0 += Q2_NBK) t += q2_nwin(n, s0);
    return t;
}

// masked load of the V parallelogram of group (s0, k) into sV[ci * LDV + r] (zero padded to LW x NBK)
template <class T>
__device__ __forceinline__ void q2_load_v(T *sV, const T *V2, long ldv, int n, int s0, int ns, int k, int nthreads) {
    constexpr int b = TRD2_B;
    const int w0 = s0 + 1 + k * b;
    for (int e = threadIdx.x; e < Q2_LW * Q2_NBK; e += nthreads) {
        const int r = e % Q2_LW, ci = e / Q2_LW;
        const int s = s0 + ci, gr = w0 + r;
        T v = Ops<T>::zero();
        if (ci < ns && gr >= s + 1 + k * b && gr <= min(s + (k + 1) * b, n - 1)) v = V2[gr + (long)s * ldv];
        sV[ci * Q2_LDV + r] = v;
    }
}

template <class T>
__global__ void __launch_bounds__(256) q2_tfactor_kernel(int n, const T *V2, long ldv, long sV2, const T *tau2, long sTau2,
                                                         T *Tst, long sTst) {
    typedef Ops<T> O;
    constexpr int NBK = Q2_NBK;
    const int I = blockIdx.x, k = blockIdx.y, item = blockIdx.z;
    const int s0 = I * NBK;
    if (k >= q2_nwin(n, s0)) return;
    const int ns = min(NBK, n - 1 - s0);
    V2 += (long)item * sV2; tau2 += (long)item * sTau2; Tst += (long)item * sTst;
    long goff = 0;
    for (int s = 0; s < s0; s += NBK) goff += q2_nwin(n, s);
    T *Tout = Tst + (goff + k) * NBK * NBK;

    extern __shared__ __align__(16) unsigned char q2t_smem[];
    T *sV = (T *)q2t_smem;                    // [NBK][LDV]
    __shared__ T sG[NBK][NBK + 1], sT[NBK][NBK + 1], s_tau[NBK];
    const int tid = threadIdx.x;
    q2_load_v<T>(sV, V2, ldv, n, s0, ns, k, 256);
    if (tid < NBK) s_tau[tid] = tid < ns ? tau2[(long)k * n + s0 + tid] : O::zero();
    for (int e = tid; e < NBK * NBK; e += 256) sT[e / NBK][e % NBK] = O::zero();
    __syncthreads();
    // G = V^H V (upper part is what the recurrence reads)
    for (int e = tid; e < NBK * NBK; e += 256) {
        const int i = e % NBK, j = e / NBK;
        T s = O::zero();
        if (i < j) for (int r = 0; r < Q2_LW; ++r) s = O::add(s, O::conj_mul(sV[i * Q2_LDV + r], sV[j * Q2_LDV + r]));
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
    for (int e = tid; e < NBK * NBK; e += 256) Tout[e] = sT[e % NBK][e / NBK];      // column-major, ld = NBK
}

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// acc (+)= A(8 x 4) B(4 x 8) for real / complex scalars; CONJA conjugates the A fragment, NEG negates it
template <class T, bool CONJA, bool NEG> struct Frag;
template <bool CONJA, bool NEG> struct Frag<double, CONJA, NEG> {
    static __device__ __forceinline__ void mma(double (&acc)[4], double a, double b) {
#ifdef Q2_SKIP_MMA
        acc[0] += a; acc[1] += b;
#else
        dmma884(acc[0], acc[1], NEG ? -a : a, b);
#endif
    }
};
template <bool CONJA, bool NEG> struct Frag<cplx, CONJA, NEG> {
    static __device__ __forceinline__ void mma(double (&acc)[4], cplx a, cplx b) {
        double ar = NEG ? -a.x : a.x, ai = (CONJA != NEG) ? -a.y : a.y;
        dmma884(acc[0], acc[1], ar, b.x);
        dmma884(acc[0], acc[1], -ai, b.y);
        dmma884(acc[2], acc[3], ar, b.y);
        dmma884(acc[2], acc[3], ai, b.x);
    }
};
template <class T> __device__ __forceinline__ T frag_out(const double (&acc)[4], int q);
template <> __device__ __forceinline__ double frag_out<double>(const double (&acc)[4], int q) { return acc[q]; }
template <> __device__ __forceinline__ cplx frag_out<cplx>(const double (&acc)[4], int q) { return make_double2(acc[q], acc[2 + q]); }

template <class T> struct Q2Cfg;
template <> struct Q2Cfg<double> { static const int NCMAX = 32; };     // most columns of Z per CTA (shared memory)
template <> struct Q2Cfg<cplx> { static const int NCMAX = 16; };

template <class T> __device__ __forceinline__ void cp_async_elem(T *s, const T *g, bool pred) {
    if constexpr (sizeof(T) == 16) cp_async16(s, g, pred); else cp_async8(s, g, pred);
}

// NW warps: warp & 3 selects the 8-row tile (of W: reflectors ci; of the window: rows w, w+4, w+8), warp >> 2 the slice of the
// slab's columns (NW = 8: two slices).  DB: V and T of the NEXT diamond are fetched into a second buffer while this one is
// applied (one CTA per SM, 8 warps, wide slab); otherwise the co-resident second CTA hides the load.
template <class T, int NC, int NW, bool DB, bool ALIAS>
__global__ void __launch_bounds__(NW * 32) q2_apply_kernel(int n, int ncols, const T *V2, long ldv, long sV2, const T *Tst,
                                                           long sTst, T *Z, long ldz, long sZ) {
    typedef Ops<T> O;
    constexpr int b = TRD2_B, NBK = Q2_NBK, LW = Q2_LW, CS = NW / 4, NCW = NC / CS, NCT = NCW / 8, LDV = Q2_LDV, LDW = Q2_LDW,
                  LDT = Q2Ldt<T>::value, NBUF = DB ? 2 : 1, NTH = NW * 32;
    static_assert(NW == 4 || NW == 8, "4 or 8 warps");
    static_assert(NC % (8 * CS) == 0 && NC % NW == 0, "slab width");
    const int item = blockIdx.y, c0 = blockIdx.x * NC;
    V2 += (long)item * sV2; Tst += (long)item * sTst; Z += (long)item * sZ;
    extern __shared__ __align__(16) unsigned char q2_smem[];
    T *sVb = (T *)q2_smem;                // [NBUF][NBK][LDV]
    T *sZ_ = sVb + NBUF * NBK * LDV;      // [NC][LDV]   window of Z, kept across the windows of an S-block
    T *sTb = sZ_ + NC * LDV;              // [NBUF][NBK][LDT]  T(i,k) at k*LDT + i
    T *sW = sTb + NBUF * NBK * LDT;       // [NC][LDW]   W(ci,c) at c*LDW + ci
    T *sW2 = ALIAS ? sW : sW + NC * LDW;  // [NC][LDW]   (ALIAS: W2 overwrites W after a barrier -- smaller footprint, 3 CTAs per SM)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, lr = lane >> 2, lc = lane & 3;
    const int wr = warp & 3, col0 = (warp >> 2) * NCW;

    // rows [ra, LW) of the window starting at global row w0 (Lw valid rows) from global memory, zero beyond Lw.
    // warp <-> columns c = warp, warp + NW, ...; lane <-> rows: no integer division anywhere in the window loop
    T *const zwarp = Z + (long)(c0 + warp) * ldz;          // this warp's first column; its columns are NW apart
    const long zstep = (long)NW * ldz;
    auto load_z = [&](int w0, int Lw, int ra) {
        const T *zc = zwarp + w0 + ra + lane;
        T *sz = sZ_ + warp * LDV + ra + lane;
#pragma unroll
        for (int jj = 0; jj < NC / NW; ++jj) {
            const bool cok = c0 + warp + jj * NW < ncols;
#pragma unroll
            for (int rr = 0; rr < LW; rr += 32) {
                const int r = ra + rr + lane;
                if (r < LW) {
                    const bool ok = cok && r < Lw;
                    cp_async_elem<T>(sz + jj * NW * LDV + rr, ok ? zc + rr : Z, ok);
                }
            }
            zc += zstep;
        }
    };
    const int nsweeps = n - 1;
    // V (masked parallelogram) and T of the diamond (s0, k), asynchronous
    auto load_vt = [&](int buf, int s0, int k, long gidx) {
        const int ns = min(NBK, nsweeps - s0), w0 = s0 + 1 + k * b;
        T *sV = sVb + buf * NBK * LDV, *sT = sTb + buf * NBK * LDT;
#pragma unroll
        for (int ci = warp; ci < NBK; ci += NW) {
            const int s = s0 + ci;
            const int a0 = s + 1 + k * b - w0, a1 = min(s + (k + 1) * b, n - 1) - w0;     // valid window rows of column ci
            const T *vc = V2 + w0 + (long)s * ldv;
#pragma unroll
            for (int rr = 0; rr < LW; rr += 32) {
                const int r = rr + lane;
                const bool ok = ci < ns && r >= a0 && r <= a1;
                cp_async_elem<T>(sV + ci * LDV + r, ok ? vc + r : V2, ok);
            }
        }
        const T *Tg = Tst + gidx * NBK * NBK;
#pragma unroll
        for (int e = tid; e < NBK * NBK; e += NTH) cp_async_elem<T>(sT + (e >> 5) * LDT + (e & 31), Tg + e, true);
    };

    const int nS = (nsweeps + NBK - 1) / NBK;
    long goff = q2_ngroups(n);
    int cur = 0;
    if (DB && nS > 0) load_vt(0, (nS - 1) * NBK, 0, goff - q2_nwin(n, (nS - 1) * NBK));
    for (int I = nS - 1; I >= 0; --I) {
        const int s0 = I * NBK, ns = min(NBK, nsweeps - s0), nwin = q2_nwin(n, s0);
        goff -= nwin;
        for (int k = 0; k < nwin; ++k) {
            const int w0 = s0 + 1 + k * b;
            const int Lw = min(s0 + ns - 1 + (k + 1) * b, n - 1) - w0 + 1;
            if (!DB) load_vt(0, s0, k, goff + k);
            if (k == 0) load_z(w0, Lw, 0);
            cp_async_commit();
            cp_async_wait<0>();
            __syncthreads();
            const T *sV = sVb + cur * NBK * LDV, *sT = sTb + cur * NBK * LDT;
            if (DB) {
                // the next diamond: (I, k+1), or the first one of S-block I-1
                if (k + 1 < nwin) load_vt(cur ^ 1, s0, k + 1, goff + k + 1);
                else if (I > 0) load_vt(cur ^ 1, s0 - NBK, 0, goff - q2_nwin(n, s0 - NBK));
                cp_async_commit();
                cur ^= 1;
            }
            // Zero structure of the parallelogram: column ci of V is non-zero only in rows ci .. ci + b - 1, so
            //   W rows 8w..8w+7 need window rows 8w .. 8w + b + 7 only (18 of 24 k-steps), and
            //   Z_w row tile m0 needs columns ci in [m0 - b + 1, m0 + 7]           (72 of 96 k-steps over the 12 tiles).
            // ---- W = V^H Z_w : warp -> 8 rows (ci) x NCW columns; fragments of step k0+4 are loaded before the DMMAs of k0
            {
                double acc[NCT][4];
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[j][q] = 0.0;
                constexpr int KS1 = (b + 8) / 4;                                  // 18 k-steps
                const T *ap = sV + (wr * 8 + lr) * LDV + lc + wr * 8;
                const T *bp = sZ_ + (col0 + lr) * LDV + lc + wr * 8;
                T a_c = ap[0], b_c[NCT];
#pragma unroll
                for (int j = 0; j < NCT; ++j) b_c[j] = bp[j * 8 * LDV];
#pragma unroll
                for (int ks = 0; ks < KS1; ++ks) {
                    T a_n = a_c, b_n[NCT];
#pragma unroll
                    for (int j = 0; j < NCT; ++j) b_n[j] = b_c[j];
                    if (ks + 1 < KS1) {
                        a_n = ap[(ks + 1) * 4];
#pragma unroll
                        for (int j = 0; j < NCT; ++j) b_n[j] = bp[j * 8 * LDV + (ks + 1) * 4];
                    }
#pragma unroll
                    for (int j = 0; j < NCT; ++j) Frag<T, true, false>::mma(acc[j], a_c, b_c[j]);
                    a_c = a_n;
#pragma unroll
                    for (int j = 0; j < NCT; ++j) b_c[j] = b_n[j];
                }
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 2; ++q) sW[(col0 + j * 8 + 2 * lc + q) * LDW + wr * 8 + lr] = frag_out<T>(acc[j], q);
            }
            __syncthreads();
            // ---- W2 = T W   (T upper triangular: rows 8w.. need k >= 8w)
            {
                double acc[NCT][4];
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[j][q] = 0.0;
                const T *ap = sT + lc * LDT + wr * 8 + lr;
                const T *bp = sW + (col0 + lr) * LDW + lc;
                for (int k0 = wr * 8; k0 < NBK; k0 += 4) {
                    const T a = ap[k0 * LDT];
#pragma unroll
                    for (int j = 0; j < NCT; ++j) Frag<T, false, false>::mma(acc[j], a, bp[j * 8 * LDW + k0]);
                }
                if (ALIAS) __syncthreads();
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 2; ++q) sW2[(col0 + j * 8 + 2 * lc + q) * LDW + wr * 8 + lr] = frag_out<T>(acc[j], q);
            }
            __syncthreads();
            // ---- Z_w -= V W2 : warp -> row tiles w, w+4, w+8 (balanced: 18 k-steps per warp), in place in shared memory
#pragma unroll
            for (int i = 0; i < 3; ++i) {
                const int m0 = (wr + i * 4) * 8;
                const int klo = max(0, m0 - b + 1) / 4 * 4, khi = min(NBK, m0 + 8);    // columns ci of V that touch the tile
                double acc[NCT][4];
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const T z = sZ_[(col0 + j * 8 + 2 * lc + q) * LDV + m0 + lr];
                        if constexpr (O::is_complex) { acc[j][q] = z.x; acc[j][2 + q] = z.y; } else { acc[j][q] = z; acc[j][2 + q] = 0.0; }
                    }
                const T *ap = sV + lc * LDV + m0 + lr;
                const T *bp = sW2 + (col0 + lr) * LDW + lc;
                T a_c = ap[klo * LDV], b_c[NCT];
#pragma unroll
                for (int j = 0; j < NCT; ++j) b_c[j] = bp[j * 8 * LDW + klo];
                for (int k0 = klo; k0 < khi; k0 += 4) {
                    T a_n = a_c, b_n[NCT];
#pragma unroll
                    for (int j = 0; j < NCT; ++j) b_n[j] = b_c[j];
                    if (k0 + 4 < khi) {
                        a_n = ap[(k0 + 4) * LDV];
#pragma unroll
                        for (int j = 0; j < NCT; ++j) b_n[j] = bp[j * 8 * LDW + k0 + 4];
                    }
#pragma unroll
                    for (int j = 0; j < NCT; ++j) Frag<T, false, true>::mma(acc[j], a_c, b_c[j]);
                    a_c = a_n;
#pragma unroll
                    for (int j = 0; j < NCT; ++j) b_c[j] = b_n[j];
                }
#pragma unroll
                for (int j = 0; j < NCT; ++j)
#pragma unroll
                    for (int q = 0; q < 2; ++q) sZ_[(col0 + j * 8 + 2 * lc + q) * LDV + m0 + lr] = frag_out<T>(acc[j], q);
            }
            __syncthreads();
            // ---- rows leaving the window go to global memory; the overlap with the next window moves to the top
            const bool last = (k + 1 == nwin);
            const int nout = last ? Lw : min(b, Lw);
            if (nout == b) {
                // the common case (b = 64 rows leave): all shared-memory reads of the warp's columns first, then the stores
                T o0[NC / NW], o1[NC / NW];
#pragma unroll
                for (int jj = 0; jj < NC / NW; ++jj) {
                    o0[jj] = sZ_[(warp + jj * NW) * LDV + lane];
                    o1[jj] = sZ_[(warp + jj * NW) * LDV + 32 + lane];
                }
                T *zc = zwarp + w0 + lane;
#pragma unroll
                for (int jj = 0; jj < NC / NW; ++jj) {
                    if (c0 + warp + jj * NW < ncols) { zc[0] = o0[jj]; zc[32] = o1[jj]; }
                    zc += zstep;
                }
            } else {
#pragma unroll
                for (int c = warp; c < NC; c += NW) {
                    if (c0 + c < ncols) {
                        T *zc = Z + w0 + (long)(c0 + c) * ldz;
                        for (int r = lane; r < nout; r += 32) zc[r] = sZ_[c * LDV + r];
                    }
                }
            }
            if (!last) {
                const int nov = Lw - b;                      // rows shared with the next window (<= NBK - 1 <= 31)
                T keep[NC / NW];
#pragma unroll
                for (int jj = 0; jj < NC / NW; ++jj)
                    if (lane < nov) keep[jj] = sZ_[(warp + jj * NW) * LDV + b + lane];
                __syncthreads();
#pragma unroll
                for (int jj = 0; jj < NC / NW; ++jj)
                    if (lane < nov) sZ_[(warp + jj * NW) * LDV + lane] = keep[jj];
                const int Lw2 = min(s0 + ns - 1 + (k + 2) * b, n - 1) - (w0 + b) + 1;
                load_z(w0 + b, Lw2, nov);                    // committed and awaited with the next window's V, T
            } else {
                __syncthreads();
            }
        }
    }
}

size_t q2_workspace(int dtype, int n, int batch) { return align_up((size_t)batch * q2_ngroups(n) * Q2_NBK * Q2_NBK * esize(dtype)); }

template <class T, int NC, int NW, bool DB, bool ALIAS>
static int q2_launch(int n, int ncols, int batch, const T *V2, long ldv, long sV2, const T *Tst, long sTst, T *Z, long ldz, long sZ,
                     cudaStream_t st) {
    const size_t smem = (size_t)(((DB ? 2 : 1) * Q2_NBK + NC) * Q2_LDV + (DB ? 2 : 1) * Q2_NBK * Q2Ldt<T>::value + (ALIAS ? 1 : 2) * NC * Q2_LDW) * sizeof(T);
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(q2_apply_kernel<T, NC, NW, DB, ALIAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    q2_apply_kernel<T, NC, NW, DB, ALIAS><<<dim3(ceil_div(ncols, NC), batch), NW * 32, smem, st>>>(n, ncols, V2, ldv, sV2, Tst, sTst, Z, ldz, sZ);
    NAO_LAUNCHED();
    return NAO_OK;
}

template <class T>
static int q2_apply_impl(int n, int ncols, int batch, const T *V2, long ldv, long sV2, const T *tau2, T *Z, long ldz, long sZ,
                         void *work, cudaStream_t st) {
    if (n < 2) return NAO_OK;
    const long ng = q2_ngroups(n), sTst = ng * Q2_NBK * Q2_NBK, sTau2 = (long)hb2st_nk(n) * n;
    T *Tst = (T *)work;
    const int nS = ceil_div(n - 1, Q2_NBK), kmax = q2_nwin(n, 0);
    const size_t smem_t = (size_t)Q2_NBK * Q2_LDV * sizeof(T);
    constexpr int NCMAX = Q2Cfg<T>::NCMAX;
    static bool attr = false;
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(q2_tfactor_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_t));
        attr = true;
    }
    q2_tfactor_kernel<T><<<dim3(nS, kmax, batch), 256, smem_t, st>>>(n, V2, ldv, sV2, tau2, sTau2, Tst, sTst);
    NAO_LAUNCHED();
    // every CTA walks through all diamonds for its slab of columns: with few columns (partial spectrum) narrower slabs keep
    // all SMs busy
    int nsm = 148, dev = 0;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    int nc = NCMAX;
    while (nc > 8 && (long)ceil_div(ncols, nc) * batch < 2L * nsm) nc /= 2;
    int rc;
    // Real slabs of NCMAX columns: with W2 written over W (one more block barrier) three CTAs fit on an SM; used when two
    // per SM would need a second round of CTAs (config 2, all columns: 416 CTAs > 2 x 148, <= 3 x 148: 117 -> 98 ms;
    // an 8-warp CTA per SM with a 96-column slab and double-buffered V, T measured 121 ms).
    const long ctas = (long)ceil_div(ncols, NCMAX) * batch;
    if (nc == NCMAX && sizeof(T) == 8 && ctas > 2L * nsm)
        rc = q2_launch<T, NCMAX, 4, false, true>(n, ncols, batch, V2, ldv, sV2, Tst, sTst, Z, ldz, sZ, st);
    else if (nc == NCMAX) rc = q2_launch<T, NCMAX, 4, false, false>(n, ncols, batch, V2, ldv, sV2, Tst, sTst, Z, ldz, sZ, st);
    else if (nc == NCMAX / 2) rc = q2_launch<T, NCMAX / 2, 4, false, false>(n, ncols, batch, V2, ldv, sV2, Tst, sTst, Z, ldz, sZ, st);
    else rc = q2_launch<T, 8, 4, false, false>(n, ncols, batch, V2, ldv, sV2, Tst, sTst, Z, ldz, sZ, st);
    if (rc) return rc;
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
