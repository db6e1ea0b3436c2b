// ormtr.cu -- blocked back-transformation Z <- Q Z of the one-stage tridiagonalisation.
#include "nao_internal.cuh"
#include "scalar.cuh"
#include <algorithm>
#include <cmath>

namespace nao {


// ----------------------------------------------------------------------------------------------------------------
// Back-transformation: Z <- Q Z, Q = H(0) H(1) ... H(n-1-shift), H(j) = I - tau_j v_j v_j^H, v_j = A[j+shift:, j] (shift = 1:
// one-stage hetrd; shift = b: dense-to-band he2hb) (unit first
// element stored explicitly by hetrd).  Blocks of KB reflectors, last block first:
//   Vb (explicit, zeros above the unit diagonal), G = Vb^H Vb, T by the xLARFT recurrence, then three GEMMs
//   X = Vb^H Z ; X <- T X ; Z -= Vb X.
// ----------------------------------------------------------------------------------------------------------------
static const int ORM_KB = 128;        // reflectors per T factor built by the recurrence (larft_kernel)
static const int ORM_BLK = 512;       // reflectors per applied block; its T is assembled from 128-blocks by doubling:
                                      // T = [T11 T12; 0 T22], T12 = -T11 (V1^H V2) T22

template <class T>
__global__ void build_v_kernel(int n, int jb, int kb, int shift, const T *A, long lda, long sA, T *V, long ldv, long sV) {
    // V (m x kb), m = n - jb - shift, row r <-> global row jb+shift+r; column k <-> reflector jb+k whose unit sits at r == k
    A += (long)blockIdx.z * sA; V += (long)blockIdx.z * sV;
    const int m = n - jb - shift;
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= m) return;
    for (int k = blockIdx.y; k < kb; k += gridDim.y) {
        T v;
        if (r < k) v = Ops<T>::zero();
        else if (r == k) v = Ops<T>::one();
        else v = A[(jb + shift + r) + (long)(jb + k) * lda];
        V[r + (long)k * ldv] = v;
    }
}

// T (kb x kb upper) from G = V^H V and tau: T(i,i) = tau_i ; T(0:i, i) = -tau_i T(0:i,0:i) G(0:i, i).
// T is built in shared memory in packed upper storage ((r,c), r <= c, at c(c+1)/2 + r) and written out dense.
template <class T>
__global__ void __launch_bounds__(256) larft_kernel(int kb, const T *G, long ldg, long sG, const T *tau, long sTau, T *Tm, long ldt, long sT) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *sT_ = (T *)smem_raw;             // packed upper, kb(kb+1)/2
    __shared__ T s_g[ORM_KB];
    // blockIdx.y: diagonal block of ORM_KB reflectors of a longer sequence (kb = total length); the blocks are independent
    const int boff = blockIdx.y * ORM_KB;
    G += (long)blockIdx.x * sG + boff + (long)boff * ldg; tau += (long)blockIdx.x * sTau + boff;
    Tm += (long)blockIdx.x * sT + boff + (long)boff * ldt;
    kb = min(ORM_KB, kb - boff);
    const int tid = threadIdx.x;
    // column i+1 of G and tau_{i+1} are fetched while step i computes (the recurrence is latency bound)
    T gnext = Ops<T>::zero(), tnext = tau[0];
    for (int i = 0; i < kb; ++i) {
        const T ti = tnext;
        if (tid < i) s_g[tid] = gnext;
        if (i + 1 < kb) { tnext = tau[i + 1]; if (tid < i + 1) gnext = G[tid + (long)(i + 1) * ldg]; }
        __syncthreads();
        {
            // row `row` of T(0:i,0:i) times g (T upper: columns c >= row): two adjacent lanes split the columns, two
            // accumulators each (the recurrence is bound by the latency of this dependent chain)
            const int row = tid >> 1, half = tid & 1;
            T acc0 = Ops<T>::zero(), acc1 = Ops<T>::zero();
            if (row < i) {
                int c = row + half;
                for (; c + 2 < i; c += 4) {
                    acc0 = Ops<T>::fma(sT_[c * (c + 1) / 2 + row], s_g[c], acc0);
                    acc1 = Ops<T>::fma(sT_[(c + 2) * (c + 3) / 2 + row], s_g[c + 2], acc1);
                }
                for (; c < i; c += 2) acc0 = Ops<T>::fma(sT_[c * (c + 1) / 2 + row], s_g[c], acc0);
            }
            T acc = Ops<T>::add(acc0, acc1);
            double *a = (double *)&acc;
#pragma unroll
            for (int w = 0; w < (int)(sizeof(T) / 8); ++w) a[w] += __shfl_xor_sync(0xffffffffu, a[w], 1);
            if (row < i && half == 0) sT_[i * (i + 1) / 2 + row] = Ops<T>::sub(Ops<T>::zero(), Ops<T>::mul(ti, acc));
        }
        if (tid == 0) sT_[i * (i + 1) / 2 + i] = ti;
        __syncthreads();
    }
    for (int e = tid; e < kb * kb; e += blockDim.x) {
        const int r = e % kb, c = e / kb;
        Tm[r + (long)c * ldt] = r <= c ? sT_[c * (c + 1) / 2 + r] : Ops<T>::zero();
    }
}

template <class T> static int larft_attr() {
    static bool attr = false;
    if (!attr) {
        const size_t smem = (size_t)ORM_KB * (ORM_KB + 1) / 2 * sizeof(T);
        NAO_CUDA_CHECK(cudaFuncSetAttribute(larft_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    return NAO_OK;
}

int build_v(int dtype, int n, int jb, int kb, int shift, const void *A, long lda, long sA, void *V, long ldv, long sV, int batch,
            cudaStream_t st) {
    const int m = n - jb - shift;
    if (m <= 0 || kb <= 0) return NAO_OK;
    dim3 grid(ceil_div(m, 256), kb, batch);
    if (dtype == NAO_COMPLEX) build_v_kernel<cplx><<<grid, 256, 0, st>>>(n, jb, kb, shift, (const cplx *)A, lda, sA, (cplx *)V, ldv, sV);
    else build_v_kernel<double><<<grid, 256, 0, st>>>(n, jb, kb, shift, (const double *)A, lda, sA, (double *)V, ldv, sV);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int larft(int dtype, int kb, const void *G, long ldg, long sG, const void *tau, long sTau, void *Tm, long sT, int batch,
          cudaStream_t st) {
    if (kb <= 0) return NAO_OK;
    if (kb > ORM_KB) return NAO_ERR_UNSUPPORTED;
    if (dtype == NAO_COMPLEX) {
        if (int rc = larft_attr<cplx>()) return rc;
        larft_kernel<cplx><<<batch, 256, (size_t)kb * (kb + 1) / 2 * sizeof(cplx), st>>>(kb, (const cplx *)G, ldg, sG, (const cplx *)tau, sTau, (cplx *)Tm, kb, sT);
    } else {
        if (int rc = larft_attr<double>()) return rc;
        larft_kernel<double><<<batch, 256, (size_t)kb * (kb + 1) / 2 * sizeof(double), st>>>(kb, (const double *)G, ldg, sG, (const double *)tau, sTau, (double *)Tm, kb, sT);
    }
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

struct OrmWork { void *V, *G, *T, *X, *X2, *P, *Vs, *tmp, *Ps; size_t bytes; int ksG, ksX; };
static OrmWork orm_plan(int dtype, int n, int ncols, int batch, void *work) {
    OrmWork w; const size_t es = esize(dtype);
    Arena ar(work, (size_t)-1);
    // split-K factors for the two tall-skinny^H products (k = m up to n): fill ~2 waves of 148 SMs
    // (one CTA per SM: with a few waves of tiles the last, partly filled wave is a measurable loss -- config 3: 624 tiles =
    // 4.2 waves; the split factor is chosen to fill the last wave: 4 slices = 16.9 waves)
    const int tilesX = (ORM_BLK / 128) * ceil_div(ncols, dtype == NAO_COMPLEX ? 64 : 128) * batch;
    const int nsm = sm_count();
    w.ksX = fill_ksplit(tilesX, nsm, std::max(1, std::min(std::min(8, ceil_div(n, 1024)), std::max(1, 20 * nsm / std::max(1, tilesX)))));
    const int tilesG = (ORM_BLK / 128) * (dtype == NAO_COMPLEX ? 4 : 2) * batch;
    w.ksG = std::max(1, std::min(std::min(148 / std::max(1, tilesG), ceil_div(n, 256)), 64));
    w.V = ar.take((size_t)batch * n * ORM_BLK * es);
    w.G = ar.take((size_t)batch * ORM_BLK * ORM_BLK * es);
    w.T = ar.take((size_t)2 * batch * ORM_BLK * ORM_BLK * es);          // two T factors: the next block's is built ahead
    w.X = ar.take((size_t)batch * ORM_BLK * ncols * es);
    w.X2 = ar.take((size_t)batch * ORM_BLK * std::max(ncols, ORM_BLK) * es);
    w.P = ar.take((size_t)batch * std::max((size_t)w.ksX * ORM_BLK * ncols, (size_t)w.ksG * ORM_BLK * ORM_BLK) * es);
    // look-ahead of the T factor (side stream): its own explicit V, small temporary and split-K scratch
    w.Vs = ar.take((size_t)batch * n * ORM_BLK * es);
    w.tmp = ar.take((size_t)batch * ORM_BLK * ORM_BLK * es);
    w.Ps = ar.take((size_t)batch * w.ksG * ORM_BLK * ORM_BLK * es);
    w.bytes = ar.off;
    return w;
}
size_t ormtr_workspace(int dtype, int n, int batch) { return orm_plan(dtype, n, n, batch, nullptr).bytes; }

template <class T>
static int ormtr_impl(int dtype, int n, int ncols, int batch, int shift, const T *A, long lda, long sA, const T *tau, T *Z,
                      long ldz, long sZ, void *work, cudaStream_t st) {
    if (n < shift + 1) return NAO_OK;
    OrmWork w = orm_plan(dtype, n, ncols, batch, work);
    const int nref = n - shift;
    static bool attr = false;
    const size_t larft_smem = (size_t)ORM_KB * (ORM_KB + 1) / 2 * sizeof(T);
    if (!attr) {
        NAO_CUDA_CHECK(cudaFuncSetAttribute(larft_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)larft_smem));
        attr = true;
    }
    // few columns (partial spectrum): the cost of building T (G = V^H V is kb^2 m flops per block) matters next to the
    // two products, so the block is halved
    const int BLK = (4 * ncols >= n) ? ORM_BLK : ORM_BLK / 2;
    const int nblocks = ceil_div(nref, BLK);
    const long sGT = (long)ORM_BLK * ORM_BLK, sX = (long)ORM_BLK * ncols, sX2 = (long)ORM_BLK * std::max(ncols, ORM_BLK);
    const long sV = (long)n * ORM_BLK;
    // The T factor of a block depends on the reflectors only, not on Z: a chain of small launches (explicit V, G = V^H V, the
    // xLARFT recurrence on the diagonal 128-blocks, off-diagonal blocks by doubling).  The factor of block blk-1 is built on
    // an internal high-priority side stream while the three large products of block blk run on the caller's stream.
    // (Not while a stream group limits the SMs: the groups overlap one another instead.)
    static SideSet ss = {};
    const bool ahead = sm_count() >= device_sms() && nblocks > 1 && n >= 1024;
    if (ahead) if (int rc = side_set_init(ss, 1, 3, true)) return rc;
    const cudaStream_t side = ss.stream[0];
    const cudaEvent_t ev_fork = ss.event[0], ev_T = ss.event[1];
    SideJoin join(side, st, ss.event[2]);      // armed at the first fork: every exit path rejoins the side stream
    // T factor of block blk into Tm (kb x kb, ld kb) on stream qs; Vx = explicit V of the block (output), Gx, tmpx, Px = scratch
    auto build_t = [&](int blk, T *Tm, T *Vx, T *Gx, T *tmpx, void *Px, cudaStream_t qs) -> int {
        const int jb = blk * BLK, kb = std::min(BLK, nref - jb), m = n - jb - shift;
        const long ldv = m;
        build_v_kernel<T><<<dim3(ceil_div(m, 256), kb, batch), 256, 0, qs>>>(n, jb, kb, shift, A, lda, sA, Vx, ldv, sV);
        NAO_LAUNCHED();
        // G = V^H V  (kb x kb, k = m: split-K)
        GemmDesc g = gemm_desc(OP_C, OP_N, kb, kb, m, 1.0, Vx, ldv, Vx, ldv, 0.0, Gx, kb);
        g.sA = sV; g.sB = sV; g.sC = sGT;
        if (int rc = gemm_splitk(dtype, g, batch, std::min(w.ksG, ceil_div(m, 256)), Px, qs)) return rc;
        // T: recurrence on the diagonal 128-blocks, then off-diagonal blocks by doubling (two small GEMMs each)
        larft_kernel<T><<<dim3(batch, ceil_div(kb, ORM_KB)), 256, larft_smem, qs>>>(kb, Gx, kb, sGT, tau + jb, n, Tm, kb, sGT);
        NAO_LAUNCHED();
        for (int sz = ORM_KB; sz < kb; sz *= 2)
            for (int off = 0; off + sz < kb; off += 2 * sz) {
                const int k1 = sz, k2 = std::min(sz, kb - off - sz), o2 = off + sz;
                // tmp = G12 T22 ; T12 = -T11 tmp
                GemmDesc t1 = gemm_desc(OP_N, OP_N, k1, k2, k2, 1.0, Gx + off + (long)o2 * kb, kb, Tm + o2 + (long)o2 * kb, kb, 0.0, tmpx, k1);
                t1.sA = sGT; t1.sB = sGT; t1.sC = sGT; t1.maskB = MASK_UPPER;
                if (int rc = gemm_launch(dtype, t1, batch, qs)) return rc;
                GemmDesc t2 = gemm_desc(OP_N, OP_N, k1, k2, k1, -1.0, Tm + off + (long)off * kb, kb, tmpx, k1, 0.0, Tm + off + (long)o2 * kb, kb);
                t2.sA = sGT; t2.sB = sGT; t2.sC = sGT; t2.maskA = MASK_UPPER;
                if (int rc = gemm_launch(dtype, t2, batch, qs)) return rc;
            }
        return NAO_OK;
    };
    T *Tbuf[2] = {(T *)w.T, (T *)w.T + (long)batch * sGT};
    // first block: everything on the caller's stream
    if (int rc = build_t(nblocks - 1, Tbuf[(nblocks - 1) & 1], (T *)w.V, (T *)w.G, (T *)w.tmp, w.P, st)) return rc;
    for (int blk = nblocks - 1; blk >= 0; --blk) {
        const int jb = blk * BLK, kb = std::min(BLK, nref - jb), m = n - jb - shift;
        const long ldv = m;
        T *Tm = Tbuf[blk & 1];
        if (blk < nblocks - 1) {
            if (ahead) NAO_CUDA_CHECK(cudaStreamWaitEvent(st, ev_T, 0));          // T(blk) built ahead on the side stream
            // explicit V of this block for the large products (the side stream used its own copy)
            build_v_kernel<T><<<dim3(ceil_div(m, 256), kb, batch), 256, 0, st>>>(n, jb, kb, shift, A, lda, sA, (T *)w.V, ldv, sV);
            NAO_LAUNCHED();
        }
        if (blk > 0) {
            if (ahead) {
                // everything enqueued so far (incl. the last use of the other T buffer) precedes the side stream's work
                NAO_CUDA_CHECK(cudaEventRecord(ev_fork, st));
                NAO_CUDA_CHECK(cudaStreamWaitEvent(side, ev_fork, 0));
                join.arm();
                if (int rc = build_t(blk - 1, Tbuf[(blk - 1) & 1], (T *)w.Vs, (T *)w.G, (T *)w.tmp, w.Ps, side)) return rc;
                NAO_CUDA_CHECK(cudaEventRecord(ev_T, side));
            }
        }
        // X = V^H Z[jb+shift:, :]  (kb x ncols, k = m: split-K)
        GemmDesc x = gemm_desc(OP_C, OP_N, kb, ncols, m, 1.0, w.V, ldv, Z + jb + shift, ldz, 0.0, w.X, kb);
        x.sA = sV; x.sB = sZ; x.sC = sX;
        if (int rc = gemm_splitk(dtype, x, batch, std::min(w.ksX, ceil_div(m, 512)), w.P, st)) return rc;
        // X2 = T X  (T upper triangular: elements below the diagonal are never read)
        GemmDesc t = gemm_desc(OP_N, OP_N, kb, ncols, kb, 1.0, Tm, kb, w.X, kb, 0.0, w.X2, kb);
        t.sA = sGT; t.sB = sX; t.sC = sX2; t.maskA = MASK_UPPER;
        if (int rc = gemm_launch(dtype, t, batch, st)) return rc;
        // Z[jb+shift:, :] -= V X2
        GemmDesc u = gemm_desc(OP_N, OP_N, m, ncols, kb, -1.0, w.V, ldv, w.X2, kb, 1.0, Z + jb + shift, ldz);
        u.sA = sV; u.sB = sX2; u.sC = sZ;
        if (int rc = gemm_launch(dtype, u, batch, st)) return rc;
        if (blk > 0 && !ahead)
            if (int rc = build_t(blk - 1, Tbuf[(blk - 1) & 1], (T *)w.V, (T *)w.G, (T *)w.tmp, w.P, st)) return rc;
    }
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

int ormtr(int dtype, int n, int ncols, int batch, int shift, const void *A, long lda, long sA, const void *tau, void *Z,
          long ldz, long sZ, void *work, cudaStream_t st) {
    return dtype == NAO_COMPLEX
               ? ormtr_impl<cplx>(dtype, n, ncols, batch, shift, (const cplx *)A, lda, sA, (const cplx *)tau, (cplx *)Z, ldz, sZ, work, st)
               : ormtr_impl<double>(dtype, n, ncols, batch, shift, (const double *)A, lda, sA, (const double *)tau, (double *)Z, ldz, sZ, work, st);
}

}  // namespace nao
