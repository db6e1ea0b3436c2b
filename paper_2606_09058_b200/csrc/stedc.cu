// stedc.cu -- symmetric tridiagonal eigensolver by divide and conquer, all eigenpairs.
//
// Tree of rank-one tears fixed on the host (leaves <= 32, all at the same depth); every level of the tree is a fixed
// sequence of launches over ALL merges of that level and ALL batch items, with no host round trip: the number K of
// non-deflated poles of each merge is known only on the device, so kernels are launched for the worst case and
// exit early, and the two merge GEMMs per node read m,n,k from descriptors written by the set-up kernel.
//   leaf    : one warp per leaf, implicit QL; every lane runs the scalar recurrence and rotates its own row of Z
//   set-up  : z vector, merge of the children's sorted orders, deflation scan (one thread, inputs staged through
//             shared memory), column grouping by type (top-only / dense / bottom-only / deflated), GEMM descriptors
//   rotate  : Givens rotations of the deflation applied to the columns of Q (thread per row)
//   permute : Q -> Qw in grouped order; deflated columns copied back
//   secular : one WARP per root (lanes split the pole sums, xor-shuffle all-reduce), origin-shifted so that the
//             differences d_i - lambda_j are accurate; they are stored in the (free) first K columns of the Q block
//   zhat    : Loewner / Gu-Eisenstat weights from those differences
//   vectors : normalised eigenvectors of D + rho z z^T, rows permuted to the grouped order
//   GEMM    : Q_top = Qw_top(types 1,2) * S ;  Q_bot = Qw_bot(types 2,3) * S   on the DMMA core (structural zeros skipped)
//   finish  : new d, merged sorted order
#include "nao_internal.cuh"
#include "scalar.cuh"
#include "stedc_core.cuh"
#include <vector>

namespace nao {

static const int DC_LEAF = 32;

struct WarpLanes {
    __device__ __forceinline__ int lane() const { return threadIdx.x & 31; }
    __device__ __forceinline__ int count() const { return 32; }
    __device__ __forceinline__ double sum(double v) const { return warp_sum(v); }
};

struct DcNode { int off, n1, n2; };
struct DcOut { int K, c1, c2, c3, nrot, pad; double rho; };

// per-item device arrays (each of length n unless noted)
struct DcBuf {
    double *d, *e;                 // working diagonal / off-diagonal (caller's arrays)
    double *Q; long ldq, sQ;       // eigenvector accumulation buffer
    double *Qw, *S;                // n x n each, ld n
    double *z, *dlam, *wz, *dcol, *dnew, *zhat, *rot_c, *rot_s, *ds, *zs, *scale;
    int *idxq, *src, *indxp, *coltyp, *gcol, *gsec, *rot_p, *rot_q;
    int *kneed;                    // per item: secular roots of the top merge among the wanted eigenvalues
    DcOut *out;                    // per node of the current level (max nodes per level entries)
    GemmDesc *desc;                // 2 per node
    int n;
};
// all per-item arrays are laid out with item stride `n` (out/desc: stride maxnodes / 2*maxnodes)

__device__ __forceinline__ double block_max(double v, double *red) {
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double m = red[0];
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, red[w]);
    __syncthreads();
    return m;
}

// ------------------------------------------------------------------------------------------------ scale + tear
__global__ void __launch_bounds__(256) dc_scale_tear_kernel(DcBuf b, const int *__restrict__ cuts, int ncuts) {
    __shared__ double red[8];
    const int item = blockIdx.x, n = b.n;
    double *d = b.d + (long)item * n, *e = b.e + (long)item * n;
    double m = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        m = fmax(m, fabs(d[i]));
        if (i + 1 < n) m = fmax(m, fabs(e[i]));
    }
    m = block_max(m, red);
    const double sc = m > 0.0 ? 1.0 / m : 1.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) { d[i] *= sc; if (i + 1 < n) e[i] *= sc; }
    if (threadIdx.x == 0) b.scale[item] = m > 0.0 ? m : 1.0;
    __syncthreads();
    for (int c = threadIdx.x; c < ncuts; c += blockDim.x) {
        const int cut = cuts[c];                    // first index of the right part
        const double r = fabs(e[cut - 1]);
        d[cut - 1] -= r; d[cut] -= r;
    }
}

// ------------------------------------------------------------------------------------------------ leaves
__global__ void __launch_bounds__(128) dc_leaf_kernel(DcBuf b, const int *__restrict__ leaf_off, int nleaves, int *info) {
    const int item = blockIdx.y, n = b.n;
    const int leaf = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (leaf >= nleaves) return;
    const int o = leaf_off[leaf], m = leaf_off[leaf + 1] - o;
    double *d = b.d + (long)item * n, *e = b.e + (long)item * n;
    double *Q = b.Q + (long)item * b.sQ;
    double dl[DC_LEAF], el[DC_LEAF], zr[DC_LEAF];
    for (int i = 0; i < DC_LEAF; ++i) {
        dl[i] = i < m ? d[o + i] : 0.0;
        el[i] = (i + 1 < m) ? e[o + i] : 0.0;
        zr[i] = (i == lane) ? 1.0 : 0.0;
    }
    auto emit = [&](int i, double c, double s) {
        const double f = zr[i + 1];
        zr[i + 1] = s * zr[i] + c * f;
        zr[i] = c * zr[i] - s * f;
    };
    const int rc = dc::ql_implicit(m, dl, el, emit);
    if (rc && lane == 0) info[item] = n + 1;
    // ascending order: rank of each eigenvalue (ties by index)
    for (int c = 0; c < m; ++c) {
        int rank = 0;
        for (int t = 0; t < m; ++t) rank += (dl[t] < dl[c]) || (dl[t] == dl[c] && t < c);
        if (lane < m) Q[(o + lane) + (long)(o + rank) * b.ldq] = zr[c];
        if (lane == 0) { d[o + rank] = dl[c]; }
    }
    if (lane < m) b.idxq[(long)item * n + o + lane] = lane;
}

// ------------------------------------------------------------------------------------------------ set-up of a merge
static const int DC_CH = 1024;

__global__ void __launch_bounds__(1024) dc_setup_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int nn) {
    __shared__ double red[32];
    __shared__ double ds_s[DC_CH], zs_s[DC_CH];
    __shared__ int src_s[DC_CH];
    __shared__ dc::DeflateState st;
    __shared__ int cnt[1024][3];
    const int node = blockIdx.x, item = blockIdx.y, n = b.n, tid = threadIdx.x, nt = blockDim.x;
    const DcNode nd = nodes[node];
    const int off = nd.off, n1 = nd.n1, n2 = nd.n2, N = n1 + n2;
    const long ib = (long)item * n + off;               // base of this node's slices in the per-item arrays
    double *d = b.d + ib; const double *e = b.e + (long)item * n;
    double *Qb = b.Q + (long)item * b.sQ + off + (long)off * b.ldq;
    double *z = b.z + ib, *dlam = b.dlam + ib, *wz = b.wz + ib, *dcol = b.dcol + ib, *ds = b.ds + ib, *zs = b.zs + ib;
    double *rot_c = b.rot_c + ib, *rot_s = b.rot_s + ib;
    int *idxq = b.idxq + ib, *src = b.src + ib, *indxp = b.indxp + ib, *coltyp = b.coltyp + ib, *gcol = b.gcol + ib,
        *gsec = b.gsec + ib, *rot_p = b.rot_p + ib, *rot_q = b.rot_q + ib;

    double rho = e[off + n1 - 1];
    const double sgn = rho < 0.0 ? -1.0 : 1.0;
    double zmax = 0.0, dmax = 0.0;
    for (int c = tid; c < N; c += nt) {
        double v = (c < n1) ? Qb[(n1 - 1) + (long)c * b.ldq] : sgn * Qb[n1 + (long)c * b.ldq];
        v *= 0.70710678118654752440;
        z[c] = v;
        zmax = fmax(zmax, fabs(v)); dmax = fmax(dmax, fabs(d[c]));
    }
    zmax = block_max(zmax, red); dmax = block_max(dmax, red);
    rho = fabs(2.0 * rho);
    const double tol = 8.0 * dc::DC_EPS * fmax(dmax, zmax);
    __syncthreads();
    // sorted order of all N values: merge of the children's sorted orders by binary search
    for (int i = tid; i < N; i += nt) {
        int pos, col;
        if (i < n1) {
            col = idxq[i];
            const double a = d[col];
            int lo = 0, hi = n2;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (d[n1 + idxq[n1 + mid]] < a) lo = mid + 1; else hi = mid; }
            pos = i + lo;
        } else {
            const int ii = i - n1;
            col = n1 + idxq[n1 + ii];
            const double bb = d[col];
            int lo = 0, hi = n1;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (d[idxq[mid]] <= bb) lo = mid + 1; else hi = mid; }
            pos = ii + lo;
        }
        src[pos] = col; ds[pos] = d[col]; zs[pos] = z[col];
    }
    if (tid == 0) dc::deflate_init(st, N, rho, tol);
    __syncthreads();
    // deflation scan: thread 0, inputs staged in chunks
    for (int jb = 0; jb < N; jb += DC_CH) {
        const int je = min(N, jb + DC_CH);
        for (int t = tid; t < je - jb; t += nt) { ds_s[t] = ds[jb + t]; zs_s[t] = zs[jb + t]; src_s[t] = src[jb + t]; }
        __syncthreads();
        if (tid == 0)
            dc::deflate_range(st, N, n1, jb, je, ds_s, zs_s, src_s, dlam, wz, indxp, coltyp, dcol, rot_p, rot_q, rot_c, rot_s);
        __syncthreads();
    }
    if (tid == 0) dc::deflate_finish(st, dlam, wz, indxp, coltyp, dcol);
    __syncthreads();
    __threadfence_block();
    const int K = st.K;
    // group the K kept columns by type 1,2,3 (stable), deflated after them in indxp order
    {
        const int chunk = (K + nt - 1) / nt;
        const int j0 = min(K, tid * chunk), j1 = min(K, j0 + chunk);
        int c[3] = {0, 0, 0};
        for (int j = j0; j < j1; ++j) c[coltyp[indxp[j]] - 1]++;
        cnt[tid][0] = c[0]; cnt[tid][1] = c[1]; cnt[tid][2] = c[2];
        __syncthreads();
        __shared__ int tot[3];
        if (tid < 3) {
            int run = 0;
            for (int t = 0; t < nt; ++t) { int v = cnt[t][tid]; cnt[t][tid] = run; run += v; }
            tot[tid] = run;
        }
        __syncthreads();
        int base[3] = {cnt[tid][0], tot[0] + cnt[tid][1], tot[0] + tot[1] + cnt[tid][2]};
        for (int j = j0; j < j1; ++j) {
            const int js = indxp[j], ct = coltyp[js] - 1;
            gcol[base[ct]] = js; gsec[base[ct]] = j; base[ct]++;
        }
        for (int j = K + tid; j < N; j += nt) gcol[j] = indxp[j];
        if (tid == 0) {
            DcOut o; o.K = K; o.c1 = tot[0]; o.c2 = tot[1]; o.c3 = tot[2]; o.nrot = st.nrot; o.pad = 0; o.rho = rho;
            b.out[(long)item * maxnodes + node] = o;
            // merge GEMMs:  Q[0:n1, 0:K] = Qw[0:n1, 0:c1+c2] S[0:c1+c2, 0:K] ;  Q[n1:N, 0:K] = Qw[n1:N, c1:K] S[c1:K, 0:K]
            double *Qwb = b.Qw + (long)item * n * n + off + (long)off * n;
            double *Sb = b.S + (long)item * n * n + off + (long)off * n;
            GemmDesc g;
            g.lda = n; g.ldb = n; g.ldc = b.ldq; g.sA = g.sB = g.sC = 0; g.opA = OP_N; g.opB = OP_N;
            g.maskA = g.maskB = MASK_NONE; g.offA = g.offB = 0; g.cmode = 0; g.conjC = 0; g.alpha = 1.0; g.beta = 0.0;
            g.scaleK = nullptr; g.sScale = 0; g.ksplit = 1; g.sSplit = 0;
            g.A = Qwb; g.B = Sb; g.C = Qb; g.m = n1; g.n = K; g.k = o.c1 + o.c2;
            b.desc[((long)item * nn + node) * 2] = g;
            g.A = Qwb + n1 + (long)o.c1 * n; g.B = Sb + o.c1; g.C = Qb + n1; g.m = n2; g.n = K; g.k = o.c2 + o.c3;
            b.desc[((long)item * nn + node) * 2 + 1] = g;
        }
    }
}

// ------------------------------------------------------------------------------------------------ rotations
__global__ void dc_rotate_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes) {
    const int node = blockIdx.y, item = blockIdx.z, n = b.n;
    const DcNode nd = nodes[node];
    const int N = nd.n1 + nd.n2;
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    const int nrot = b.out[(long)item * maxnodes + node].nrot;
    if (row >= N || nrot == 0) return;
    const long ib = (long)item * n + nd.off;
    double *Qb = b.Q + (long)item * b.sQ + nd.off + (long)nd.off * b.ldq;
    const int *rp = b.rot_p + ib, *rq = b.rot_q + ib;
    const double *rc = b.rot_c + ib, *rs = b.rot_s + ib;
    for (int r = 0; r < nrot; ++r) {
        const int p = rp[r], q = rq[r];
        const double c = rc[r], s = rs[r];
        const double x = Qb[row + (long)p * b.ldq], y = Qb[row + (long)q * b.ldq];
        Qb[row + (long)p * b.ldq] = c * x + s * y;
        Qb[row + (long)q * b.ldq] = c * y - s * x;
    }
}

// ------------------------------------------------------------------------------------------------ permute / copy back
__global__ void dc_permute_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int nodes_in_level) {
    const int node = blockIdx.z % nodes_in_level, item = blockIdx.z / nodes_in_level, n = b.n;
    const DcNode nd = nodes[node];
    const int N = nd.n1 + nd.n2;
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= N) return;
    const long ib = (long)item * n + nd.off;
    const double *Qb = b.Q + (long)item * b.sQ + nd.off + (long)nd.off * b.ldq;
    double *Qwb = b.Qw + (long)item * n * n + nd.off + (long)nd.off * n;
    const int *gcol = b.gcol + ib;
    const int K = b.out[(long)item * maxnodes + node].K;
    for (int g = blockIdx.y; g < N; g += gridDim.y) {
        const int c = gcol[g];
        Qwb[row + (long)g * n] = Qb[row + (long)c * b.ldq];
        if (row == 0 && g >= K) b.dnew[ib + g] = b.dcol[ib + c];
    }
}
__global__ void dc_copyback_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int nodes_in_level) {
    const int node = blockIdx.z % nodes_in_level, item = blockIdx.z / nodes_in_level, n = b.n;
    const DcNode nd = nodes[node];
    const int N = nd.n1 + nd.n2;
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= N) return;
    double *Qb = b.Q + (long)item * b.sQ + nd.off + (long)nd.off * b.ldq;
    const double *Qwb = b.Qw + (long)item * n * n + nd.off + (long)nd.off * n;
    const int K = b.out[(long)item * maxnodes + node].K;
    for (int g = K + blockIdx.y; g < N; g += gridDim.y) Qb[row + (long)g * b.ldq] = Qwb[row + (long)g * n];
}

// ------------------------------------------------------------------------------------------------ secular equation
__global__ void __launch_bounds__(256) dc_secular_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int *info) {
    const int node = blockIdx.y, item = blockIdx.z, n = b.n;
    const DcNode nd = nodes[node];
    const DcOut o = b.out[(long)item * maxnodes + node];
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (j >= o.K) return;
    const long ib = (long)item * n + nd.off;
    double *Qb = b.Q + (long)item * b.sQ + nd.off + (long)nd.off * b.ldq;
    WarpLanes L;
    double lam;
    dc::secular_root(L, o.K, j, b.dlam + ib, b.wz + ib, o.rho, Qb + (long)j * b.ldq, &lam);
    if ((threadIdx.x & 31) == 0) {
        b.dnew[ib + j] = lam;
        if (!isfinite(lam)) info[item] = n + 1;
    }
}

// zhat_i = sign(w_i) sqrt | prod_j (d_i - lambda_j) / prod_{j != i} (d_i - d_j) |
// 32 values of i per CTA (lanes, coalesced rows of Q), the j-range split over the 8 warps; the 8 partial products are
// multiplied in a fixed order
__global__ void __launch_bounds__(256) dc_zhat_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes) {
    __shared__ double part[8][32];
    const int node = blockIdx.y, item = blockIdx.z, n = b.n;
    const DcNode nd = nodes[node];
    const int K = b.out[(long)item * maxnodes + node].K;
    if ((int)blockIdx.x * 32 >= K) return;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int i = blockIdx.x * 32 + lane;
    const long ib = (long)item * n + nd.off;
    const double *Qb = b.Q + (long)item * b.sQ + nd.off + (long)nd.off * b.ldq;
    const double *dlam = b.dlam + ib;
    double p = 1.0;
    if (i < K) {
        const double di = dlam[i];
        const int jc = (K + 7) / 8, j0 = w * jc, j1 = min(K, j0 + jc);
        for (int j = j0; j < j1; ++j) {
            const double q = Qb[i + (long)j * b.ldq];
            p *= (j == i) ? q : q / (di - dlam[j]);
        }
    }
    part[w][lane] = p;
    __syncthreads();
    if (w == 0 && i < K) {
        double t = part[0][lane];
#pragma unroll
        for (int k = 1; k < 8; ++k) t *= part[k][lane];
        b.zhat[ib + i] = copysign(sqrt(fabs(t)), b.wz[ib + i]);
    }
}

// column j of S (grouped row order): s_i = zhat_i / (d_i - lambda_j), normalised
__global__ void __launch_bounds__(128) dc_vectors_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int restricted) {
    __shared__ double red[4];
    const int node = blockIdx.y, item = blockIdx.z, n = b.n;
    const DcNode nd = nodes[node];
    const int K = b.out[(long)item * maxnodes + node].K;
    const int j = blockIdx.x;
    if (j >= K) return;
    if (restricted && j >= b.kneed[item]) return;          // top merge, partial spectrum: unwanted columns are skipped
    const long ib = (long)item * n + nd.off;
    const double *dl = b.Q + (long)item * b.sQ + nd.off + (long)(nd.off + j) * b.ldq;
    double *Sc = b.S + (long)item * n * n + nd.off + (long)(nd.off + j) * n;
    const double *zh = b.zhat + ib;
    const int *gsec = b.gsec + ib;
    double s = 0.0;
    for (int i = threadIdx.x; i < K; i += blockDim.x) { const double t = zh[i] / dl[i]; s += t * t; }
    s = warp_sum(s);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    const double rn = 1.0 / sqrt(red[0] + red[1] + red[2] + red[3]);
    for (int g = threadIdx.x; g < K; g += blockDim.x) { const int i = gsec[g]; Sc[g] = zh[i] / dl[i] * rn; }
}

// ------------------------------------------------------------------------------------------------ finish a merge
__global__ void __launch_bounds__(256) dc_finish_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes) {
    const int node = blockIdx.x, item = blockIdx.y, n = b.n;
    const DcNode nd = nodes[node];
    const int N = nd.n1 + nd.n2;
    const int K = b.out[(long)item * maxnodes + node].K;
    const long ib = (long)item * n + nd.off;
    double *d = b.d + ib; const double *dnew = b.dnew + ib; int *idxq = b.idxq + ib;
    const int nb = N - K;
    // sorted order = merge of dnew[0:K) (ascending) with dnew[K:N) read backwards (ascending)
    for (int i = threadIdx.x; i < N; i += blockDim.x) {
        d[i] = dnew[i];
        if (i < K) {
            const double a = dnew[i];
            int lo = 0, hi = nb;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (dnew[N - 1 - mid] < a) lo = mid + 1; else hi = mid; }
            idxq[i + lo] = i;
        } else {
            const int ii = N - 1 - i;             // position in the ascending view of the deflated run
            const double bb = dnew[i];
            int lo = 0, hi = K;
            while (lo < hi) { int mid = (lo + hi) >> 1; if (dnew[mid] <= bb) lo = mid + 1; else hi = mid; }
            idxq[ii + lo] = i;
        }
    }
}

// Top merge with only the nvec lowest eigenpairs wanted: the secular roots dnew[0:K) are ascending, so the
// wanted ones are a prefix; its length (sorted position of root i = i + #{deflated values below it} < nvec) becomes the
// column count of the two merge GEMMs.  Runs after dc_finish_kernel-style ranking data (dnew) is complete.
__global__ void __launch_bounds__(256) dc_restrict_kernel(DcBuf b, const DcNode *__restrict__ nodes, int maxnodes, int nvec) {
    __shared__ int red[8];
    const int item = blockIdx.x, n = b.n;
    const DcNode nd = nodes[0];
    const int N = nd.n1 + nd.n2;
    const int K = b.out[(long)item * maxnodes].K;
    const double *dnew = b.dnew + (long)item * n + nd.off;
    const int nb = N - K;
    int cnt = 0;
    for (int i = threadIdx.x; i < K; i += blockDim.x) {
        const double a = dnew[i];
        int lo = 0, hi = nb;
        while (lo < hi) { int mid = (lo + hi) >> 1; if (dnew[N - 1 - mid] < a) lo = mid + 1; else hi = mid; }
        if (i + lo < nvec) ++cnt;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += red[w];
        b.kneed[item] = t;
        b.desc[(long)item * 2].n = t;
        b.desc[(long)item * 2 + 1].n = t;
    }
}

// eigenvalues (rescaled) in ascending order ...
__global__ void dc_final_evals_kernel(DcBuf b, double *evals) {
    const int item = blockIdx.y, n = b.n;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n) return;
    evals[(long)item * n + c] = b.scale[item] * b.d[(long)item * n + b.idxq[(long)item * n + c]];
}
// ... and the matching permutation of the first ncols eigenvector columns
__global__ void dc_final_kernel(DcBuf b, double *Qout, long ldo, long sO, int ncols) {
    const int item = blockIdx.z, n = b.n;
    const int row = blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= n) return;
    const double *Q = b.Q + (long)item * b.sQ;
    double *Qo = Qout + (long)item * sO;
    const int *idxq = b.idxq + (long)item * n;
    for (int c = blockIdx.y; c < ncols; c += gridDim.y) Qo[row + (long)c * ldo] = Q[row + (long)idxq[c] * b.ldq];
}

// Tree of the divide step, written by the device (mirrors dc_plan): a complete binary tree of `depth` levels in which a
// node of size s splits into s/2 and s - s/2.  leaf_off[0..2^depth], cuts[i-1] = leaf_off[i] (1 <= i < 2^depth), and the
// merge nodes level by level, bottom-up (level lv holds 2^(depth-1-lv) nodes).
__device__ __forceinline__ void dc_descend(int n, int steps, int q, int &off, int &s) {
    off = 0; s = n;
    for (int lev = steps - 1; lev >= 0; --lev) {
        const int h = s / 2;
        if ((q >> lev) & 1) { off += h; s -= h; } else s = h;
    }
}
__global__ void dc_tree_kernel(int n, int depth, int *leaf_off, int *cuts, DcNode *nodes) {
    const int nleaves = 1 << depth;
    for (int q = threadIdx.x; q <= nleaves; q += blockDim.x) {
        int off = n, s = 0;
        if (q < nleaves) dc_descend(n, depth, q, off, s);
        leaf_off[q] = off;
        if (q >= 1 && q < nleaves) cuts[q - 1] = off;
    }
    int base = 0;
    for (int lv = 0; lv < depth; ++lv) {
        const int nn = 1 << (depth - 1 - lv);
        for (int q = threadIdx.x; q < nn; q += blockDim.x) {
            int off, s;
            dc_descend(n, depth - 1 - lv, q, off, s);
            nodes[base + q] = DcNode{off, s / 2, s - s / 2};
        }
        base += nn;
    }
}

// ------------------------------------------------------------------------------------------------ host driver
struct DcPlan {
    std::vector<int> leaf_off;                       // nleaves + 1
    std::vector<std::vector<DcNode>> levels;         // bottom-up
    int maxnodes;
};

static DcPlan dc_plan(int n) {
    DcPlan p;
    std::vector<int> sizes{n};
    for (;;) {
        int mx = 0; for (int s : sizes) mx = s > mx ? s : mx;
        if (mx <= DC_LEAF) break;
        std::vector<int> s2;
        for (int s : sizes) { s2.push_back(s / 2); s2.push_back(s - s / 2); }
        sizes.swap(s2);
    }
    p.leaf_off.assign(sizes.size() + 1, 0);
    for (size_t i = 0; i < sizes.size(); ++i) p.leaf_off[i + 1] = p.leaf_off[i] + sizes[i];
    std::vector<int> cs = sizes, co(p.leaf_off.begin(), p.leaf_off.end() - 1);
    p.maxnodes = 1;
    while (cs.size() > 1) {
        std::vector<DcNode> lvl; std::vector<int> ns, no;
        for (size_t q = 0; q < cs.size(); q += 2) {
            lvl.push_back(DcNode{co[q], cs[q], cs[q + 1]});
            ns.push_back(cs[q] + cs[q + 1]); no.push_back(co[q]);
        }
        if ((int)lvl.size() > p.maxnodes) p.maxnodes = (int)lvl.size();
        p.levels.push_back(lvl);
        cs.swap(ns); co.swap(no);
    }
    return p;
}

struct DcWork { DcBuf b; int *cuts; int *leaf_off; DcNode *nodes; size_t bytes; };
static DcWork dc_carve(int n, int batch, const DcPlan &p, void *work) {
    DcWork w; Arena ar(work, (size_t)-1);
    const size_t bn = (size_t)batch * n;
    w.b.n = n;
    w.b.Q = ar.get<double>(bn * n); w.b.ldq = n; w.b.sQ = (long)n * n;
    w.b.Qw = ar.get<double>(bn * n); w.b.S = ar.get<double>(bn * n);
    double **dp[] = {&w.b.z, &w.b.dlam, &w.b.wz, &w.b.dcol, &w.b.dnew, &w.b.zhat, &w.b.rot_c, &w.b.rot_s, &w.b.ds, &w.b.zs};
    for (auto q : dp) *q = ar.get<double>(bn);
    w.b.scale = ar.get<double>(batch);
    int **ip[] = {&w.b.idxq, &w.b.src, &w.b.indxp, &w.b.coltyp, &w.b.gcol, &w.b.gsec, &w.b.rot_p, &w.b.rot_q};
    for (auto q : ip) *q = ar.get<int>(bn);
    w.b.kneed = ar.get<int>(batch);
    w.b.out = ar.get<DcOut>((size_t)batch * p.maxnodes);
    w.b.desc = ar.get<GemmDesc>((size_t)batch * p.maxnodes * 2);
    size_t nnodes = 0; for (auto &l : p.levels) nnodes += l.size();
    w.cuts = ar.get<int>(p.leaf_off.size());
    w.leaf_off = ar.get<int>(p.leaf_off.size());
    w.nodes = ar.get<DcNode>(nnodes + 1);
    w.bytes = ar.off;
    return w;
}
size_t stedc_workspace(int n, int batch) { DcPlan p = dc_plan(n); return dc_carve(n, batch, p, nullptr).bytes; }

// phase bit 0: everything up to the eigenvalues (all levels; of the top merge: deflation, secular equation, ranking);
// phase bit 1: eigenvectors of the top merge -- only the columns that end up among the nvec lowest -- and the sorted copy of
// the first nvec columns into Qout.  A phase-2 call continues a phase-1 call on the same workspace.
int stedc(int n, int batch, double *d, double *e, double *evals, double *Qout, long ldq, long sQ, void *work, int *d_info,
          cudaStream_t st, int nvec, int phase) {
    if (nvec < 0 || nvec > n) nvec = n;
    DcPlan p = dc_plan(n);
    DcWork w = dc_carve(n, batch, p, work);
    w.b.d = d; w.b.e = e;
    const int nleaves = (int)p.leaf_off.size() - 1;
    std::vector<size_t> lvl_off;
    { size_t o = 0; for (auto &l : p.levels) { lvl_off.push_back(o); o += l.size(); } }
    const size_t nlev = p.levels.size();
    auto level_geometry = [&](size_t lv, int &nn, int &Nmax, int &hmax) {
        nn = (int)p.levels[lv].size(); Nmax = 0; hmax = 0;
        for (auto &nd : p.levels[lv]) { Nmax = max(Nmax, nd.n1 + nd.n2); hmax = max(hmax, max(nd.n1, nd.n2)); }
    };
    if (phase & 1) {
        // tree description (leaf offsets, tear points, merge nodes of every level) built on the device: no host copy, so the
        // call only enqueues work
        dc_tree_kernel<<<1, 256, 0, st>>>(n, (int)nlev, w.leaf_off, w.cuts, w.nodes);
        NAO_LAUNCHED();
        const int ncuts = nleaves - 1;

        NAO_CUDA_CHECK(cudaMemsetAsync(w.b.Q, 0, (size_t)batch * n * n * 8, st));
        dc_scale_tear_kernel<<<batch, 256, 0, st>>>(w.b, w.cuts, ncuts);
        NAO_LAUNCHED();
        dc_leaf_kernel<<<dim3(ceil_div(nleaves, 4), batch), 128, 0, st>>>(w.b, w.leaf_off, nleaves, d_info);
        NAO_LAUNCHED();
        for (size_t lv = 0; lv < nlev; ++lv) {
            int nn, Nmax, hmax; level_geometry(lv, nn, Nmax, hmax);
            const DcNode *nodes = w.nodes + lvl_off[lv];
            const bool top = (lv + 1 == nlev);
            dc_setup_kernel<<<dim3(nn, batch), 1024, 0, st>>>(w.b, nodes, p.maxnodes, nn);
            NAO_LAUNCHED();
            dc_rotate_kernel<<<dim3(ceil_div(Nmax, 256), nn, batch), 256, 0, st>>>(w.b, nodes, p.maxnodes);
            NAO_LAUNCHED();
            const int cy = min(Nmax, 1024);
            dc_permute_kernel<<<dim3(ceil_div(Nmax, 256), cy, nn * batch), 256, 0, st>>>(w.b, nodes, p.maxnodes, nn);
            NAO_LAUNCHED();
            dc_copyback_kernel<<<dim3(ceil_div(Nmax, 256), cy, nn * batch), 256, 0, st>>>(w.b, nodes, p.maxnodes, nn);
            NAO_LAUNCHED();
            dc_secular_kernel<<<dim3(ceil_div(Nmax, 8), nn, batch), 256, 0, st>>>(w.b, nodes, p.maxnodes, d_info);
            NAO_LAUNCHED();
            dc_zhat_kernel<<<dim3(ceil_div(Nmax, 32), nn, batch), 256, 0, st>>>(w.b, nodes, p.maxnodes);
            NAO_LAUNCHED();
            if (!top) {
                dc_vectors_kernel<<<dim3(Nmax, nn, batch), 128, 0, st>>>(w.b, nodes, p.maxnodes, 0);
                NAO_LAUNCHED();
                if (int rc = gemm_launch_grouped(NAO_REAL, w.b.desc, batch * nn * 2, hmax, Nmax, 1, OP_N, OP_N, false, st)) return rc;
            }
            dc_finish_kernel<<<dim3(nn, batch), 256, 0, st>>>(w.b, nodes, p.maxnodes);      // eigenvalue order of the merged node
            NAO_LAUNCHED();
        }
        dc_final_evals_kernel<<<dim3(ceil_div(n, 256), batch), 256, 0, st>>>(w.b, evals);
        NAO_LAUNCHED();
    }
    if (phase & 2) {
        if (nlev > 0) {
            int nn, Nmax, hmax; level_geometry(nlev - 1, nn, Nmax, hmax);
            const DcNode *nodes = w.nodes + lvl_off[nlev - 1];
            const int restricted = nvec < n ? 1 : 0;
            if (restricted) {
                dc_restrict_kernel<<<batch, 256, 0, st>>>(w.b, nodes, p.maxnodes, nvec);
                NAO_LAUNCHED();
            }
            dc_vectors_kernel<<<dim3(Nmax, nn, batch), 128, 0, st>>>(w.b, nodes, p.maxnodes, restricted);
            NAO_LAUNCHED();
            if (int rc = gemm_launch_grouped(NAO_REAL, w.b.desc, batch * nn * 2, hmax, Nmax, 1, OP_N, OP_N, false, st)) return rc;
        }
        dc_final_kernel<<<dim3(ceil_div(n, 256), min(nvec, 1024), batch), 256, 0, st>>>(w.b, Qout, ldq, sQ, nvec);
        NAO_LAUNCHED();
    }
    NAO_CUDA_CHECK(cudaGetLastError());
    return NAO_OK;
}

}  // namespace nao

NAO_EXPORT int nao_stedc_workspace(int n, int batch, size_t *bytes) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!bytes) return -3;
    *bytes = nao::stedc_workspace(n, batch);
    return NAO_OK;
}
NAO_EXPORT int nao_stedc(int n, int batch, double *dD, double *dEoff, double *dE, double *dQ, long ldq, long strideQ,
                         void *dwork, size_t work_bytes, int *d_info, void *cuda_stream) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!dD) return -3;
    if (!dEoff) return -4;
    if (!dE) return -5;
    if (!dQ) return -6;
    if (ldq < n) return -7;
    if (batch > 1 && strideQ < ldq * (long)n) return -8;
    if (!dwork) return -9;
    if (work_bytes < nao::stedc_workspace(n, batch)) return NAO_ERR_WORKSPACE;
    if (!d_info) return -11;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaMemsetAsync(d_info, 0, sizeof(int) * batch, st) != cudaSuccess) return NAO_ERR_CUDA;
    return nao::stedc(n, batch, dD, dEoff, dE, dQ, ldq, strideQ, dwork, d_info, st);
}
