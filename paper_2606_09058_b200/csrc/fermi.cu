// fermi.cu -- Fermi level and occupations (Fermi-Dirac f_i: PAPER.md:42; reading C5).
//
//   N(mu) = sum_j w_j f_j,  f_j = 1/(1+exp((e_j-mu)/kT)),  strictly increasing in mu.  Root of N(mu) = N_e.
// Solved in particle/hole form so that mu is resolved inside a gap: with the states sorted by energy and m the
// largest count whose cumulated weight W_m <= N_e, r = N_e - W_m,
//   G(mu) = sum_{j>=m} w_j f_j - sum_{j<m} w_j (1-f_j) - r        ( == N(mu) - N_e identically ),
// and when r == 0 the sign of G is taken from log P - log Q with log f = -softplus(x), log(1-f) = -softplus(-x)
// (log-sum-exp: no cancellation, no underflow).  Plain ALU/SFU work on at most a few 10^4 states:
//   1. rank sort (each state counts the states before it; ns^2 compares spread over the grid),
//   2. one CTA: inclusive scan for m, then bisection on [e_min - 50 kT, e_max + 50 kT] until the interval cannot shrink,
//   3. occupations for all states.
#include "nao_internal.cuh"

namespace nao {

__device__ __forceinline__ double softplus(double x) { return x > 0 ? x + log1p(exp(-x)) : log1p(exp(x)); }

// rank[j] = number of states that sort before state j (ties broken by index); scatter into sorted arrays
__global__ void fermi_rank_kernel(int ns, int n, const double *__restrict__ e, const double *__restrict__ wItem,
                                  double *__restrict__ es, double *__restrict__ ws) {
    __shared__ double tile[1024];
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    double ej = j < ns ? e[j] : 0.0;
    int rank = 0;
    for (int base = 0; base < ns; base += 1024) {
        for (int t = threadIdx.x; t < 1024; t += blockDim.x) tile[t] = (base + t < ns) ? e[base + t] : 0.0;
        __syncthreads();
        int lim = min(1024, ns - base);
        if (j < ns)
            for (int t = 0; t < lim; ++t) {
                double o = tile[t];
                rank += (o < ej) || (o == ej && base + t < j);
            }
        __syncthreads();
    }
    if (j < ns) { es[rank] = ej; ws[rank] = wItem[j / n]; }
}

// Block-wide sum / max with ONE block barrier per call: butterfly inside the warp, one partial per warp into one of two
// alternating buffers, every thread adds the (at most 32) partials in index order.  Fixed order: deterministic.
struct BlockSum {
    double *buf;     // 2 x 32 doubles of shared memory
    int flip;
    __device__ double sum(double v) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        double *b = buf + 32 * flip; flip ^= 1;
        if ((threadIdx.x & 31) == 0) b[threadIdx.x >> 5] = v;
        __syncthreads();
        double s = 0.0;
        const int nw = (blockDim.x + 31) >> 5;
        for (int w = 0; w < nw; ++w) s += b[w];
        return s;
    }
    __device__ double max(double v) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        double *b = buf + 32 * flip; flip ^= 1;
        if ((threadIdx.x & 31) == 0) b[threadIdx.x >> 5] = v;
        __syncthreads();
        double s = -INFINITY;
        const int nw = (blockDim.x + 31) >> 5;
        for (int w = 0; w < nw; ++w) s = fmax(s, b[w]);
        return s;
    }
};

// one CTA of 1024 threads.  Each thread owns a CONTIGUOUS chunk of the sorted states so that partial sums are
// formed in sorted order (deterministic).
__global__ void __launch_bounds__(1024) fermi_bisect_kernel(int ns, const double *__restrict__ es,
                                                             const double *__restrict__ ws, double n_electrons,
                                                             double kT, double *__restrict__ mu_out, int cache) {
    extern __shared__ double s_tj[];          // ns doubles when cache != 0
    __shared__ double red[1024];
    __shared__ int s_m;
    __shared__ double s_W;
    __shared__ double red2[4 * 32];
    BlockSum bs{red2, 0};
    const int tid = threadIdx.x, nt = blockDim.x;
    const int chunk = (ns + nt - 1) / nt;
    const int j0 = min(ns, tid * chunk), j1 = min(ns, j0 + chunk);

    // --- split index m: largest count with W_m <= N_e (sequential semantics of the definition, done as a scan)
    double local = 0.0;
    for (int j = j0; j < j1; ++j) local += ws[j];
    __syncthreads();
    red[tid] = local;
    __syncthreads();
    if (tid == 0) {                       // exclusive prefix over the 1024 chunk sums, in order
        double run = 0.0;
        for (int t = 0; t < nt; ++t) { double v = red[t]; red[t] = run; run += v; }
        s_m = 0; s_W = 0.0;
    }
    __syncthreads();
    {
        // thread whose chunk contains the crossing decides m
        double W = red[tid];
        int m_local = -1; double W_local = 0.0;
        // the sequential rule "take states while W + w <= N_e" stops at the FIRST failure; with positive weights
        // the cumulated weight is monotone, so the first failure is where the running sum first exceeds N_e.
        for (int j = j0; j < j1; ++j) {
            if (W + ws[j] <= n_electrons) { W += ws[j]; }
            else { m_local = j; W_local = W; break; }
        }
        __syncthreads();
        red[tid] = (m_local >= 0) ? (double)m_local : (double)ns + 1.0;
        __syncthreads();
        // first failing index over all threads = min; but a thread only sees a valid failure if its prefix fit,
        // which holds for every thread up to and including the first failing one (monotone sums).
        for (int s = nt >> 1; s > 0; s >>= 1) {
            if (tid < s) red[tid] = fmin(red[tid], red[tid + s]);
            __syncthreads();
        }
        double mmin = red[0];
        __syncthreads();
        if (m_local >= 0 && (double)m_local == mmin) { s_m = m_local; s_W = W_local; }
        if (mmin > (double)ns && tid == nt - 1) { s_m = ns; s_W = W; }   // never happens for valid N_e
        __syncthreads();
    }
    const int m = s_m;
    const double r = n_electrons - s_W;
    double lo = es[0] - 50.0 * kT, hi = es[ns - 1] + 50.0 * kT;
    const bool logform = (r == 0.0 && m > 0);
    // States far from mu cost nothing: the bisection would otherwise spend three FP64 transcendentals per state and step on one
    // SM.  XCUT = 100: exp(-100) = 3.7e-44.  Plain form: for x < -XCUT the occupation is 1 to that accuracy (the sum gets w
    // itself, which is also what the full expression rounds to), for x > XCUT the term is below 3.7e-44 w and is dropped.
    // Log form: a term is dropped when it is more than e^-100 below the term of the state next to the split on its side,
    // which the sorted order makes the largest up to the weight ratio (lw = log(w_max / w_min)).
    // The states that are left lie next to one another in the sorted order, so inside the bisection the states are dealt
    // round-robin (thread t takes t, t + 1024, ...) instead of in the contiguous chunks of the scan above: the few hundred
    // live states then cost one or two evaluations per thread, not 13 in a handful of threads.  Still a fixed order.
    const double XCUT = 100.0;
    double lw = 0.0;
    if (logform) {
        double wmx = 0.0, wmn = -INFINITY;
        for (int j = tid; j < ns; j += nt) { wmx = fmax(wmx, ws[j]); wmn = fmax(wmn, -ws[j]); }
        wmx = bs.max(wmx); wmn = -bs.max(wmn);
        lw = log(wmx / wmn);
    }

    for (int it = 0; it < 400; ++it) {
        double mu = 0.5 * (lo + hi);
        if (!(mu > lo && mu < hi)) break;
        bool positive;
        if (logform) {
            // t_j = log w_j + log f_j (j >= m) or log w_j + log(1 - f_j) (j < m); kept in shared memory between the two passes
            // when the states fit there (cache != 0)
            const double cutP = (m < ns ? fmax((es[m] - mu) / kT, 0.0) : 0.0) + XCUT + 1.0 + lw;
            const double cutQ = fmax((mu - es[m - 1]) / kT, 0.0) + XCUT + 1.0 + lw;
            double mp = -INFINITY, mq = -INFINITY;
            for (int j = tid; j < ns; j += nt) {
                const double xs = (j >= m) ? (es[j] - mu) / kT : (mu - es[j]) / kT;
                double t = -INFINITY;
                if (fmax(xs, 0.0) <= (j >= m ? cutP : cutQ)) t = log(ws[j]) - softplus(xs);
                if (cache) s_tj[j] = t;
                if (j >= m) mp = fmax(mp, t); else mq = fmax(mq, t);
            }
            mp = bs.max(mp); mq = bs.max(mq);
            double sp = 0.0, sq = 0.0;
            for (int j = tid; j < ns; j += nt) {
                double t;
                if (cache) t = s_tj[j];
                else {
                    const double xs = (j >= m) ? (es[j] - mu) / kT : (mu - es[j]) / kT;
                    t = (fmax(xs, 0.0) <= (j >= m ? cutP : cutQ)) ? log(ws[j]) - softplus(xs) : -INFINITY;
                }
                if (t == -INFINITY) continue;
                if (j >= m) sp += exp(t - mp); else sq += exp(t - mq);
            }
            sp = bs.sum(sp); sq = bs.sum(sq);
            positive = (mp + log(sp)) > (mq + log(sq));
        } else {
            double P = 0.0, Q = 0.0;
            for (int j = tid; j < ns; j += nt) {
                const double x = (es[j] - mu) / kT;
                if (j >= m) {
                    if (x > XCUT) continue;
                    P += (x < -XCUT) ? ws[j] : ws[j] * exp(-softplus(x));
                } else {
                    if (x < -XCUT) continue;
                    Q += (x > XCUT) ? ws[j] : ws[j] * exp(-softplus(-x));
                }
            }
            P = bs.sum(P); Q = bs.sum(Q);
            positive = (P - Q - r) > 0.0;
        }
        if (positive) hi = mu; else lo = mu;
    }
    if (tid == 0) *mu_out = 0.5 * (lo + hi);
}

__global__ void fermi_occ_kernel(int ns, const double *__restrict__ e, const double *__restrict__ mu, double kT,
                                 double *__restrict__ f) {
    int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < ns) f[j] = exp(-softplus((e[j] - *mu) / kT));
}

int fermi_mu(int n, int batch, const double *dE, const double *h_weight, double n_electrons, double kT, double *h_mu,
             double *dF, void *dwork, cudaStream_t st) {
    const int ns = n * batch;
    Arena ar(dwork, (size_t)-1);
    double *es = ar.get<double>(ns), *ws = ar.get<double>(ns), *wItem = ar.get<double>(batch), *mu = ar.get<double>(1);
    NAO_CUDA_CHECK(cudaMemcpyAsync(wItem, h_weight, sizeof(double) * batch, cudaMemcpyHostToDevice, st));
    fermi_rank_kernel<<<ceil_div(ns, 256), 256, 0, st>>>(ns, n, dE, wItem, es, ws);
    NAO_LAUNCHED();
    {
        const size_t tbytes = (size_t)ns * 8;
        const int cache = tbytes <= 200 * 1024 ? 1 : 0;
        static bool attr = false;
        if (!attr) {
            NAO_CUDA_CHECK(cudaFuncSetAttribute(fermi_bisect_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
            attr = true;
        }
        fermi_bisect_kernel<<<1, 1024, cache ? tbytes : 0, st>>>(ns, es, ws, n_electrons, kT, mu, cache);
    }
    NAO_LAUNCHED();
    fermi_occ_kernel<<<ceil_div(ns, 256), 256, 0, st>>>(ns, dE, mu, kT, dF);
    NAO_LAUNCHED();
    NAO_CUDA_CHECK(cudaGetLastError());
    NAO_CUDA_CHECK(cudaMemcpyAsync(h_mu, mu, sizeof(double), cudaMemcpyDeviceToHost, st));
    NAO_CUDA_CHECK(cudaStreamSynchronize(st));
    return NAO_OK;
}

}  // namespace nao

NAO_EXPORT int nao_fermi_workspace(int n, int batch, size_t *bytes) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!bytes) return -3;
    size_t ns = (size_t)n * batch;
    *bytes = 2 * nao::align_up(ns * 8) + nao::align_up((size_t)batch * 8) + 256;
    return NAO_OK;
}

NAO_EXPORT int nao_fermi_mu(int n, int batch, const double *dE, const double *h_weight, double n_electrons, double kT,
                            double *h_mu, double *dF, void *dwork, void *cuda_stream) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!dE) return -3;
    if (!h_weight) return -4;
    if (!h_mu) return -7;
    if (!dF) return -8;
    if (!dwork) return -9;
    if (int rc = nao::check_occupation_args(n, batch, h_weight, n_electrons, kT, 4)) return rc;
    if (int rcb = nao::bind_device()) return rcb;
    return nao::fermi_mu(n, batch, dE, h_weight, n_electrons, kT, h_mu, dF, dwork, (cudaStream_t)cuda_stream);
}

// ---------------------------------------------------------------------------------------------------------------------
// nao_fermi_mu_static: the Fermi-level search for callers that have no device workspace to hand over (include/nao.h).
//
// The sorted energies, their weights, the per-item weights and the device copy of mu -- everything nao_fermi_mu keeps in
// the caller's `dwork` -- live in the file-scope array below instead.  It is part of the library image: every GPU on
// which this library's kernels are loaded carries its NAO_FERMI_STATIC_BYTES (1.5 MiB) until the process ends, whether
// or not this entry point is ever called.  Nothing in the array has to start at zero: each word a kernel reads was
// written earlier in the same call (the rank sort scatters a permutation of all ns sorted slots), so what the previous
// call left behind is harmless -- and calls that are on the GPU at the same time (two streams, two host threads) share
// these bytes and race.
//
// In host code `g_fermi_static` is only a handle for the runtime, not an address the GPU understands; the device address
// is asked for once per device (cudaGetSymbolAddress, with that device current) and remembered.
// ---------------------------------------------------------------------------------------------------------------------
namespace nao {

static __device__ __align__(256) unsigned char g_fermi_static[NAO_FERMI_STATIC_BYTES];

enum { FERMI_STATIC_MAX_DEVICES = 64 };
static void *g_fermi_static_addr[FERMI_STATIC_MAX_DEVICES] = {};   // device address of the array, per device ordinal

// device address of g_fermi_static on the CURRENT device (looked up on the first call made with that device current)
static int fermi_static_scratch(void **out) {
    int dev = -1;
    NAO_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= FERMI_STATIC_MAX_DEVICES) return NAO_ERR_UNSUPPORTED;
    if (!g_fermi_static_addr[dev]) {
        void *p = nullptr;
        NAO_CUDA_CHECK(cudaGetSymbolAddress(&p, g_fermi_static));
        if (!p) return NAO_ERR_CUDA;
        g_fermi_static_addr[dev] = p;
    }
    *out = g_fermi_static_addr[dev];
    return NAO_OK;
}

}  // namespace nao

NAO_EXPORT int nao_fermi_mu_static(int n, int batch, const double *dE, const double *h_weight, double n_electrons,
                                   double kT, double *h_mu, double *dF, void *cuda_stream) {
    if (n < 1) return -1;
    if (batch < 1) return -2;
    if (!dE) return -3;
    if (!h_weight) return -4;
    if (!h_mu) return -7;
    if (!dF) return -8;
    // the limit is on the number of states, checked before anything touches the device
    if ((long)n * (long)batch > (long)NAO_FERMI_STATIC_MAX_STATES) return NAO_ERR_STATIC_LIMIT;
    size_t need = 0;
    if (nao_fermi_workspace(n, batch, &need) != NAO_OK || need > (size_t)NAO_FERMI_STATIC_BYTES) return NAO_ERR_STATIC_LIMIT;
    if (int rc = nao::check_occupation_args(n, batch, h_weight, n_electrons, kT, 4)) return rc;
    if (int rc = nao::bind_device()) return rc;
    void *scratch = nullptr;
    if (int rc = nao::fermi_static_scratch(&scratch)) return rc;
    return nao::fermi_mu(n, batch, dE, h_weight, n_electrons, kT, h_mu, dF, scratch, (cudaStream_t)cuda_stream);
}
