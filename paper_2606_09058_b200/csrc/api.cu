// api.cu -- status strings, version, launch counter (C-ABI).
#include "nao_internal.cuh"


NAO_EXPORT const char *nao_status_string(int status) {
    switch (status) {
        case NAO_OK: return "ok";
        case NAO_ERR_WORKSPACE: return "workspace too small";
        case NAO_ERR_CUDA: return "CUDA runtime or launch error";
        case NAO_ERR_ELECTRONS: return "n_electrons outside (0, sum of weights * n) or kT <= 0";
        case NAO_ERR_UNSUPPORTED: return "unsupported combination of arguments";
        case NAO_ERR_STATIC_LIMIT: return "n * batch exceeds NAO_FERMI_STATIC_MAX_STATES (65536): the built-in scratch of nao_fermi_mu_static is too small, use nao_fermi_mu with a workspace";
        default: return status < 0 ? "invalid argument (index = -status)" : "unknown status";
    }
}
NAO_EXPORT const char *nao_version(void) { return "nao-b200 0.1 (sm_100a)"; }
NAO_EXPORT long nao_launch_count(void) { return nao::g_launch_count; }

namespace nao {
static int g_sm_limit = 0;
void set_sm_limit(int limit) { g_sm_limit = limit > 0 ? limit : 0; }
// The process-wide state (side streams, events, kernel attributes, pinned words) lives on ONE device: the one that is
// current at the first call that launches.  Later calls made with another device current are refused instead of using that
// state across devices.
static int g_bound_dev = -1, g_bound_sms = 0;
int bind_device() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return NAO_ERR_CUDA;
    if (g_bound_dev < 0) {
        int nsm = 0;
        if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm <= 0) return NAO_ERR_CUDA;
        g_bound_dev = dev; g_bound_sms = nsm;
    }
    return dev == g_bound_dev ? NAO_OK : NAO_ERR_CUDA;
}
int device_sms() {
    if (g_bound_dev < 0 && bind_device() != NAO_OK) return 148;
    return g_bound_sms;
}
int sm_count() {
    const int nsm = device_sms();
    return (g_sm_limit > 0 && g_sm_limit < nsm) ? g_sm_limit : nsm;
}
// Streams and events are created into locals and published only when every one of them exists.
int side_set_init(SideSet &out, int nstreams, int nevents, bool high_priority) {
    if (out.ready) return NAO_OK;
    if (nstreams > SideSet::MAX_STREAMS || nevents > SideSet::MAX_EVENTS) return NAO_ERR_UNSUPPORTED;
    SideSet tmp = {};
    int prio_lo = 0, prio_hi = 0;
    bool ok = true;
    if (high_priority) ok = cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi) == cudaSuccess;
    int ns = 0, ne = 0;
    for (; ok && ns < nstreams; ++ns)
        ok = (high_priority ? cudaStreamCreateWithPriority(&tmp.stream[ns], cudaStreamNonBlocking, prio_hi)
                            : cudaStreamCreateWithFlags(&tmp.stream[ns], cudaStreamNonBlocking)) == cudaSuccess;
    for (; ok && ne < nevents; ++ne) ok = cudaEventCreateWithFlags(&tmp.event[ne], cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        for (int i = 0; i < SideSet::MAX_STREAMS; ++i) if (tmp.stream[i]) cudaStreamDestroy(tmp.stream[i]);
        for (int i = 0; i < SideSet::MAX_EVENTS; ++i) if (tmp.event[i]) cudaEventDestroy(tmp.event[i]);
        return NAO_ERR_CUDA;
    }
    tmp.ready = true;
    out = tmp;
    return NAO_OK;
}
}  // namespace nao

// ---- optional phase timing (CUDA events recorded on the caller's stream at phase boundaries of nao_geneig) ----
namespace nao {
static const int NPH = 9;
static const char *kPhaseNames[NPH - 1] = {"potrf_trtri", "reduce_WHWh", "tridiagonalise", "band_to_tridiagonal", "stedc", "back_transform_band", "back_transform", "C_WhZ"};
static bool g_prof_on = false;
// While nao_geneig runs its batch as stream groups the launches go to internal streams: events recorded there would time
// nothing meaningful, so the grouped call records nothing (the timers keep what earlier ungrouped calls recorded).
static bool g_prof_suspended = false;
void prof_suspend(bool on) { g_prof_suspended = on; }
static inline bool prof_active() { return g_prof_on && !g_prof_suspended; }
static cudaEvent_t g_ev[NPH];
static bool g_ev_made = false, g_ev_rec[NPH];
void prof_mark(int idx, cudaStream_t st) {
    if (!prof_active() || idx < 0 || idx >= NPH) return;
    if (!g_ev_made) { for (int i = 0; i < NPH; ++i) cudaEventCreate(&g_ev[i]); g_ev_made = true; }
    if (idx == 0) for (int i = 0; i < NPH; ++i) g_ev_rec[i] = false;
    cudaEventRecord(g_ev[idx], st); g_ev_rec[idx] = true;
}
}  // namespace nao
namespace nao {
// per-kernel-class timers: pairs of events around individual launches (only while profiling is enabled)
static const int NSLOT = 2, SLOT_CAP = 2048;
static const char *kSlotNames[NSLOT] = {"hetrd_panel_kernel", "gemm_kernel"};
static cudaEvent_t g_sev[NSLOT][SLOT_CAP][2];
static int g_scount[NSLOT] = {0, 0}, g_smade[NSLOT] = {0, 0};
static double g_swork[NSLOT] = {0.0, 0.0};
int prof_kernel_begin(int slot, double work, cudaStream_t st) {
    if (!prof_active() || slot < 0 || slot >= NSLOT || g_scount[slot] >= SLOT_CAP) return -1;
    int k = g_scount[slot];
    if (k >= g_smade[slot]) { cudaEventCreate(&g_sev[slot][k][0]); cudaEventCreate(&g_sev[slot][k][1]); g_smade[slot] = k + 1; }
    cudaEventRecord(g_sev[slot][k][0], st);
    g_swork[slot] += work;
    return k;
}
// Flops of grouped launches: their dimensions are written by kernels (deflated sizes of the D&C merges), so the count is
// summed on the device from the descriptors, behind the launch, while profiling is enabled.
__device__ double g_grouped_flops;
__global__ void grouped_flops_kernel(const GemmDesc *d, int ngroups, double per_mnk) {
    double s = 0.0;
    for (int g = threadIdx.x; g < ngroups; g += blockDim.x)
        if (d[g].m > 0 && d[g].n > 0 && d[g].k > 0)
            s += per_mnk * d[g].m * (double)d[g].n * d[g].k * (d[g].cmode != 0 ? 0.5 : 1.0) *
                 ((d[g].maskA != MASK_NONE || d[g].maskB != MASK_NONE) ? 0.5 : 1.0);
    // one warp, fixed order, one plain add: launches on a stream are ordered, so the total does not depend on timing
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (threadIdx.x == 0 && s != 0.0) g_grouped_flops += s;
}
void prof_grouped_flops(const GemmDesc *d_descs, int ngroups, double per_mnk, cudaStream_t st) {
    if (!prof_active() || !d_descs || ngroups <= 0) return;
    grouped_flops_kernel<<<1, 32, 0, st>>>(d_descs, ngroups, per_mnk);
}
void prof_kernel_end(int slot, int k, cudaStream_t st) {
    if (k < 0) return;
    cudaEventRecord(g_sev[slot][k][1], st);
    g_scount[slot] = k + 1;
}
}  // namespace nao
NAO_EXPORT int nao_profile_enable(int on) {
    nao::g_prof_on = on != 0;
    for (int s = 0; s < nao::NSLOT; ++s) { nao::g_scount[s] = 0; nao::g_swork[s] = 0.0; }
    const double zero = 0.0;
    cudaMemcpyToSymbol(nao::g_grouped_flops, &zero, sizeof(double));
    return NAO_OK;
}
NAO_EXPORT int nao_profile_kernel(int slot, double *h_ms, double *h_work, int *h_launches) {
    using namespace nao;
    if (slot < 0 || slot >= NSLOT) return -1;
    double tot = 0.0;
    for (int k = 0; k < g_scount[slot]; ++k) {
        cudaEventSynchronize(g_sev[slot][k][1]);
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, g_sev[slot][k][0], g_sev[slot][k][1]) == cudaSuccess) tot += ms;
    }
    if (h_ms) *h_ms = tot;
    double grouped = 0.0;
    if (slot == 1) cudaMemcpyFromSymbol(&grouped, g_grouped_flops, sizeof(double));      // after the event waits above
    if (h_work) *h_work = g_swork[slot] + grouped;
    if (h_launches) *h_launches = g_scount[slot];
    return NAO_OK;
}
NAO_EXPORT int nao_profile_kernel_launches(int slot, double *h_ms, int max_launches) {
    using namespace nao;
    if (slot < 0 || slot >= NSLOT) return -1;
    if (!h_ms) return -2;
    int k = 0;
    for (; k < g_scount[slot] && k < max_launches; ++k) {
        cudaEventSynchronize(g_sev[slot][k][1]);
        float ms = 0.f;
        h_ms[k] = (cudaEventElapsedTime(&ms, g_sev[slot][k][0], g_sev[slot][k][1]) == cudaSuccess) ? ms : -1.0;
    }
    return k;
}
NAO_EXPORT const char *nao_profile_kernel_name(int slot) { return (slot >= 0 && slot < nao::NSLOT) ? nao::kSlotNames[slot] : ""; }
NAO_EXPORT int nao_profile_read(double *h_ms, int max_phases) {
    using namespace nao;
    if (!h_ms) return -1;
    int np = 0;
    for (int i = 0; i + 1 < NPH && i < max_phases; ++i) {
        h_ms[i] = 0.0;
        if (g_ev_made && g_ev_rec[i] && g_ev_rec[i + 1]) {
            cudaEventSynchronize(g_ev[i + 1]);
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, g_ev[i], g_ev[i + 1]) == cudaSuccess) h_ms[i] = ms;
        }
        np = i + 1;
    }
    return np;
}
NAO_EXPORT const char *nao_profile_phase_name(int i) { return (i >= 0 && i < nao::NPH - 1) ? nao::kPhaseNames[i] : ""; }

// ---- FP64 tensor-pipe peak: register-resident DMMA.8x8x4 loop (no memory traffic), the measured counterpart of the derived
// ---- 148 SMs x 128 flop/clk x clock roof used in DESIGN.md 5 and bench.py
namespace nao {
__global__ void __launch_bounds__(512) dmma_peak_kernel(int iters, double *sink) {
    double c[16][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) { c[i][0] = 0.0; c[i][1] = 0.0; }
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}
}  // namespace nao
NAO_EXPORT int nao_dmma_peak(double *h_tflops, void *cuda_stream) {
    using namespace nao;
    if (!h_tflops) return -1;
    if (int rcb = nao::bind_device()) return rcb;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev); cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    static double *h_sink = nullptr, *d_sink = nullptr;          // pinned host word, never written in practice
    if (!h_sink) {
        if (cudaHostAlloc((void **)&h_sink, 8, cudaHostAllocMapped) != cudaSuccess) return NAO_ERR_CUDA;
        if (cudaHostGetDevicePointer((void **)&d_sink, h_sink, 0) != cudaSuccess) return NAO_ERR_CUDA;
    }
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return NAO_ERR_CUDA;
    // exactly ONE CTA of 16 warps per SM: the dynamic shared-memory request (not used by the kernel) keeps a second CTA off the
    // SM -- with several small CTAs per SM the block scheduler places them unevenly (5 on some SMs, 3 on others) and the
    // slowest SM decides the time (measured: 29.7 instead of 37.1 TF/s in about half of the calls)
    const int iters = 40000, ctas = nsm;
    const size_t smem = 120 * 1024;
    static bool attr = false;
    if (!attr) {
        if (cudaFuncSetAttribute(dmma_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return NAO_ERR_CUDA;
        attr = true;
    }
    dmma_peak_kernel<<<ctas, 512, smem, st>>>(iters / 10, d_sink);                 // warm-up
    cudaEventRecord(e0, st);
    dmma_peak_kernel<<<ctas, 512, smem, st>>>(iters, d_sink);
    cudaEventRecord(e1, st);
    NAO_LAUNCHED(); NAO_LAUNCHED();
    if (cudaEventSynchronize(e1) != cudaSuccess) return NAO_ERR_CUDA;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double flops = (double)ctas * 16 /*warps*/ * iters * 16.0 * 512.0;      // one DMMA.8x8x4 = 8*8*4*2 flop
    *h_tflops = flops / (ms * 1e-3) / 1e12;
    return NAO_OK;
}
