// scalar.cuh -- real/complex FP64 scalar helpers so kernels can be written once for both dtypes.
#pragma once
#include "nao_internal.cuh"

namespace nao {

template <class T> struct Ops;
template <> struct Ops<double> {
    static const bool is_complex = false;
    __host__ __device__ static double zero() { return 0.0; }
    __host__ __device__ static double one() { return 1.0; }
    __host__ __device__ static double real(double x) { return x; }
    __host__ __device__ static double imag(double) { return 0.0; }
    __host__ __device__ static double from_real(double x) { return x; }
    __host__ __device__ static double conj(double a) { return a; }
    __host__ __device__ static double add(double a, double b) { return a + b; }
    __host__ __device__ static double sub(double a, double b) { return a - b; }
    __host__ __device__ static double mul(double a, double b) { return a * b; }
    __host__ __device__ static double mul_conj(double a, double b) { return a * b; }     // a * conj(b)
    __host__ __device__ static double conj_mul(double a, double b) { return a * b; }     // conj(a) * b
    __host__ __device__ static double scale(double a, double s) { return a * s; }
    __host__ __device__ static double abs2(double a) { return a * a; }
    __host__ __device__ static double fma(double a, double b, double c) { return a * b + c; }   // a*b + c
};
template <> struct Ops<cplx> {
    static const bool is_complex = true;
    __host__ __device__ static cplx zero() { return make_double2(0.0, 0.0); }
    __host__ __device__ static cplx one() { return make_double2(1.0, 0.0); }
    __host__ __device__ static double real(cplx x) { return x.x; }
    __host__ __device__ static double imag(cplx x) { return x.y; }
    __host__ __device__ static cplx from_real(double x) { return make_double2(x, 0.0); }
    __host__ __device__ static cplx conj(cplx a) { return make_double2(a.x, -a.y); }
    __host__ __device__ static cplx add(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
    __host__ __device__ static cplx sub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
    __host__ __device__ static cplx mul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
    __host__ __device__ static cplx mul_conj(cplx a, cplx b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
    __host__ __device__ static cplx conj_mul(cplx a, cplx b) { return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }
    __host__ __device__ static cplx scale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
    __host__ __device__ static double abs2(cplx a) { return a.x * a.x + a.y * a.y; }
    __host__ __device__ static cplx fma(cplx a, cplx b, cplx c) {
        return make_double2(c.x + a.x * b.x - a.y * b.y, c.y + a.x * b.y + a.y * b.x);
    }
};

// loads that bypass L1 (data produced by other CTAs of the same kernel)
__device__ __forceinline__ double ldcg(const double *p) { return __ldcg(p); }
__device__ __forceinline__ cplx ldcg(const cplx *p) { return __ldcg(p); }
__device__ __forceinline__ int ldcg(const int *p) { return __ldcg(p); }

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ cplx warp_sum(cplx v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    return v;
}

// asynchronous global -> shared copies (LDGSTS); pred = false zero-fills the destination
__device__ __forceinline__ void cp_async8(void *smem, const void *g, bool pred) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    int sz = pred ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(g), "r"(sz));
}
__device__ __forceinline__ void cp_async16(void *smem, const void *g, bool pred) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    int sz = pred ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(g), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// Grid-wide barrier among the `nctas` CTAs that share `ctr` (all co-resident: cooperative launch).
// `ordinal` = 1 for the first barrier on this counter, 2 for the second, ...
__device__ __forceinline__ void group_barrier(unsigned *ctr, unsigned nctas, unsigned ordinal) {
    __syncthreads();
    if (nctas > 1 && threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        const unsigned target = nctas * ordinal;
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
        } while (v < target);
        __threadfence();
    }
    __syncthreads();
}

}  // namespace nao
