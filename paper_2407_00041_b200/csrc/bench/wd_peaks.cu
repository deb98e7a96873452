// wd_peaks.cu — register-only FP64 FMA microbenchmark (the paper's section 3.1 method): the
// second roof of the multi-RHS application (cfg 5) and the issue rate one warp per SM
// sub-partition can reach, which is what the TMA kernels' compute side runs on.
#include <cuda_runtime.h>

#include "../../include/wd.h"

namespace {

// DISTINCT = false: a = fma(a, b, c) with b, c shared by all chains (two of the three operands are re-used
// registers).  DISTINCT = true: a_j = fma(x_j, y_j, a_j) with every operand a register pair of its own, which is
// what the SU(3) and 6x6 arithmetic of the operator looks like to the register file.
template <int ILP, bool DISTINCT> __global__ void k_dfma(double *out, int iters, double b, double c) {
    extern __shared__ unsigned char pad[];  // only sizes the CTA so that one CTA fits per SM when asked to
    double a[ILP], x[ILP], y[ILP];
#pragma unroll
    for (int j = 0; j < ILP; j++) {
        a[j] = 1.0 + 1e-3 * (threadIdx.x + j);
        x[j] = b + 1e-9 * j;
        y[j] = c * (j + 1);
    }
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int j = 0; j < ILP; j++) a[j] = DISTINCT ? fma(x[j], y[(j + 1) % ILP], a[j]) : fma(a[j], b, c);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < ILP; j++) s += a[j];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;  // never true: keeps the chain alive
}

template <int ILP, bool D> cudaError_t run(int grid, int threads, size_t smem, int iters, double *out, float *ms) {
    cudaError_t e = cudaFuncSetAttribute(k_dfma<ILP, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    k_dfma<ILP, D><<<grid, threads, smem>>>(out, iters / 8, 1.0000001, 1e-9);  // warm-up
    cudaEventRecord(e0);
    k_dfma<ILP, D><<<grid, threads, smem>>>(out, iters, 1.0000001, 1e-9);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return e;
}

}  // namespace

extern "C" int wd_measure_fp64(int threads_per_sm, int ilp, int one_cta_per_sm, int distinct_operands, double *tflops,
                               double *cycles_per_fma_per_warp) {
    if (!tflops || threads_per_sm < 32 || threads_per_sm > 1024 || threads_per_sm % 32) return WD_EINVAL;
    int dev = 0, nsm = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return WD_ECUDA;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    const size_t smem = one_cta_per_sm ? 200 * 1024 : 0;
    const int ctas_per_sm = one_cta_per_sm ? 1 : 2048 / threads_per_sm;
    const int grid = nsm * ctas_per_sm, iters = 1 << 16;
    double *out = nullptr;
    if (cudaMalloc((void **)&out, (size_t)grid * threads_per_sm * sizeof(double)) != cudaSuccess) return WD_ENOMEM;
    float ms = 0.f;
    cudaError_t e;
#define WD_RUN(I) (distinct_operands ? run<I, true>(grid, threads_per_sm, smem, iters, out, &ms) : run<I, false>(grid, threads_per_sm, smem, iters, out, &ms))
    switch (ilp) {
    case 1: e = WD_RUN(1); break;
    case 2: e = WD_RUN(2); break;
    case 4: e = WD_RUN(4); break;
    case 8: e = WD_RUN(8); break;
    case 16: e = WD_RUN(16); break;
    default: cudaFree(out); return WD_EINVAL;
    }
#undef WD_RUN
    cudaFree(out);
    if (e != cudaSuccess) return WD_ECUDA;
    const double fmas = (double)grid * threads_per_sm * (double)iters * ilp;
    *tflops = 2.0 * fmas / (ms * 1e-3) / 1e12;
    if (cycles_per_fma_per_warp) {  // at the nominal maximum clock; one warp's issue interval when ctas_per_sm * warps share the SM
        const double warps_per_sm = (double)ctas_per_sm * threads_per_sm / 32.0;
        const double warp_fmas_per_sm = (double)iters * ilp * warps_per_sm;
        *cycles_per_fma_per_warp = (ms * 1e-3) * (khz * 1e3) / warp_fmas_per_sm * (warps_per_sm < 4 ? warps_per_sm : 4.0);
    }
    return WD_OK;
}
