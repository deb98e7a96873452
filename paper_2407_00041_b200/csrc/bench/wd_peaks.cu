// wd_peaks.cu (libwdbench.so, bench-only) — streaming ceilings of the device memory, and a register-only FP64 FMA microbenchmark (the paper's section 3.1 method): the
// second roof of the multi-RHS application (cfg 5) and the issue rate one warp per SM
// sub-partition can reach, which is what the TMA kernels' compute side runs on.
#include <cuda_runtime.h>

#include <stddef.h>

#include "../../../include/wd_bench.h"

enum { WD_OK = 0, WD_EINVAL = -1, WD_ENOMEM = -2, WD_ECUDA = -4 };

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

extern "C" int wdb_measure_fp64(int threads_per_sm, int ilp, int one_cta_per_sm, int distinct_operands, double *tflops,
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

// ---------------------------------------------------------------- streaming ceilings
namespace {
// MODE 0: read only.  1: copy.  2: seven 16-byte reads per 16-byte write (the operator's mix).
template <int MODE> __global__ void __launch_bounds__(256) k_stream(const double2 *__restrict__ src, double2 *__restrict__ dst, size_t n,
                                                                     double *sink) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    double s = 0.0;
    if (MODE == 0) {
        size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n; i += 4 * stride) {  // four independent 16-byte loads in flight per thread
            const double2 a = __ldcs(src + i), b = __ldcs(src + i + stride), c = __ldcs(src + i + 2 * stride),
                          d = __ldcs(src + i + 3 * stride);
            s += a.x + b.y + c.x + d.y;
        }
        for (; i < n; i += stride) s += __ldcs(src + i).x;
    } else if (MODE == 1) {
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) __stcs(dst + i, __ldcs(src + i));
    } else {
        const size_t m = n / 7;  // 7 source planes of m elements, one destination plane
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < m; i += stride) {
            double2 v = __ldcs(src + i);
#pragma unroll
            for (int k = 1; k < 7; k++) {
                const double2 w = __ldcs(src + (size_t)k * m + i);
                v.x += w.x;
                v.y += w.y;
            }
            __stcs(dst + i, v);
        }
    }
    if (s == 123.456) *sink = s;  // never true
}
}  // namespace

extern "C" int wdb_measure_stream(int mode, size_t bytes, int reps, double *gbs) {
    if (!gbs || mode < 0 || mode > 2 || bytes < (1u << 20) || reps < 1) return WD_EINVAL;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return WD_ECUDA;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const size_t n = bytes / sizeof(double2);
    double2 *src = nullptr, *dst = nullptr;
    double *sink = nullptr;
    const size_t dst_n = (mode == 1) ? n : (mode == 2) ? n / 7 : 1;
    if (cudaMalloc((void **)&src, n * sizeof(double2)) != cudaSuccess) return WD_ENOMEM;
    if (cudaMalloc((void **)&dst, dst_n * sizeof(double2)) != cudaSuccess) { cudaFree(src); return WD_ENOMEM; }
    cudaMalloc((void **)&sink, sizeof(double));
    cudaMemset(src, 0, n * sizeof(double2));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = nsm * 8;
    float best = 1e30f;
    cudaError_t e = cudaSuccess;
    for (int r = 0; r < reps + 1 && e == cudaSuccess; r++) {  // first repetition = warm-up
        cudaEventRecord(e0);
        if (mode == 0) k_stream<0><<<grid, 256>>>(src, dst, n, sink);
        else if (mode == 1) k_stream<1><<<grid, 256>>>(src, dst, n, sink);
        else k_stream<2><<<grid, 256>>>(src, dst, n, sink);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(src);
    cudaFree(dst);
    cudaFree(sink);
    if (e != cudaSuccess) return WD_ECUDA;
    const double moved = (mode == 0) ? (double)n * 16 : (mode == 1) ? 2.0 * n * 16 : (double)(n / 7) * 8 * 16;
    *gbs = moved / (best * 1e-3) / 1e9;
    return WD_OK;
}

// ---------------------------------------------------------------- LDS.128 lane-pattern probe (wd_bench.h)
namespace {
__device__ __forceinline__ void lds128(double &a, double &b, unsigned addr) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(addr) : "memory");
}
__global__ void k_lds_pattern(double *out, long long *cyc, int iters, int pattern) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31;
    for (int i = tid; i < 98304 / 8; i += blockDim.x) reinterpret_cast<double *>(smem)[i] = i;
    __syncthreads();
    const unsigned base = (unsigned)__cvta_generic_to_shared(smem);
    unsigned off = 0;
    switch (pattern) {
    case 0: off = lane * 16; break;
    case 1: off = (lane & 7) * 16; break;
    case 2: off = (lane >> 2) * 16; break;
    case 3: off = 0; break;
    case 4: off = (lane & 3) * 12288 + (lane >> 2) * 16; break;
    case 5: off = (lane >> 3) * 12288 + (lane & 7) * 16; break;
    default: off = (lane >> 1) * 16; break;
    }
    double s0 = 0, s1 = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; it++) {
        const unsigned a = base + off + ((it & 3) * 512);
#pragma unroll
        for (int j = 0; j < 16; j++) {  // sixteen different addresses: nothing for the compiler to merge
            double x, y;
            lds128(x, y, a + j * 2048);
            s0 += x;
            s1 += y;
        }
    }
    const long long t1 = clock64();
    if (tid == 0) cyc[blockIdx.x] = t1 - t0;
    out[blockIdx.x * blockDim.x + tid] = s0 + s1;
}
}  // namespace

extern "C" int wdb_measure_lds(int pattern, double *cycles) {
    if (!cycles || pattern < 0 || pattern > 6) return WD_EINVAL;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return WD_ECUDA;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) return WD_ECUDA;
    const int threads = 256, iters = 4096, smem = 98304;
    double *out = nullptr;
    long long *cyc = nullptr;
    if (cudaMalloc((void **)&out, (size_t)nsm * threads * sizeof(double)) != cudaSuccess) return WD_ENOMEM;
    if (cudaMalloc((void **)&cyc, (size_t)nsm * sizeof(long long)) != cudaSuccess) {
        cudaFree(out);
        return WD_ENOMEM;
    }
    cudaError_t e = cudaFuncSetAttribute(k_lds_pattern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    long long *host = new long long[nsm];
    for (int rep = 0; rep < 2 && e == cudaSuccess; rep++) {
        k_lds_pattern<<<nsm, threads, smem>>>(out, cyc, iters, pattern);
        e = cudaDeviceSynchronize();
    }
    if (e == cudaSuccess) e = cudaMemcpy(host, cyc, (size_t)nsm * sizeof(long long), cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) {
        double sum = 0.0;
        for (int k = 0; k < nsm; k++) sum += (double)host[k];
        *cycles = sum / nsm / ((double)iters * 16 * (threads / 32));
    }
    delete[] host;
    cudaFree(out);
    cudaFree(cyc);
    return (e == cudaSuccess) ? WD_OK : WD_ECUDA;
}
