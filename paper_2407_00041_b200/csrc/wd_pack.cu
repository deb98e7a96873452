// wd_pack.cu — layout conversion between the canonical site-major AoS layouts (include/wd.h,
// PAPER.md:538-554) and the device SoA layout (wd_internal.h).  Step a0 of SURVEY.md §8(a): a
// permutation only, done at load time, never inside wd_apply.  The paper's counterpart is the
// chunkwise -> componentwise reorder kernel of Listing 4.4.
//
// Two implementations of the same permutation:
//   host packers      : OpenMP loops over a chunk of sites into a pinned staging buffer
//   device transposes : shared-memory tiled kernels on a device staging buffer (used by
//                       wd_apply_host and by WD_OPT_DEVICE_PACK)
#include "wd_internal.h"

namespace wd {

// ---------------------------------------------------------------- host side
void host_pack_aos_to_soa(double2 *dst, const double2 *src_aos, long long i0, long long cnt, int ncomp) {
    // dst [ncomp][cnt]  <-  src_aos [V][ncomp] rows i0 .. i0+cnt
    const long long B = 64;
#pragma omp parallel for schedule(static)
    for (long long b = 0; b < (cnt + B - 1) / B; b++) {
        const long long lo = b * B, hi = (lo + B < cnt) ? lo + B : cnt;
        for (int c = 0; c < ncomp; c++)
            for (long long j = lo; j < hi; j++) dst[(long long)c * cnt + j] = src_aos[(i0 + j) * ncomp + c];
    }
}

void host_unpack_soa_to_aos(double2 *dst_aos, const double2 *src, long long i0, long long cnt, int ncomp) {
    const long long B = 64;
#pragma omp parallel for schedule(static)
    for (long long b = 0; b < (cnt + B - 1) / B; b++) {
        const long long lo = b * B, hi = (lo + B < cnt) ? lo + B : cnt;
        for (long long j = lo; j < hi; j++)
            for (int c = 0; c < ncomp; c++) dst_aos[(i0 + j) * ncomp + c] = src[(long long)c * cnt + j];
    }
}

// canonical 42 complex -> 36 slots (wd_internal.h): pair q of the real diagonal -> slot_diag(q/3, q%3),
// strict-upper entry k of c[12..41] -> slot_off(k/15, k%15)
__host__ __device__ static inline int slot_of_pair(int q) { return slot_diag(q / 3, q % 3); }
__host__ __device__ static inline int slot_of_upper(int k) { return slot_off(k / 15, k % 15); }
void host_pack_clover(double2 *dst, const double2 *src42, long long i0, long long cnt) {
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < cnt; j++) {
        const double2 *s = src42 + (i0 + j) * kCloverCanon;
        for (int q = 0; q < 6; q++) dst[(long long)slot_of_pair(q) * cnt + j] = make_double2(s[2 * q].x, s[2 * q + 1].x);
        for (int k = 0; k < 30; k++) dst[(long long)slot_of_upper(k) * cnt + j] = s[12 + k];
    }
}

void host_unpack_clover(double2 *dst42, const double2 *src, long long i0, long long cnt) {
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < cnt; j++) {
        double2 *d = dst42 + (i0 + j) * kCloverCanon;
        for (int q = 0; q < 6; q++) {
            const double2 v = src[(long long)slot_of_pair(q) * cnt + j];
            d[2 * q] = make_double2(v.x, 0.0);
            d[2 * q + 1] = make_double2(v.y, 0.0);
        }
        for (int k = 0; k < 30; k++) d[12 + k] = src[(long long)slot_of_upper(k) * cnt + j];
    }
}

void host_pack_spinor_blocked(double2 *dst, const double2 *const *src, int B, int nlive, long long i0, long long cnt) {
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < cnt; j++)
        for (int r = 0; r < B; r++)
            for (int c = 0; c < kSpinorComps; c++)
                dst[((long long)c * cnt + j) * B + r] = (r < nlive) ? src[r][(i0 + j) * kSpinorComps + c] : make_double2(0.0, 0.0);
}

void host_unpack_spinor_blocked(double2 *const *dst, const double2 *src, int B, int nlive, long long i0, long long cnt) {
#pragma omp parallel for schedule(static)
    for (long long j = 0; j < cnt; j++)
        for (int r = 0; r < nlive; r++)
            for (int c = 0; c < kSpinorComps; c++) dst[r][(i0 + j) * kSpinorComps + c] = src[((long long)c * cnt + j) * B + r];
}

// ---------------------------------------------------------------- device side
// A CTA moves TS sites x ncomp components through shared memory: the AoS side is accessed as one
// contiguous run of TS*ncomp elements, the SoA side as ncomp runs of TS elements.
constexpr int TS = 64;

template <bool TO_SOA>
__global__ void __launch_bounds__(256) k_transpose(double2 *__restrict__ dst, const double2 *__restrict__ src,
                                                  long long V, long long Vs, int ncomp) {
    extern __shared__ double2 tile[];  // [TS][ncomp + 1]
    const long long i0 = (long long)blockIdx.x * TS;
    const int cnt = (int)((V - i0 < TS) ? (V - i0) : TS);
    const int pitch = ncomp + 1;
    const int n = cnt * ncomp;
    if (TO_SOA) {
        for (int e = threadIdx.x; e < n; e += blockDim.x) tile[(e / ncomp) * pitch + (e % ncomp)] = src[i0 * ncomp + e];
        __syncthreads();
        for (int e = threadIdx.x; e < ncomp * TS; e += blockDim.x) {
            const int c = e / TS, j = e % TS;
            if (j < cnt) dst[(long long)c * Vs + i0 + j] = tile[j * pitch + c];
        }
    } else {
        for (int e = threadIdx.x; e < ncomp * TS; e += blockDim.x) {
            const int c = e / TS, j = e % TS;
            if (j < cnt) tile[j * pitch + c] = src[(long long)c * Vs + i0 + j];
        }
        __syncthreads();
        for (int e = threadIdx.x; e < n; e += blockDim.x) dst[i0 * ncomp + e] = tile[(e / ncomp) * pitch + (e % ncomp)];
    }
}

cudaError_t launch_aos_to_soa(double2 *dst_soa, const double2 *src_aos, long long V, long long Vs, int ncomp, cudaStream_t st) {
    const unsigned grid = (unsigned)((V + TS - 1) / TS);
    k_transpose<true><<<grid, 256, TS * (ncomp + 1) * sizeof(double2), st>>>(dst_soa, src_aos, V, Vs, ncomp);
    return cudaGetLastError();
}

cudaError_t launch_soa_to_aos(double2 *dst_aos, const double2 *src_soa, long long V, long long Vs, int ncomp, cudaStream_t st) {
    const unsigned grid = (unsigned)((V + TS - 1) / TS);
    k_transpose<false><<<grid, 256, TS * (ncomp + 1) * sizeof(double2), st>>>(dst_aos, src_soa, V, Vs, ncomp);
    return cudaGetLastError();
}

template <bool TO_DEV>
__global__ void __launch_bounds__(256) k_clover_convert(double2 *__restrict__ dst, const double2 *__restrict__ src, long long V,
                                                       long long Vs) {
    __shared__ double2 tile[TS * (kCloverCanon + 1)];
    const long long i0 = (long long)blockIdx.x * TS;
    const int cnt = (int)((V - i0 < TS) ? (V - i0) : TS);
    constexpr int pitch = kCloverCanon + 1;
    if (TO_DEV) {
        for (int e = threadIdx.x; e < cnt * kCloverCanon; e += blockDim.x)
            tile[(e / kCloverCanon) * pitch + (e % kCloverCanon)] = src[i0 * kCloverCanon + e];
        __syncthreads();
        for (int e = threadIdx.x; e < kCloverSlots * TS; e += blockDim.x) {
            const int q = e / TS, j = e % TS;  // q = 0..5 diagonal pairs, 6..35 strict-upper entries
            if (j >= cnt) continue;
            double2 v;
            if (q < 6) v = make_double2(tile[j * pitch + 2 * q].x, tile[j * pitch + 2 * q + 1].x);
            else v = tile[j * pitch + 6 + q];
            const int slot = (q < 6) ? slot_of_pair(q) : slot_of_upper(q - 6);
            dst[(long long)slot * Vs + i0 + j] = v;
        }
    } else {
        for (int e = threadIdx.x; e < kCloverSlots * TS; e += blockDim.x) {
            const int q = e / TS, j = e % TS;
            if (j >= cnt) continue;
            const int slot = (q < 6) ? slot_of_pair(q) : slot_of_upper(q - 6);
            const double2 v = src[(long long)slot * Vs + i0 + j];
            if (q < 6) {
                tile[j * pitch + 2 * q] = make_double2(v.x, 0.0);
                tile[j * pitch + 2 * q + 1] = make_double2(v.y, 0.0);
            } else {
                tile[j * pitch + 6 + q] = v;
            }
        }
        __syncthreads();
        for (int e = threadIdx.x; e < cnt * kCloverCanon; e += blockDim.x)
            dst[i0 * kCloverCanon + e] = tile[(e / kCloverCanon) * pitch + (e % kCloverCanon)];
    }
}

cudaError_t launch_clover_canon_to_dev(double2 *dst_slots, const double2 *src42, long long V, long long Vs, cudaStream_t st) {
    k_clover_convert<true><<<(unsigned)((V + TS - 1) / TS), 256, 0, st>>>(dst_slots, src42, V, Vs);
    return cudaGetLastError();
}

cudaError_t launch_clover_dev_to_canon(double2 *dst42, const double2 *src_slots, long long V, long long Vs, cudaStream_t st) {
    k_clover_convert<false><<<(unsigned)((V + TS - 1) / TS), 256, 0, st>>>(dst42, src_slots, V, Vs);
    return cudaGetLastError();
}

// two-row copy of the gauge field: rows 0 and 1 of every link, double2 [4][6][Vs]
__global__ void __launch_bounds__(256) k_compress_gauge(double2 *__restrict__ U2, const double2 *__restrict__ U, long long V, long long Vs) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= V) return;
    const int mu = blockIdx.y / 6, k = blockIdx.y % 6;
    U2[(long long)(6 * mu + k) * Vs + i] = U[(long long)(9 * mu + k) * Vs + i];
}

cudaError_t launch_compress_gauge(double2 *U2, const double2 *U, long long V, long long Vs, cudaStream_t st) {
    k_compress_gauge<<<dim3((unsigned)((V + 255) / 256), 24), 256, 0, st>>>(U2, U, V, Vs);
    return cudaGetLastError();
}

}  // namespace wd
