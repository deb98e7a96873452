// wd_kernels.cu — hopping / fused Wilson-clover kernels for sm_100a (FP64, one thread per site).
//
// out(x) = S(x) psi(x) - 1/2 sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^H psi(x-mu) ]
// (eq. 1.13) in ONE pass: every psi, U, S byte is requested once per use and the
// result is written once — the paper's Alg. 4 needed 17 launches and eight
// intermediate half-spinor fields in global memory for the same thing.
//
// Geometries:
//   linear    : thread i <-> site i, any lattice extents (coordinates by div/mod).
//   tile BTxBZxBYxBX : a CTA owns a 4-D tile of sites and marches it along T for `tchunk` slices,
//               so that psi(t+1) fetched for slice t is an L1/L2 hit for slices t+1 and t+2, and
//               the CTAs in flight cover a compact Z-slab (rasterisation groups) whose T-window
//               stays L2-resident (SURVEY.md §7 "T-direction reuse").
// Neighbour indices and the periodic wrap are computed in-kernel (step a1): no neighbour table
// (the paper's int[4V] table, would add 16 B/site of traffic).
#include "wd_internal.h"
#include "wd_math.cuh"

namespace wd {

__device__ __forceinline__ cd ldg(const cd *p) { return __ldg(p); }

// fwd / bwd = false: the hop crosses an open boundary of a domain-decomposed sub-lattice (KParams::open_mask) and is
// left to the exterior kernel of wd_dd.cu.
template <int MU>
__device__ __forceinline__ void hop_direction(cd acc[12], const cd *__restrict__ psi, const cd *__restrict__ U,
                                              long long V, long long i, long long ip, long long im, bool fwd, bool bwd) {
    cd p[12], u[9];
    if (fwd) {  // forward: (1 - gamma_mu) (x) U_mu(x) psi(x+mu)
#pragma unroll
        for (int k = 0; k < 9; k++) u[k] = ldg(U + (long long)(MU * 9 + k) * V + i);
#pragma unroll
        for (int c = 0; c < 12; c++) p[c] = ldg(psi + (long long)c * V + ip);
        hop_term<MU, -1>(acc, p, u);
    }
    if (bwd) {  // backward: (1 + gamma_mu) (x) U_mu(x-mu)^H psi(x-mu)
#pragma unroll
        for (int k = 0; k < 9; k++) u[k] = ldg(U + (long long)(MU * 9 + k) * V + im);
#pragma unroll
        for (int c = 0; c < 12; c++) p[c] = ldg(psi + (long long)c * V + im);
        hop_term<MU, +1>(acc, p, u);
    }
}

template <int SELF>
__device__ __forceinline__ void site_apply(const KParams &p, long long i, int t, int z, int y, int x) {
    const cd *__restrict__ psi = p.psi;
    const cd *__restrict__ U = p.U;
    const long long V = p.Vs;  // component stride
    const int open = p.open_mask;
    cd acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);

    {
        const long long s = p.stride[0];
        const long long ip = (t + 1 < p.n[0]) ? i + s : i - (long long)(p.n[0] - 1) * s;
        const long long im = (t > 0) ? i - s : i + (long long)(p.n[0] - 1) * s;
        hop_direction<0>(acc, psi, U, V, i, ip, im, !(open & 1) || t + 1 < p.n[0], !(open & 1) || t > 0);
    }
    {
        const long long s = p.stride[1];
        const long long ip = (z + 1 < p.n[1]) ? i + s : i - (long long)(p.n[1] - 1) * s;
        const long long im = (z > 0) ? i - s : i + (long long)(p.n[1] - 1) * s;
        hop_direction<1>(acc, psi, U, V, i, ip, im, !(open & 2) || z + 1 < p.n[1], !(open & 2) || z > 0);
    }
    {
        const long long s = p.stride[2];
        const long long ip = (y + 1 < p.n[2]) ? i + s : i - (long long)(p.n[2] - 1) * s;
        const long long im = (y > 0) ? i - s : i + (long long)(p.n[2] - 1) * s;
        hop_direction<2>(acc, psi, U, V, i, ip, im, !(open & 4) || y + 1 < p.n[2], !(open & 4) || y > 0);
    }
    {
        const long long ip = (x + 1 < p.n[3]) ? i + 1 : i - (long long)(p.n[3] - 1);
        const long long im = (x > 0) ? i - 1 : i + (long long)(p.n[3] - 1);
        hop_direction<3>(acc, psi, U, V, i, ip, im, !(open & 8) || x + 1 < p.n[3], !(open & 8) || x > 0);
    }

    cd *__restrict__ out = p.out;
    if (SELF == SELF_NONE) {
#pragma unroll
        for (int c = 0; c < 12; c++) out[(long long)c * V + i] = make_double2(-0.5 * acc[c].x, -0.5 * acc[c].y);
    } else if (SELF == SELF_MASS) {
#pragma unroll
        for (int c = 0; c < 12; c++) {
            const cd q = ldg(psi + (long long)c * V + i);
            out[(long long)c * V + i] = make_double2(fma(p.mass, q.x, -0.5 * acc[c].x), fma(p.mass, q.y, -0.5 * acc[c].y));
        }
    } else {
        const cd *__restrict__ S = p.S;
#pragma unroll
        for (int b = 0; b < 2; b++) {
            cd q[6], a[15], r[6];
            double d[6];
#pragma unroll
            for (int j = 0; j < 3; j++) {
                const cd dd = ldg(S + (long long)slot_diag(b, j) * V + i);
                d[2 * j] = dd.x;
                d[2 * j + 1] = dd.y;
            }
#pragma unroll
            for (int k = 0; k < 15; k++) a[k] = ldg(S + (long long)slot_off(b, k) * V + i);
#pragma unroll
            for (int c = 0; c < 6; c++) q[c] = ldg(psi + (long long)(6 * b + c) * V + i);
            herm6_mul(r, d, a, q);
#pragma unroll
            for (int c = 0; c < 6; c++)
                out[(long long)(6 * b + c) * V + i] =
                    make_double2(fma(-0.5, acc[6 * b + c].x, r[c].x), fma(-0.5, acc[6 * b + c].y, r[c].y));
        }
    }
}

// ---- linear geometry ------------------------------------------------------------------------
template <int SELF, int NT> __global__ void __launch_bounds__(NT) k_linear(const KParams p) {
    const long long i = (long long)blockIdx.x * NT + threadIdx.x;
    if (i >= p.V) return;
    long long r = i;
    const int x = (int)(r % p.n[3]); r /= p.n[3];
    const int y = (int)(r % p.n[2]); r /= p.n[2];
    const int z = (int)(r % p.n[1]); r /= p.n[1];
    const int t = (int)r;
    site_apply<SELF>(p, i, t, z, y, x);
}

template <int NT> static cudaError_t launch_linear(const KParams &p, int self, cudaStream_t st) {
    const unsigned grid = (unsigned)((p.V + NT - 1) / NT);
    if (self == SELF_NONE) k_linear<SELF_NONE, NT><<<grid, NT, 0, st>>>(p);
    else if (self == SELF_MASS) k_linear<SELF_MASS, NT><<<grid, NT, 0, st>>>(p);
    else k_linear<SELF_CLOVER, NT><<<grid, NT, 0, st>>>(p);
    return cudaGetLastError();
}

// ---- tiled geometry with T-marching ---------------------------------------------------------
// CTA order (blockIdx.x ascending = dispatch order): Z-slab group slowest, then T-chunk, then the
// Z/Y/X tiles of the slab.  All CTAs in flight therefore work on the same few T-slices of one
// slab, and consecutive T-chunks of a slab follow each other.
template <int SELF, int BT, int BZ, int BY, int BX>
__global__ void __launch_bounds__(BT *BZ *BY *BX) k_tiled(const KParams p) {
    const int tiles_per_slab = p.gz * p.nty * p.ntx;
    const int per_group = tiles_per_slab * p.ntc;
    int lb = blockIdx.x;
    const int g = lb / per_group;
    lb -= g * per_group;
    const int tc = lb / tiles_per_slab;
    lb -= tc * tiles_per_slab;
    const int zt = g * p.gz + lb / (p.nty * p.ntx);
    lb %= (p.nty * p.ntx);
    const int yt = lb / p.ntx, xt = lb % p.ntx;

    const int tid = threadIdx.x;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = (tid / (BX * BY)) % BZ, lt = tid / (BX * BY * BZ);
    const int x = xt * BX + lx, y = yt * BY + ly, z = zt * BZ + lz;
    const int t0 = tc * p.tchunk + lt;
    const long long base = ((long long)z * p.n[2] + y) * p.n[3] + x;
    for (int tt = 0; tt < p.tchunk; tt += BT) {
        const int t = t0 + tt;
        site_apply<SELF>(p, (long long)t * p.stride[0] + base, t, z, y, x);
    }
}

template <int BT, int BZ, int BY, int BX> static cudaError_t launch_tiled(const KParams &p, int self, cudaStream_t st) {
    constexpr int NT = BT * BZ * BY * BX;
    const unsigned grid = (unsigned)(p.ntx * p.nty * p.ntz * p.ntc);
    if (self == SELF_NONE) k_tiled<SELF_NONE, BT, BZ, BY, BX><<<grid, NT, 0, st>>>(p);
    else if (self == SELF_MASS) k_tiled<SELF_MASS, BT, BZ, BY, BX><<<grid, NT, 0, st>>>(p);
    else k_tiled<SELF_CLOVER, BT, BZ, BY, BX><<<grid, NT, 0, st>>>(p);
    return cudaGetLastError();
}

// ---- self-coupling kernel of the unfused variant: out += S psi / out += mass psi -------------
template <int SELF> __global__ void __launch_bounds__(256) k_selfcoupling(const KParams p) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= p.V) return;
    const long long V = p.Vs;  // component stride
    const cd *__restrict__ psi = p.psi;
    cd *__restrict__ out = p.out;
    if (SELF == SELF_MASS) {
#pragma unroll
        for (int c = 0; c < 12; c++) {
            const cd q = ldg(psi + (long long)c * V + i);
            cd o = out[(long long)c * V + i];
            o.x = fma(p.mass, q.x, o.x);
            o.y = fma(p.mass, q.y, o.y);
            out[(long long)c * V + i] = o;
        }
    } else {
        const cd *__restrict__ S = p.S;
#pragma unroll
        for (int b = 0; b < 2; b++) {
            cd q[6], a[15], r[6];
            double d[6];
#pragma unroll
            for (int j = 0; j < 3; j++) {
                const cd dd = ldg(S + (long long)slot_diag(b, j) * V + i);
                d[2 * j] = dd.x;
                d[2 * j + 1] = dd.y;
            }
#pragma unroll
            for (int k = 0; k < 15; k++) a[k] = ldg(S + (long long)slot_off(b, k) * V + i);
#pragma unroll
            for (int c = 0; c < 6; c++) q[c] = ldg(psi + (long long)(6 * b + c) * V + i);
            herm6_mul(r, d, a, q);
#pragma unroll
            for (int c = 0; c < 6; c++) {
                cd o = out[(long long)(6 * b + c) * V + i];
                o.x += r[c].x;
                o.y += r[c].y;
                out[(long long)(6 * b + c) * V + i] = o;
            }
        }
    }
}

cudaError_t launch_selfcoupling(const KParams &p, int self, cudaStream_t st) {
    const unsigned grid = (unsigned)((p.V + 255) / 256);
    if (self == SELF_MASS) k_selfcoupling<SELF_MASS><<<grid, 256, 0, st>>>(p);
    else k_selfcoupling<SELF_CLOVER><<<grid, 256, 0, st>>>(p);
    return cudaGetLastError();
}

// ---- registry -------------------------------------------------------------------------------
// linear: any lattice.  tile_*: LDG kernels for lattices no TMA tile divides (cfg 1: 4^4).  tma/tmb/tmc: the TMA kernels.
static const KernelInfo kKernels[] = {
    {"linear256", 0, 0, 0, 0, 256, false, launch_linear<256>},
    {"tile_1x4x4x16", 1, 4, 4, 16, 256, false, launch_tiled<1, 4, 4, 16>},
    {"tile_2x4x4x4", 2, 4, 4, 4, 128, false, launch_tiled<2, 4, 4, 4>},
    {"tma_2x4x16", 1, 2, 4, 16, 160, true, launch_tma_2x4x16},
    {"tmb_4x4x8", 1, 4, 4, 8, 160, true, launch_tmb_4x4x8},
    {"tmb_2x8x8", 1, 2, 8, 8, 160, true, launch_tmb_2x8x8},
    {"tmc_2x4x16", 1, 2, 4, 16, 160, true, launch_tmc_2x4x16},
};

int kernel_count() { return (int)(sizeof(kKernels) / sizeof(kKernels[0])); }
const KernelInfo &kernel_info(int id) { return kKernels[id]; }

}  // namespace wd
