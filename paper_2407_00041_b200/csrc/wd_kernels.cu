// wd_kernels.cu — FP64 instantiation of the LDG kernels (wd_ldg_kernels.cuh), the self-coupling kernel of the unfused
// variant, and the kernel registry.
#include "wd_ldg_kernels.cuh"

namespace wd {

template <int NT> static cudaError_t launch_linear(const KParams &p, int self, cudaStream_t st) {
    return launch_linear_t<NT, cd>(make_kp<cd>(p, p.psi, p.U, p.S, p.out), self, st);
}
template <int BT, int BZ, int BY, int BX> static cudaError_t launch_tiled(const KParams &p, int self, cudaStream_t st) {
    return launch_tiled_t<BT, BZ, BY, BX, cd>(make_kp<cd>(p, p.psi, p.U, p.S, p.out), self, st);
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
// linear256: any lattice (the automatic choice where no TMA tile divides it, and for small lattices).  tile_1x4x4x16: the
// tiled one-thread-per-site kernel, used by the FP32 variant and selectable.  tma / tmb / tmw / tmq / tmqb: the TMA kernels.
static const KernelInfo kKernels[] = {
    {"linear256", 0, 0, 0, 0, 256, false, 1, launch_linear<256>},
    {"tile_1x4x4x16", 1, 4, 4, 16, 256, false, 1, launch_tiled<1, 4, 4, 16>},
    {"tma_2x4x16", 1, 2, 4, 16, 160, true, 1, launch_tma_2x4x16},
    {"tmb_4x4x8", 1, 4, 4, 8, 160, true, 1, launch_tmb_4x4x8},
    {"tmb_2x4x16", 1, 2, 4, 16, 160, true, 1, launch_tmb_2x4x16},
    {"tmw_2x4x16", 1, 2, 4, 16, 384, true, 1, launch_tmw_2x4x16},
    {"tmq_2x4x8", 1, 2, 4, 8, 384, true, 1, launch_tmq_2x4x8},
    {"tmqb_2x4x8", 1, 2, 4, 8, 384, true, 4, launch_tmqb_2x4x8},
};

int kernel_count() { return (int)(sizeof(kKernels) / sizeof(kKernels[0])); }
const KernelInfo &kernel_info(int id) { return kKernels[id]; }

}  // namespace wd
