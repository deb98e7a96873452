// wd_smem_ops.cuh — per-site arithmetic of the TMA kernels with operands in shared memory (SoA boxes
// [component][site], one complex double per 16-byte element): the two hops of one direction, and half of
// a 6x6 Hermitian block of S folded into the accumulator.  Used by wd_tmb.cu and wd_tmr.cu.
#pragma once
#include <stdint.h>

#include "wd_math.cuh"

namespace wd {

// ---------------------------------------------------------------- shared-memory operand fetch
template <class C = cd> __device__ __forceinline__ C lds(const unsigned char *smem, uint32_t off) {
    return *reinterpret_cast<const C *>(smem + off);
}

// One direction MU != T of the stencil for the thread's site: both hops, operands from shared
// memory.  (base, stride) pairs select interior or face storage per thread (no divergence: both
// are shared-memory addresses).
// One link from a shared-memory SoA box into registers.  UC = 9: all nine entries.  UC = 6 (two-row storage): rows 0
// and 1 are loaded, row 2 = conj(row 0 x row 1), which holds for every SU(3) matrix (unitary, determinant 1).
template <int UC, class C = cd> __device__ __forceinline__ void load_link(C u[9], const unsigned char *smem, uint32_t off, uint32_t stride) {
#pragma unroll
    for (int k = 0; k < UC; k++) u[k] = lds<C>(smem, off + k * stride);
    if (UC == 6) {
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const C a = u[(k + 1) % 3], b = u[3 + (k + 2) % 3], c = u[(k + 2) % 3], d = u[3 + (k + 1) % 3];
            // conj(a b - c d)
            u[6 + k] = mk<C>(fma(a.x, b.x, -a.y * b.y) - fma(c.x, d.x, -c.y * d.y),
                             -(fma(a.x, b.y, a.y * b.x) - fma(c.x, d.y, c.y * d.x)));
        }
    }
}

// fwd / bwd = false: that hop crosses an open boundary of a domain-decomposed sub-lattice and is left out here (the
// exterior kernel of wd_dd.cu adds it from the neighbour's half-spinor); always true on a periodic lattice.
template <int MU, int UC = 9, class C = cd>
__device__ __forceinline__ void hop_pair_smem(C acc[12], const unsigned char *smem, uint32_t u_own, uint32_t u_own_stride,
                                              uint32_t pf, uint32_t pf_stride, uint32_t ub, uint32_t ub_stride,
                                              uint32_t pb, uint32_t pb_stride, bool fwd = true, bool bwd = true) {
    C p[12], u[9];
    if (fwd) {
        load_link<UC, C>(u, smem, u_own, u_own_stride);
#pragma unroll
        for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, pf + c * pf_stride);
        hop_term<MU, -1>(acc, p, u);
    }
    if (bwd) {
        load_link<UC, C>(u, smem, ub, ub_stride);
#pragma unroll
        for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, pb + c * pb_stride);
        hop_term<MU, +1>(acc, p, u);
    }
}

// acc[0..5] += (part of B) q for one 6x6 Hermitian block B.  H = 0: the 6 real diagonal entries (slots
// 0..2, as pairs) and strict-upper entries 0..5 (slots 3..8); H = 1: strict-upper entries 6..14 (slots
// 0..8).  q is the block's half of psi already scaled by -2 (out = S psi - 1/2 hops = -1/2 (hops - 2 S psi)).
template <int H>
__device__ __forceinline__ void herm6_half_add(cd acc[6], const unsigned char *smem, uint32_t so, uint32_t stride,
                                               const cd q[6]) {
    cd a[9];
#pragma unroll
    for (int k = 0; k < 9; k++) a[k] = lds(smem, so + k * stride);
    if (H == 0) {
#pragma unroll
        for (int i = 0; i < 3; i++) {
            acc[2 * i].x = fma(a[i].x, q[2 * i].x, acc[2 * i].x);
            acc[2 * i].y = fma(a[i].x, q[2 * i].y, acc[2 * i].y);
            acc[2 * i + 1].x = fma(a[i].y, q[2 * i + 1].x, acc[2 * i + 1].x);
            acc[2 * i + 1].y = fma(a[i].y, q[2 * i + 1].y, acc[2 * i + 1].y);
        }
    }
    int k = 0;
#pragma unroll
    for (int i = 0; i < 6; i++)
#pragma unroll
        for (int j = i + 1; j < 6; j++, k++) {
            const int slot = (H == 0) ? k + 3 : k - 6;
            if ((H == 0 && k < 6) || (H == 1 && k >= 6)) {
                cfma(acc[i], a[slot], q[j]);
                cfma_conj(acc[j], a[slot], q[i]);
            }
        }
}

}  // namespace wd
