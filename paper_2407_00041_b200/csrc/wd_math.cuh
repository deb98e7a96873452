// wd_math.cuh — per-site arithmetic of the Wilson-clover hot path (device code, FP64).
//
// Steps of SURVEY.md §8(a): a2 spin projection, a3 SU(3) multiply, a4 reconstruct + accumulate,
// a5 self-coupling (two 6x6 Hermitian blocks).  Everything is resolved at compile time: the
// gamma matrices of DESIGN.md R1 have one entry of modulus one per row, so projection and
// reconstruction are adds / swaps only (no multiplies), cf. Listing 4.2.
#pragma once
#include <cuda_runtime.h>

namespace wd {

typedef double2 cd;  // complex double: x = re, y = im (one 16-byte LDG.128 / STG.128)
typedef float2 cf;   // complex float (the FP32 variant): one 8-byte LDG.64 / STG.64

// Everything below is a template on the complex type C (double2 or float2); R<C> is its real type.
template <class C> struct RealOf;
template <> struct RealOf<double2> { typedef double type; };
template <> struct RealOf<float2> { typedef float type; };
template <class C> using R = typename RealOf<C>::type;
template <class C> __host__ __device__ __forceinline__ C mk(R<C> x, R<C> y) {
    C c;
    c.x = x;
    c.y = y;
    return c;
}

// gamma_mu, mu = 0..3 = T,Z,Y,X (R1): (gamma_mu psi)_s = i^GK[mu][s] * psi_{GC[mu][s]}.
//   gamma_T: 0->(2,1)  1->(3,1)  2->(0,1)  3->(1,1)
//   gamma_Z: 0->(2,i)  1->(3,-i) 2->(0,-i) 3->(1,i)
//   gamma_Y: 0->(3,1)  1->(2,-1) 2->(1,-1) 3->(0,1)
//   gamma_X: 0->(3,i)  1->(2,i)  2->(1,-i) 3->(0,-i)
template <int MU, int S> struct Gam;
#define WD_GAM(MU, S, COL, K) \
    template <> struct Gam<MU, S> { static constexpr int col = COL, k = K; };
WD_GAM(0, 0, 2, 0) WD_GAM(0, 1, 3, 0) WD_GAM(0, 2, 0, 0) WD_GAM(0, 3, 1, 0)
WD_GAM(1, 0, 2, 1) WD_GAM(1, 1, 3, 3) WD_GAM(1, 2, 0, 3) WD_GAM(1, 3, 1, 1)
WD_GAM(2, 0, 3, 0) WD_GAM(2, 1, 2, 2) WD_GAM(2, 2, 1, 2) WD_GAM(2, 3, 0, 0)
WD_GAM(3, 0, 3, 1) WD_GAM(3, 1, 2, 1) WD_GAM(3, 2, 1, 3) WD_GAM(3, 3, 0, 3)
#undef WD_GAM

// a + i^K b
template <int K, class C> __device__ __forceinline__ C add_ik(C a, C b) {
    constexpr int k = K & 3;
    if (k == 0) return mk<C>(a.x + b.x, a.y + b.y);
    if (k == 1) return mk<C>(a.x - b.y, a.y + b.x);
    if (k == 2) return mk<C>(a.x - b.x, a.y - b.y);
    return mk<C>(a.x + b.y, a.y - b.x);
}

// r += a * b
template <class C> __device__ __forceinline__ void cfma(C &r, C a, C b) {
    r.x = fma(a.x, b.x, r.x);
    r.y = fma(a.x, b.y, r.y);
    r.x = fma(-a.y, b.y, r.x);
    r.y = fma(a.y, b.x, r.y);
}
// r += conj(a) * b
template <class C> __device__ __forceinline__ void cfma_conj(C &r, C a, C b) {
    r.x = fma(a.x, b.x, r.x);
    r.y = fma(a.x, b.y, r.y);
    r.x = fma(a.y, b.y, r.x);
    r.y = fma(-a.y, b.x, r.y);
}
template <class C> __device__ __forceinline__ C cmul(C a, C b) {
    return mk<C>(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
template <class C> __device__ __forceinline__ C cmul_conj(C a, C b) {  // conj(a) * b
    return mk<C>(fma(a.x, b.x, a.y * b.y), fma(a.x, b.y, -a.y * b.x));
}

// a2: half-spinor h = rows 0,1 of (I4 + SIGN*gamma_MU) psi   (6 of 12 entries)
template <int MU, int SIGN, class C> __device__ __forceinline__ void project(C h[6], const C psi[12]) {
    constexpr int KS = (SIGN < 0) ? 2 : 0;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        h[c] = add_ik<Gam<MU, 0>::k + KS>(psi[c], psi[3 * Gam<MU, 0>::col + c]);
        h[3 + c] = add_ik<Gam<MU, 1>::k + KS>(psi[3 + c], psi[3 * Gam<MU, 1>::col + c]);
    }
}

// a3: g = U h (DAG = false) or g = U^H h (DAG = true) on both colour vectors; u row-major 3x3.
template <bool DAG, class C> __device__ __forceinline__ void su3_mul(C g[6], const C u[9], const C h[6]) {
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            C r;
            if (!DAG) {
                r = cmul(u[3 * c], h[3 * s]);
                cfma(r, u[3 * c + 1], h[3 * s + 1]);
                cfma(r, u[3 * c + 2], h[3 * s + 2]);
            } else {
                r = cmul_conj(u[c], h[3 * s]);
                cfma_conj(r, u[3 + c], h[3 * s + 1]);
                cfma_conj(r, u[6 + c], h[3 * s + 2]);
            }
            g[3 * s + c] = r;
        }
}

// a4: acc += (I4 + SIGN*gamma_MU)-reconstruction of g.  With phi = (1 + SIGN*gamma) psi one has
// gamma phi = SIGN*phi, hence phi_s = SIGN * i^k_s * phi_{col(s)} for the lower rows s = 2,3.
template <int MU, int SIGN, class C> __device__ __forceinline__ void reconstruct_add(C acc[12], const C g[6]) {
    constexpr int KS = (SIGN < 0) ? 2 : 0;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = add_ik<0>(acc[c], g[c]);
        acc[3 + c] = add_ik<0>(acc[3 + c], g[3 + c]);
        acc[6 + c] = add_ik<Gam<MU, 2>::k + KS>(acc[6 + c], g[3 * Gam<MU, 2>::col + c]);
        acc[9 + c] = add_ik<Gam<MU, 3>::k + KS>(acc[9 + c], g[3 * Gam<MU, 3>::col + c]);
    }
}

// The same without an accumulator to start from — a sum that begins with 0 + g costs a DADD per real number (0.0 + x is
// not x in IEEE arithmetic, the compiler keeps it):
//   i^K b
template <int K, class C> __device__ __forceinline__ C mul_ik(C b) {
    constexpr int k = K & 3;
    if (k == 0) return b;
    if (k == 1) return mk<C>(-b.y, b.x);
    if (k == 2) return mk<C>(-b.x, -b.y);
    return mk<C>(b.y, -b.x);
}
//   a + s i^K b, s real: the phase is folded into the sign of s and the choice of operand (no extra instruction)
template <int K, class C> __device__ __forceinline__ C axpy_ik(C a, R<C> s, C b) {
    constexpr int k = K & 3;
    if (k == 0) return mk<C>(fma(s, b.x, a.x), fma(s, b.y, a.y));
    if (k == 1) return mk<C>(fma(-s, b.y, a.x), fma(s, b.x, a.y));
    if (k == 2) return mk<C>(fma(-s, b.x, a.x), fma(-s, b.y, a.y));
    return mk<C>(fma(s, b.y, a.x), fma(-s, b.x, a.y));
}
// acc = (I4 + SIGN*gamma_MU)-reconstruction of g   (the first hop of a sum; bit-identical to 0 + reconstruct_add
// except for the sign of a zero)
template <int MU, int SIGN, class C> __device__ __forceinline__ void reconstruct_set(C acc[12], const C g[6]) {
    constexpr int KS = (SIGN < 0) ? 2 : 0;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = g[c];
        acc[3 + c] = g[3 + c];
        acc[6 + c] = mul_ik<Gam<MU, 2>::k + KS>(g[3 * Gam<MU, 2>::col + c]);
        acc[9 + c] = mul_ik<Gam<MU, 3>::k + KS>(g[3 * Gam<MU, 3>::col + c]);
    }
}
// out = base + s * (I4 + SIGN*gamma_MU)-reconstruction of g, s real   (the last hop of a sum, scaled: out = outp - 1/2 f)
template <int MU, int SIGN, class C>
__device__ __forceinline__ void reconstruct_axpy(C out[12], const C base[12], R<C> s, const C g[6]) {
    constexpr int KS = (SIGN < 0) ? 2 : 0;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        out[c] = axpy_ik<0>(base[c], s, g[c]);
        out[3 + c] = axpy_ik<0>(base[3 + c], s, g[3 + c]);
        out[6 + c] = axpy_ik<Gam<MU, 2>::k + KS>(base[6 + c], s, g[3 * Gam<MU, 2>::col + c]);
        out[9 + c] = axpy_ik<Gam<MU, 3>::k + KS>(base[9 + c], s, g[3 * Gam<MU, 3>::col + c]);
    }
}

// One hopping term: acc += [(I4 + SIGN*gamma_MU) (x) W] psi,  W = U (SIGN = -1, forward
// neighbour) or U^H (SIGN = +1, backward neighbour)   — eq. 1.13 lines 2 and 3 without the -1/2.
template <int MU, int SIGN, class C> __device__ __forceinline__ void hop_term(C acc[12], const C psi[12], const C u[9]) {
    C h[6], g[6];
    project<MU, SIGN>(h, psi);
    su3_mul<(SIGN > 0)>(g, u, h);
    reconstruct_add<MU, SIGN>(acc, g);
}

// a5: r = B p for one 6x6 Hermitian block: d = 6 real diagonal entries, a = 15 strict-upper
// entries row-major (R6).  2*(6 real x cplx + 30 cmul) per site = 504 flop.
template <class C> __device__ __forceinline__ void herm6_mul(C r[6], const R<C> d[6], const C a[15], const C p[6]) {
#pragma unroll
    for (int i = 0; i < 6; i++) r[i] = mk<C>(d[i] * p[i].x, d[i] * p[i].y);
    int k = 0;
#pragma unroll
    for (int i = 0; i < 6; i++)
#pragma unroll
        for (int j = i + 1; j < 6; j++, k++) {
            cfma(r[i], a[k], p[j]);
            cfma_conj(r[j], a[k], p[i]);
        }
}

}  // namespace wd
