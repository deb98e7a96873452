// wd_clover.cu — on-device construction of the self-coupling matrix S(x).
//
//   S(x) = (m0+4) I12 - csw/32 sum_{(mu,nu) in D^2} (gamma_mu gamma_nu) (x) (Q_mu_nu(x) - Q_nu_mu(x))
// (eq. 2.5) with the clover leaves Q_mu_nu of eq. 1.12.  Since
// Q_nu_mu = Q_mu_nu^H leaf by leaf and gamma_nu gamma_mu = -gamma_mu gamma_nu, the 16 ordered
// pairs collapse to the six planes mu < nu (R8):
//   S = (m0+4) I - csw/16 sum_{mu<nu} (gamma_mu gamma_nu) (x) (Q_mu_nu - Q_mu_nu^H).
// Run once per gauge field ("calculated once"), but 60 3x3 products per site are 9 ms of FP64 at 64^4 even at
// the pipe's peak, so it is written to keep the pipe busy:
//   * one thread per (site, plane): a block is 32 consecutive sites x the six planes mu < nu (six warps, the plane is
//     warp-uniform and a template parameter).  A thread holds one plane's products (about 100 registers instead of 255 and a
//     spill for all six), so four times as many warps hide the latency of the link loads;
//   * the six F_mu_nu of a site meet in shared memory; the same 192 threads then assemble the 36 stored slots of S (the
//     real diagonals and strict upper triangles of the two 6x6 blocks: S is Hermitian), six slots each, with the
//     gamma_mu gamma_nu pattern resolved at compile time;
//   * only F = Q - Q^H is needed and F = X - X^H for X = l1 + l2 - l3^H - l4^H (l1..l4 the four leaves of eq. 1.12 in the
//     paper's order): l1 and l4^H both start with U_mu(x), l2 and l3^H both end with U_mu(x-mu), so
//         l1 - l4^H = U_mu(x) [ U_nu(x+mu) U_mu(x+nu)^H U_nu(x)^H - U_nu(x-nu+mu)^H U_mu(x-nu)^H U_nu(x-nu) ]
//         l2 - l3^H = [ U_nu(x) U_mu(x-mu+nu)^H U_nu(x-mu)^H - U_nu(x-nu)^H U_mu(x-mu-nu)^H U_nu(x-mu-nu) ] U_mu(x-mu)
//     — ten 3x3 products and twelve link loads per plane instead of twelve and sixteen.  Pure algebra: no unitarity is
//     assumed (links are general 3x3 matrices, R11).
#include "wd_internal.h"
#include "wd_math.cuh"

namespace wd {

struct M3 { cd m[3][3]; };

__device__ __forceinline__ static M3 m3_load(const cd *__restrict__ U, long long V, int mu, long long i) {
    M3 a;
#pragma unroll
    for (int k = 0; k < 9; k++) a.m[k / 3][k % 3] = __ldg(U + (long long)(mu * 9 + k) * V + i);
    return a;
}
// op(a) op(b) with op = ^H where the flag is set: the conjugate transposes are index swaps and sign flips of the FMAs
template <bool DA, bool DB> __device__ __forceinline__ static M3 m3_mul(const M3 &a, const M3 &b) {
    M3 r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            double re = 0.0, im = 0.0;
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const cd x = DA ? a.m[k][i] : a.m[i][k], y = DB ? b.m[j][k] : b.m[k][j];
                const double xi = DA ? -x.y : x.y, yi = DB ? -y.y : y.y;
                re = fma(x.x, y.x, re);
                re = fma(-xi, yi, re);
                im = fma(x.x, yi, im);
                im = fma(xi, y.x, im);
            }
            r.m[i][j] = make_double2(re, im);
        }
    return r;
}
__device__ __forceinline__ static M3 m3_sub(const M3 &a, const M3 &b) {
    M3 r;
#pragma unroll
    for (int k = 0; k < 9; k++) r.m[k / 3][k % 3] = make_double2(a.m[k / 3][k % 3].x - b.m[k / 3][k % 3].x, a.m[k / 3][k % 3].y - b.m[k / 3][k % 3].y);
    return r;
}

// gamma_mu as (column, power of i) per row — the table of wd_math.cuh (Gam<MU, S>) as constexpr functions of loop indices
// that unrolling makes constant:  col: T,Z {2,3,0,1}; Y,X {3,2,1,0}.  k: T {0,0,0,0}; Z {1,3,3,1}; Y {0,2,2,0}; X {1,1,3,3}
__host__ __device__ constexpr int gam_col(int mu, int s) { return (mu < 2) ? (s ^ 2) : (3 - s); }
__host__ __device__ constexpr int gam_k(int mu, int s) {
    return mu == 0 ? 0 : mu == 1 ? ((s == 0 || s == 3) ? 1 : 3) : mu == 2 ? ((s == 0 || s == 3) ? 0 : 2) : (s < 2 ? 1 : 3);
}
static_assert(gam_col(1, 0) == Gam<1, 0>::col && gam_col(2, 1) == Gam<2, 1>::col && gam_col(3, 3) == Gam<3, 3>::col && gam_col(0, 2) == Gam<0, 2>::col, "gamma table");
static_assert(gam_k(1, 1) == Gam<1, 1>::k && gam_k(1, 3) == Gam<1, 3>::k && gam_k(2, 2) == Gam<2, 2>::k && gam_k(2, 3) == Gam<2, 3>::k && gam_k(3, 1) == Gam<3, 1>::k && gam_k(3, 2) == Gam<3, 2>::k, "gamma table");

struct CloverParams {
    double2 *S;
    const double2 *U;
    long long V, Vs;
    int n[4], stride[4];
    double mass, csw;
};

constexpr int tri(int r, int q) { return r * (11 - r) / 2 + (q - r - 1); }  // (r, q), r < q, in the row-major strict upper triangle of a 6x6 block
constexpr int tri_row(int k) { return k < 5 ? 0 : k < 9 ? 1 : k < 12 ? 2 : k < 14 ? 3 : 4; }
constexpr int tri_col(int k) { return k - tri(tri_row(k), tri_row(k) + 1) + tri_row(k) + 1; }
static_assert(tri(0, 1) == 0 && tri(0, 5) == 4 && tri(1, 2) == 5 && tri(4, 5) == 14 && tri_row(11) == 2 && tri_col(11) == 5 && tri_col(0) == 1 && tri_col(14) == 5, "triangle order");
// the six planes mu < nu
constexpr int plane_mu(int q) { return q < 3 ? 0 : q < 5 ? 1 : 2; }
constexpr int plane_nu(int q) { return q < 3 ? q + 1 : q < 5 ? q - 1 : 3; }

struct Site {
    long long i;
    int c[4];
};
// x + s*mu (s = +-1) with periodic wrap; mu is a run-time value, so the coordinate is picked with selects (indexing c[]
// with it would put the array in local memory)
__device__ __forceinline__ static Site hop(const CloverParams &p, const Site &x, int mu, int s) {
    const int cm = (mu == 0) ? x.c[0] : (mu == 1) ? x.c[1] : (mu == 2) ? x.c[2] : x.c[3];
    const int n = p.n[mu];
    const long long st = p.stride[mu];
    const bool w = (s > 0) ? (cm + 1 == n) : (cm == 0);
    const int cnew = (s > 0) ? (w ? 0 : cm + 1) : (w ? n - 1 : cm - 1);
    Site y;
    y.i = (s > 0) ? (w ? x.i - (long long)(n - 1) * st : x.i + st) : (w ? x.i + (long long)(n - 1) * st : x.i - st);
#pragma unroll
    for (int d = 0; d < 4; d++) y.c[d] = (d == mu) ? cnew : x.c[d];
    return y;
}

constexpr int kCloverSites = 32;  // sites per block: 6 warps, warp q computes plane q of the 32 sites

// F_{MU NU}(x) = X - X^H, entry (a, e) in sF[3 a + e]
// (MU, NU are run-time values on purpose: the six warps of a block then run ONE copy of these ten unrolled products.  As
// template parameters they made six copies, and the kernel spent most of its time waiting for instruction fetches.)
__device__ __forceinline__ static void plane_F(const CloverParams &p, const Site &x, const int MU, const int NU, cd *__restrict__ sF) {
    const cd *U = p.U;
    const long long V = p.Vs;  // component stride
    const Site xpm = hop(p, x, MU, +1), xpn = hop(p, x, NU, +1), xmm = hop(p, x, MU, -1), xmn = hop(p, x, NU, -1);
    const Site xmnpm = hop(p, xmn, MU, +1), xmmpn = hop(p, xmm, NU, +1), xmmmn = hop(p, xmm, NU, -1);
    M3 X;
    {   // U_mu(x) [ U_nu(x+mu) U_mu(x+nu)^H U_nu(x)^H - U_nu(x-nu+mu)^H U_mu(x-nu)^H U_nu(x-nu) ]
        const M3 a = m3_mul<false, true>(m3_mul<false, true>(m3_load(U, V, NU, xpm.i), m3_load(U, V, MU, xpn.i)), m3_load(U, V, NU, x.i));
        const M3 b = m3_mul<false, false>(m3_mul<true, true>(m3_load(U, V, NU, xmnpm.i), m3_load(U, V, MU, xmn.i)), m3_load(U, V, NU, xmn.i));
        X = m3_mul<false, false>(m3_load(U, V, MU, x.i), m3_sub(a, b));
    }
    {   // [ U_nu(x) U_mu(x-mu+nu)^H U_nu(x-mu)^H - U_nu(x-nu)^H U_mu(x-mu-nu)^H U_nu(x-mu-nu) ] U_mu(x-mu)
        const M3 a = m3_mul<false, true>(m3_mul<false, true>(m3_load(U, V, NU, x.i), m3_load(U, V, MU, xmmpn.i)), m3_load(U, V, NU, xmm.i));
        const M3 b = m3_mul<false, false>(m3_mul<true, true>(m3_load(U, V, NU, xmn.i), m3_load(U, V, MU, xmmmn.i)), m3_load(U, V, NU, xmmmn.i));
        const M3 y = m3_mul<false, false>(m3_sub(a, b), m3_load(U, V, MU, xmm.i));
#pragma unroll
        for (int k = 0; k < 9; k++) X.m[k / 3][k % 3] = make_double2(X.m[k / 3][k % 3].x + y.m[k / 3][k % 3].x, X.m[k / 3][k % 3].y + y.m[k / 3][k % 3].y);
    }
#pragma unroll
    for (int a = 0; a < 3; a++)
#pragma unroll
        for (int e = 0; e < 3; e++) sF[3 * a + e] = make_double2(X.m[a][e].x - X.m[e][a].x, X.m[a][e].y + X.m[e][a].y);
}

// Entry (row, col), row <= col, of block B of  S = mass - csw/16 sum_planes (gamma_mu gamma_nu) (x) F:
// (gamma_mu gamma_nu)_{s,s2} = i^(k_mu(s) + k_nu(col_mu(s))) at s2 = col_nu(col_mu(s)), which lies in the chirality block of s
template <int B, int ROW, int COL> __device__ __forceinline__ static cd block_entry(const cd *__restrict__ sF, double mass, double w) {
    constexpr int s = 2 * B + ROW / 3, s2 = 2 * B + COL / 3, a = ROW % 3, e = COL % 3;
    cd v = make_double2((ROW == COL) ? mass : 0.0, 0.0);
#pragma unroll
    for (int q = 0; q < 6; q++) {
        const int mu = plane_mu(q), nu = plane_nu(q), s1 = gam_col(mu, s);
        if (gam_col(nu, s1) != s2) continue;
        const int k = (gam_k(mu, s) + gam_k(nu, s1)) & 3;
        const cd f = sF[(q * 9 + 3 * a + e) * kCloverSites];
        const cd t = (k == 0) ? make_double2(f.x, f.y) : (k == 1) ? make_double2(-f.y, f.x) : (k == 2) ? make_double2(-f.x, -f.y) : make_double2(f.y, -f.x);
        v.x = fma(w, t.x, v.x);
        v.y = fma(w, t.y, v.y);
    }
    return v;
}

// six of the 36 slots of a site (wd_internal.h: per block three real diagonal pairs, then the 15 strict-upper entries)
template <int G> __device__ __forceinline__ static void assemble(const CloverParams &p, const cd *__restrict__ sF, long long i) {
    constexpr int B = G / 3, J0 = 6 * (G % 3);
    const double w = -p.csw / 16.0;
    double2 *S = p.S + i;
    const long long V = p.Vs;
#define WD_SLOT(JJ)                                                                                                  \
    {                                                                                                                \
        constexpr int J = J0 + JJ;                                                                                   \
        if constexpr (J < 3) {                                                                                       \
            S[(long long)slot_diag(B, J) * V] = make_double2(block_entry<B, 2 * J, 2 * J>(sF, p.mass, w).x,          \
                                                             block_entry<B, 2 * J + 1, 2 * J + 1>(sF, p.mass, w).x); \
        } else {                                                                                                     \
            constexpr int K = J - 3;                                                                                 \
            S[(long long)slot_off(B, K) * V] = block_entry<B, tri_row(K), tri_col(K)>(sF, p.mass, w);                \
        }                                                                                                            \
    }
    WD_SLOT(0) WD_SLOT(1) WD_SLOT(2) WD_SLOT(3) WD_SLOT(4) WD_SLOT(5)
#undef WD_SLOT
}

__global__ void __launch_bounds__(6 * kCloverSites, 2) k_build_clover(const CloverParams p) {
    __shared__ cd sF[6 * 9 * kCloverSites];
    const int lane = threadIdx.x & 31, q = threadIdx.x >> 5;  // site of the block; plane, then slot group
    Site x;
    x.i = (long long)blockIdx.x * kCloverSites + lane;
    const bool live = x.i < p.V;
    if (live) {
        long long r = x.i;
        x.c[3] = (int)(r % p.n[3]); r /= p.n[3];
        x.c[2] = (int)(r % p.n[2]); r /= p.n[2];
        x.c[1] = (int)(r % p.n[1]); r /= p.n[1];
        x.c[0] = (int)r;
        cd *f = sF + q * 9 * kCloverSites + lane;  // entry k of this thread at f[k * 32]
        cd mine[9];
        plane_F(p, x, plane_mu(q), plane_nu(q), mine);  // warp-uniform
#pragma unroll
        for (int k = 0; k < 9; k++) f[k * kCloverSites] = mine[k];
    }
    __syncthreads();
    if (!live) return;
    switch (q) {
    case 0: assemble<0>(p, sF + lane, x.i); break;
    case 1: assemble<1>(p, sF + lane, x.i); break;
    case 2: assemble<2>(p, sF + lane, x.i); break;
    case 3: assemble<3>(p, sF + lane, x.i); break;
    case 4: assemble<4>(p, sF + lane, x.i); break;
    default: assemble<5>(p, sF + lane, x.i); break;
    }
}

cudaError_t launch_build_clover(double2 *S_slots, const double2 *U, const int n[4], long long V, long long Vs,
                                double mass, double csw, cudaStream_t st) {
    CloverParams p;
    p.S = S_slots;
    p.U = U;
    p.V = V;
    p.Vs = Vs;
    for (int a = 0; a < 4; a++) p.n[a] = n[a];
    p.stride[3] = 1;
    p.stride[2] = n[3];
    p.stride[1] = n[3] * n[2];
    p.stride[0] = n[3] * n[2] * n[1];
    p.mass = mass;
    p.csw = csw;
    k_build_clover<<<(unsigned)((V + kCloverSites - 1) / kCloverSites), 6 * kCloverSites, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace wd
