// wd_clover.cu — on-device construction of the self-coupling matrix S(x).
//
//   S(x) = (m0+4) I12 - csw/32 sum_{(mu,nu) in D^2} (gamma_mu gamma_nu) (x) (Q_mu_nu(x) - Q_nu_mu(x))
// (eq. 2.5) with the clover leaves Q_mu_nu of eq. 1.12.  Since
// Q_nu_mu = Q_mu_nu^H leaf by leaf and gamma_nu gamma_mu = -gamma_mu gamma_nu, the 16 ordered
// pairs collapse to the six planes mu < nu (R8):
//   S = (m0+4) I - csw/16 sum_{mu<nu} (gamma_mu gamma_nu) (x) (Q_mu_nu - Q_mu_nu^H).
// One thread per site; run once per gauge field, not on the hot path ("calculated once",
// PAPER.md:449), so it is written for clarity: the two 6x6 blocks are accumulated in local memory.
#include "wd_internal.h"
#include "wd_math.cuh"

namespace wd {

struct M3 { cd m[3][3]; };

__device__ static M3 m3_load(const cd *__restrict__ U, long long V, int mu, long long i) {
    M3 a;
#pragma unroll
    for (int k = 0; k < 9; k++) a.m[k / 3][k % 3] = U[(long long)(mu * 9 + k) * V + i];
    return a;
}
__device__ static M3 m3_dag(const M3 &a) {
    M3 r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) r.m[i][j] = make_double2(a.m[j][i].x, -a.m[j][i].y);
    return r;
}
__device__ static M3 m3_mul(const M3 &a, const M3 &b) {
    M3 r;
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            cd s = cmul(a.m[i][0], b.m[0][j]);
            cfma(s, a.m[i][1], b.m[1][j]);
            cfma(s, a.m[i][2], b.m[2][j]);
            r.m[i][j] = s;
        }
    return r;
}

// gamma_mu as (column, power of i) per row — the same table as wd_math.cuh, in runtime form.
__constant__ int c_gcol[4][4] = {{2, 3, 0, 1}, {2, 3, 0, 1}, {3, 2, 1, 0}, {3, 2, 1, 0}};
__constant__ int c_gk[4][4] = {{0, 0, 0, 0}, {1, 3, 3, 1}, {0, 2, 2, 0}, {1, 1, 3, 3}};

__device__ static long long shift(long long i, const int n[4], const int stride[4], const int c[4], int mu, int s) {
    // site index of x + s*mu (s = +-1) with periodic wrap
    if (s > 0) return (c[mu] + 1 < n[mu]) ? i + stride[mu] : i - (long long)(n[mu] - 1) * stride[mu];
    return (c[mu] > 0) ? i - stride[mu] : i + (long long)(n[mu] - 1) * stride[mu];
}

struct CloverParams {
    double2 *S;
    const double2 *U;
    long long V, Vs;
    int n[4], stride[4];
    double mass, csw;
};

__global__ void __launch_bounds__(128) k_build_clover(const CloverParams p) {
    const long long i = (long long)blockIdx.x * 128 + threadIdx.x;
    if (i >= p.V) return;
    int c[4];
    {
        long long r = i;
        c[3] = (int)(r % p.n[3]); r /= p.n[3];
        c[2] = (int)(r % p.n[2]); r /= p.n[2];
        c[1] = (int)(r % p.n[1]); r /= p.n[1];
        c[0] = (int)r;
    }
    cd blk[2][6][6];
    for (int b = 0; b < 2; b++)
        for (int r = 0; r < 6; r++)
            for (int q = 0; q < 6; q++) blk[b][r][q] = make_double2((r == q) ? p.mass : 0.0, 0.0);

    const cd *U = p.U;
    const long long V = p.Vs;  // component stride
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            int cm[4] = {c[0], c[1], c[2], c[3]};  // coordinates of x - mu
            cm[mu] = (c[mu] > 0) ? c[mu] - 1 : p.n[mu] - 1;
            int cn[4] = {c[0], c[1], c[2], c[3]};  // coordinates of x - nu
            cn[nu] = (c[nu] > 0) ? c[nu] - 1 : p.n[nu] - 1;
            const long long xpm = shift(i, p.n, p.stride, c, mu, +1);
            const long long xpn = shift(i, p.n, p.stride, c, nu, +1);
            const long long xmm = shift(i, p.n, p.stride, c, mu, -1);
            const long long xmn = shift(i, p.n, p.stride, c, nu, -1);
            const long long xmmpn = shift(xmm, p.n, p.stride, cm, nu, +1);
            const long long xmmmn = shift(xmm, p.n, p.stride, cm, nu, -1);
            const long long xmnpm = shift(xmn, p.n, p.stride, cn, mu, +1);
            // the four leaves of eq. 1.12
            M3 q = m3_mul(m3_mul(m3_load(U, V, mu, i), m3_load(U, V, nu, xpm)),
                          m3_mul(m3_dag(m3_load(U, V, mu, xpn)), m3_dag(m3_load(U, V, nu, i))));
            M3 l = m3_mul(m3_mul(m3_load(U, V, nu, i), m3_dag(m3_load(U, V, mu, xmmpn))),
                          m3_mul(m3_dag(m3_load(U, V, nu, xmm)), m3_load(U, V, mu, xmm)));
            for (int a = 0; a < 9; a++) { q.m[a / 3][a % 3].x += l.m[a / 3][a % 3].x; q.m[a / 3][a % 3].y += l.m[a / 3][a % 3].y; }
            l = m3_mul(m3_mul(m3_dag(m3_load(U, V, mu, xmm)), m3_dag(m3_load(U, V, nu, xmmmn))),
                       m3_mul(m3_load(U, V, mu, xmmmn), m3_load(U, V, nu, xmn)));
            for (int a = 0; a < 9; a++) { q.m[a / 3][a % 3].x += l.m[a / 3][a % 3].x; q.m[a / 3][a % 3].y += l.m[a / 3][a % 3].y; }
            l = m3_mul(m3_mul(m3_dag(m3_load(U, V, nu, xmn)), m3_load(U, V, mu, xmn)),
                       m3_mul(m3_load(U, V, nu, xmnpm), m3_dag(m3_load(U, V, mu, i))));
            for (int a = 0; a < 9; a++) { q.m[a / 3][a % 3].x += l.m[a / 3][a % 3].x; q.m[a / 3][a % 3].y += l.m[a / 3][a % 3].y; }
            // F = Q - Q^H
            M3 F;
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++)
                    F.m[a][b] = make_double2(q.m[a][b].x - q.m[b][a].x, q.m[a][b].y + q.m[b][a].y);
            // (gamma_mu gamma_nu)_{s,s2} = i^(k_mu(s) + k_nu(col_mu(s))) at s2 = col_nu(col_mu(s))
            const double w = -p.csw / 16.0;
            for (int s = 0; s < 4; s++) {
                const int s1 = c_gcol[mu][s];
                const int s2 = c_gcol[nu][s1];
                const int k = (c_gk[mu][s] + c_gk[nu][s1]) & 3;
                const int b = s >> 1;  // s2 lies in the same chirality block as s
                for (int a = 0; a < 3; a++)
                    for (int e = 0; e < 3; e++) {
                        const cd f = F.m[a][e];
                        cd v;
                        if (k == 0) v = make_double2(f.x, f.y);
                        else if (k == 1) v = make_double2(-f.y, f.x);
                        else if (k == 2) v = make_double2(-f.x, -f.y);
                        else v = make_double2(f.y, -f.x);
                        cd &dst = blk[b][3 * (s & 1) + a][3 * (s2 & 1) + e];
                        dst.x = fma(w, v.x, dst.x);
                        dst.y = fma(w, v.y, dst.y);
                    }
            }
        }
    // store the 36 slots (wd_internal.h): real diagonal pairs, then the strict upper triangles
    for (int j = 0; j < 6; j++) {
        const int b = j / 3, r = 2 * (j % 3);
        p.S[(long long)slot_diag(b, j % 3) * V + i] = make_double2(blk[b][r][r].x, blk[b][r + 1][r + 1].x);
    }
    for (int b = 0; b < 2; b++) {
        int k = 0;
        for (int r = 0; r < 6; r++)
            for (int q2 = r + 1; q2 < 6; q2++, k++) p.S[(long long)slot_off(b, k) * V + i] = blk[b][r][q2];
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
    k_build_clover<<<(unsigned)((V + 127) / 128), 128, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace wd
