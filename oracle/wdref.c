/* oracle/wdref.c — CPU ORACLE for the Wilson(-clover) Dirac operator.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct restatement of what the hot path computes,
 * written from the paper (arxiv 2407.00041, /root/reference/PAPER.md), in FP64 complex, with
 * generic 4x4 gamma tables and full 12-component loops: no half-spinor trick, no 6x6 block
 * trick, no blocking, no fusion.  It shares NO code with the CUDA library (paper_2407_00041_b200/)
 * and must never be imported, linked or executed by the product path; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * What it follows:
 *   wdref_apply          eq. 1.13 term by term, a = 1 (R3),
 *                        = D_sc psi - D_nc psi of eqs. 2.5-2.7
 *   wdref_build_clover   eq. 2.5 self-coupling matrix, with Q_mu_nu of
 *                        eq. 1.12 — the four plaquette leaves as printed
 *   wdref_dense          the same eq. 1.13 assembled as a dense matrix out of Kronecker
 *                        products (A (x) B)_{(s,c),(s',c')} = A_ss' B_cc'
 *   gamma tables         DESIGN.md R1 (the paper never prints them: PAPER.md:134,556)
 *
 * Conventions (R1-R12): directions mu = 0..3 = T,Z,Y,X; site index
 * i = ((t*Z+z)*Y+y)*X+x, 0-based; periodic in all four directions; spinor
 * component index 3*spin + colour; links row-major 3x3, forward links of the own
 * site only, [site][mu][9]; self-coupling 42 entries per site:
 * 12 real diagonal entries, then the strict upper triangle (row-major) of the spin-{0,1} 6x6
 * block, then of the spin-{2,3} block; it INCLUDES the (m0+4) diagonal (eq. 2.5).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): free-field plane-wave closed form,
 * gamma5-hermiticity, gauge covariance, dense brute force on 2^4 and 2x4x2x4, constant abelian
 * flux closed form for the clover term, structure of S, linearity / multi-RHS, translation
 * covariance, csw -> 0.  PARITY UNPINNED (paper silent, DDalphaAMG source and [Fro+14] not
 * available): the choice of gamma basis, the order of the 42 entries and the site enumeration
 * relative to DDalphaAMG's.  Every pin holds for any valid choice of those.
 */
#include "wdref.h"

#include <complex.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* ---- gamma matrices (R1): chiral basis, gamma_mu = [[0, a_mu], [a_mu^H, 0]] in 2x2
 * blocks with a_T = 1, a_Z = i sigma_3, a_Y = i sigma_2, a_X = i sigma_1. ------------------- */
void wdref_gamma(int mu, double *g_out /* [4][4][2] */) {
    cplx a[2][2];
    switch (mu) {
    case 0: a[0][0] = 1; a[0][1] = 0;  a[1][0] = 0;  a[1][1] = 1;  break;
    case 1: a[0][0] = I; a[0][1] = 0;  a[1][0] = 0;  a[1][1] = -I; break;
    case 2: a[0][0] = 0; a[0][1] = 1;  a[1][0] = -1; a[1][1] = 0;  break;
    default: a[0][0] = 0; a[0][1] = I; a[1][0] = I;  a[1][1] = 0;  break;
    }
    cplx g[4][4];
    memset(g, 0, sizeof g);
    for (int r = 0; r < 2; r++)
        for (int c = 0; c < 2; c++) {
            g[r][2 + c] = a[r][c];
            g[2 + r][c] = conj(a[c][r]);
        }
    for (int r = 0; r < 4; r++)
        for (int c = 0; c < 4; c++) {
            g_out[2 * (4 * r + c)] = creal(g[r][c]);
            g_out[2 * (4 * r + c) + 1] = cimag(g[r][c]);
        }
}

static void gamma_c(int mu, cplx g[4][4]) {
    double t[32];
    wdref_gamma(mu, t);
    for (int k = 0; k < 16; k++) g[k / 4][k % 4] = t[2 * k] + I * t[2 * k + 1];
}

/* ---- lattice indexing ------------------------------------------------------------------- */
typedef struct { int n[4]; } dims_t;

static inline int64_t site_index(const dims_t *d, const int c[4]) {
    return (((int64_t)c[0] * d->n[1] + c[1]) * d->n[2] + c[2]) * d->n[3] + c[3];
}
static inline void site_coords(const dims_t *d, int64_t i, int c[4]) {
    c[3] = (int)(i % d->n[3]); i /= d->n[3];
    c[2] = (int)(i % d->n[2]); i /= d->n[2];
    c[1] = (int)(i % d->n[1]); i /= d->n[1];
    c[0] = (int)i;
}
/* x + s1*mu + s2*nu with periodic identification */
static inline int64_t shifted(const dims_t *d, int64_t i, int mu, int s1, int nu, int s2) {
    int c[4];
    site_coords(d, i, c);
    c[mu] = ((c[mu] + s1) % d->n[mu] + d->n[mu]) % d->n[mu];
    if (nu >= 0) c[nu] = ((c[nu] + s2) % d->n[nu] + d->n[nu]) % d->n[nu];
    return site_index(d, c);
}

static inline const cplx *link(const double *U, int64_t i, int mu) {
    return (const cplx *)U + (i * 4 + mu) * 9;
}

/* Expand the 42 stored entries of one site into the full Hermitian 12x12 S (R6). */
static void expand_selfcoupling(const cplx *c42, cplx S[12][12]) {
    memset(S, 0, sizeof(cplx) * 144);
    for (int k = 0; k < 12; k++) S[k][k] = creal(c42[k]);
    for (int b = 0; b < 2; b++) {
        int k = 12 + 15 * b;
        for (int r = 0; r < 6; r++)
            for (int c = r + 1; c < 6; c++, k++) {
                S[6 * b + r][6 * b + c] = c42[k];
                S[6 * b + c][6 * b + r] = conj(c42[k]);
            }
    }
}

/* ---- eq. 1.13, a = 1 ------------------------------------------------- */
/* One site: acc = S(x) psi(x) - 1/2 sum_mu [...]; S == NULL means S = (m0+4) I. */
static void apply_site(const dims_t *d, double m0, const double *U, cplx (*S)[12], const cplx *psi,
                       int64_t x, cplx gam[4][4][4], cplx acc[12]) {
    /* first line of eq. 1.13: the self-coupling term S(x) psi(x) */
    if (S) {
        for (int i = 0; i < 12; i++) {
            cplx s = 0;
            for (int j = 0; j < 12; j++) s += S[i][j] * psi[x * 12 + j];
            acc[i] = s;
        }
    } else {
        for (int i = 0; i < 12; i++) acc[i] = (m0 + 4.0) * psi[x * 12 + i];
    }
    for (int mu = 0; mu < 4; mu++) {
        const int64_t xp = shifted(d, x, mu, +1, -1, 0);
        const int64_t xm = shifted(d, x, mu, -1, -1, 0);
        const cplx *Uf = link(U, x, mu);  /* U_mu(x)     */
        const cplx *Ub = link(U, xm, mu); /* U_mu(x-mu)  */
        cplx fw[4][3], bw[4][3];
        for (int s = 0; s < 4; s++)
            for (int c = 0; c < 3; c++) {
                cplx f = 0, b = 0;
                for (int k = 0; k < 3; k++) {
                    f += Uf[3 * c + k] * psi[xp * 12 + 3 * s + k];       /* U psi(x+mu)   */
                    b += conj(Ub[3 * k + c]) * psi[xm * 12 + 3 * s + k]; /* U^H psi(x-mu) */
                }
                fw[s][c] = f;
                bw[s][c] = b;
            }
        /* second and third line of eq. 1.13 */
        for (int s = 0; s < 4; s++)
            for (int c = 0; c < 3; c++) {
                cplx f = 0, b = 0;
                for (int sp = 0; sp < 4; sp++) {
                    cplx delta = (s == sp) ? 1.0 : 0.0;
                    f += (delta - gam[mu][s][sp]) * fw[sp][c];
                    b += (delta + gam[mu][s][sp]) * bw[sp][c];
                }
                acc[3 * s + c] -= 0.5 * f;
                acc[3 * s + c] -= 0.5 * b;
            }
    }
}

int wdref_apply(int T, int Z, int Y, int X, double m0, const double *U, const double *C,
                double *out, const double *in, int nrhs) {
    if (T < 1 || Z < 1 || Y < 1 || X < 1 || !U || !out || !in || nrhs < 1) return -1;
    dims_t d = {{T, Z, Y, X}};
    const int64_t V = (int64_t)T * Z * Y * X;
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_c(mu, gam[mu]);

    for (int r = 0; r < nrhs; r++) {
        const cplx *psi = (const cplx *)in + (int64_t)r * V * 12;
        cplx *eta = (cplx *)out + (int64_t)r * V * 12;
#pragma omp parallel for schedule(static)
        for (int64_t x = 0; x < V; x++) {
            cplx acc[12], S[12][12];
            if (C) expand_selfcoupling((const cplx *)C + x * 42, S);
            apply_site(&d, m0, U, C ? S : NULL, psi, x, gam, acc);
            for (int i = 0; i < 12; i++) eta[x * 12 + i] = acc[i];
        }
    }
    return 0;
}

/* ---- 3x3 helpers for eq. 1.12 ----------------------------------------------------------- */
typedef struct { cplx m[3][3]; } m3;

static m3 m3_load(const cplx *p) {
    m3 a;
    for (int k = 0; k < 9; k++) a.m[k / 3][k % 3] = p[k];
    return a;
}
static m3 m3_dag(m3 a) {
    m3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.m[i][j] = conj(a.m[j][i]);
    return r;
}
static m3 m3_mul(m3 a, m3 b) {
    m3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a.m[i][k] * b.m[k][j];
            r.m[i][j] = s;
        }
    return r;
}
static m3 m3_add(m3 a, m3 b) {
    m3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.m[i][j] = a.m[i][j] + b.m[i][j];
    return r;
}
static m3 m3_sub(m3 a, m3 b) {
    m3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.m[i][j] = a.m[i][j] - b.m[i][j];
    return r;
}

/* Q_mu_nu(x), eq. 1.12, the four leaves in the order printed. */
static m3 clover_leaves(const dims_t *d, const double *U, int64_t x, int mu, int nu) {
#define LK(site, dir) m3_load(link(U, (site), (dir)))
    const int64_t xpm = shifted(d, x, mu, +1, -1, 0);    /* x+mu       */
    const int64_t xpn = shifted(d, x, nu, +1, -1, 0);    /* x+nu       */
    const int64_t xmm = shifted(d, x, mu, -1, -1, 0);    /* x-mu       */
    const int64_t xmn = shifted(d, x, nu, -1, -1, 0);    /* x-nu       */
    const int64_t xmmpn = shifted(d, x, mu, -1, nu, +1); /* x-mu+nu    */
    const int64_t xmmmn = shifted(d, x, mu, -1, nu, -1); /* x-mu-nu    */
    const int64_t xmnpm = shifted(d, x, nu, -1, mu, +1); /* x-nu+mu    */
    m3 l1 = m3_mul(m3_mul(LK(x, mu), LK(xpm, nu)), m3_mul(m3_dag(LK(xpn, mu)), m3_dag(LK(x, nu))));
    m3 l2 = m3_mul(m3_mul(LK(x, nu), m3_dag(LK(xmmpn, mu))), m3_mul(m3_dag(LK(xmm, nu)), LK(xmm, mu)));
    m3 l3 = m3_mul(m3_mul(m3_dag(LK(xmm, mu)), m3_dag(LK(xmmmn, nu))), m3_mul(LK(xmmmn, mu), LK(xmn, nu)));
    m3 l4 = m3_mul(m3_mul(m3_dag(LK(xmn, nu)), LK(xmn, mu)), m3_mul(LK(xmnpm, nu), m3_dag(LK(x, mu))));
#undef LK
    return m3_add(m3_add(l1, l2), m3_add(l3, l4));
}

/* S(x) = (m0+4) I_12 - csw/32 sum_{(mu,nu) in D^2} (gamma_mu gamma_nu) (x) (Q_mu_nu - Q_nu_mu),
 * eq. 2.5, all 16 ordered pairs (R8). */
static void selfcoupling_full(const dims_t *d, double m0, double csw, const double *U, int64_t x,
                              cplx gam[4][4][4], cplx S[12][12]) {
    memset(S, 0, sizeof(cplx) * 144);
    for (int i = 0; i < 12; i++) S[i][i] = m0 + 4.0;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = 0; nu < 4; nu++) {
            m3 F = m3_sub(clover_leaves(d, U, x, mu, nu), clover_leaves(d, U, x, nu, mu));
            cplx gg[4][4];
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    cplx s = 0;
                    for (int k = 0; k < 4; k++) s += gam[mu][a][k] * gam[nu][k][b];
                    gg[a][b] = s;
                }
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++)
                    for (int i = 0; i < 3; i++)
                        for (int j = 0; j < 3; j++)
                            S[3 * a + i][3 * b + j] -= (csw / 32.0) * gg[a][b] * F.m[i][j];
        }
}

int wdref_build_clover_full(int T, int Z, int Y, int X, double m0, double csw, const double *U,
                            double *S_out /* [V][12][12][2] */) {
    if (T < 1 || Z < 1 || Y < 1 || X < 1 || !U || !S_out) return -1;
    dims_t d = {{T, Z, Y, X}};
    const int64_t V = (int64_t)T * Z * Y * X;
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_c(mu, gam[mu]);
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < V; x++) {
        cplx S[12][12];
        selfcoupling_full(&d, m0, csw, U, x, gam, S);
        memcpy((cplx *)S_out + x * 144, S, sizeof S);
    }
    return 0;
}

static void pack_selfcoupling(cplx S[12][12], cplx *c) {
    for (int k = 0; k < 12; k++) c[k] = creal(S[k][k]);
    for (int b = 0; b < 2; b++) {
        int k = 12 + 15 * b;
        for (int r = 0; r < 6; r++)
            for (int cc = r + 1; cc < 6; cc++, k++) c[k] = S[6 * b + r][6 * b + cc];
    }
}

/* Stores the 42 entries of DESIGN.md R6.  Entries outside the two 6x6 blocks and the imaginary
 * parts of the diagonal are dropped (pin P6 checks on wdref_build_clover_full that they vanish);
 * the lower triangle is the conjugate of the upper one (S Hermitian, same pin). */
int wdref_build_clover(int T, int Z, int Y, int X, double m0, double csw, const double *U,
                       double *C /* [V][42][2] */) {
    if (T < 1 || Z < 1 || Y < 1 || X < 1 || !U || !C) return -1;
    dims_t d = {{T, Z, Y, X}};
    const int64_t V = (int64_t)T * Z * Y * X;
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_c(mu, gam[mu]);
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < V; x++) {
        cplx S[12][12];
        selfcoupling_full(&d, m0, csw, U, x, gam, S);
        pack_selfcoupling(S, (cplx *)C + x * 42);
    }
    return 0;
}

/* ---- dense assembly of eq. 1.13 from Kronecker products (tiny lattices only) ------------ */
static void kron_4x3(cplx A[4][4], m3 B, cplx K[12][12]) {
    for (int s = 0; s < 4; s++)
        for (int sp = 0; sp < 4; sp++)
            for (int c = 0; c < 3; c++)
                for (int cp = 0; cp < 3; cp++) K[3 * s + c][3 * sp + cp] = A[s][sp] * B.m[c][cp];
}

int wdref_dense(int T, int Z, int Y, int X, double m0, double csw, const double *U,
                double *M_out /* [12V][12V][2], row-major */) {
    if (T < 1 || Z < 1 || Y < 1 || X < 1 || !U || !M_out) return -1;
    dims_t d = {{T, Z, Y, X}};
    const int64_t V = (int64_t)T * Z * Y * X, N = 12 * V;
    if (N > 6144) return -2;
    cplx *M = (cplx *)M_out;
    memset(M, 0, sizeof(cplx) * (size_t)N * (size_t)N);
    cplx gam[4][4][4];
    for (int mu = 0; mu < 4; mu++) gamma_c(mu, gam[mu]);
    for (int64_t x = 0; x < V; x++) {
        cplx S[12][12];
        if (csw != 0.0) {
            selfcoupling_full(&d, m0, csw, U, x, gam, S);
        } else {
            memset(S, 0, sizeof S);
            for (int i = 0; i < 12; i++) S[i][i] = m0 + 4.0;
        }
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) M[(12 * x + i) * N + 12 * x + j] += S[i][j];
        for (int mu = 0; mu < 4; mu++) {
            const int64_t xp = shifted(&d, x, mu, +1, -1, 0), xm = shifted(&d, x, mu, -1, -1, 0);
            cplx Pm[4][4], Pp[4][4], K[12][12];
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) {
                    Pm[a][b] = ((a == b) ? 1.0 : 0.0) - gam[mu][a][b];
                    Pp[a][b] = ((a == b) ? 1.0 : 0.0) + gam[mu][a][b];
                }
            kron_4x3(Pm, m3_load(link(U, x, mu)), K);
            for (int i = 0; i < 12; i++)
                for (int j = 0; j < 12; j++) M[(12 * x + i) * N + 12 * xp + j] += -0.5 * K[i][j];
            kron_4x3(Pp, m3_dag(m3_load(link(U, xm, mu))), K);
            for (int i = 0; i < 12; i++)
                for (int j = 0; j < 12; j++) M[(12 * x + i) * N + 12 * xm + j] += -0.5 * K[i][j];
        }
    }
    return 0;
}

int wdref_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void wdref_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
