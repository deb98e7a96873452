/* wdinputs/gen.c — seeded, counter-based generators of SYNTHETIC input fields.
 *
 * This module serves both the CPU oracle (oracle/) and the CUDA library (tests, bench) with
 * the same input arrays.  It holds NONE of the method's arithmetic: no gamma matrices, no
 * Dirac operator, no plaquettes, no clover construction.  It only draws random numbers and
 * shapes them into the value distributions DESIGN.md §"Input recipe" lists (stand-ins for the
 * paper's gauge configurations, which are not available):
 *
 *   - i.i.d. N(0,1) reals                      (spinor entries, BASELINE.json configs)
 *   - Haar-random SU(3) 3x3 matrices           (Gram-Schmidt of a complex Gaussian matrix,
 *                                               determinant phase divided out)
 *   - U = exp(i*eps*H), H traceless Hermitian  (near-unit "smooth-like" links)
 *   - random Hermitian block-diagonal self-coupling arrays in the 42-entry format
 *
 * Every value depends only on (seed, element index), so fields of any size are generated in
 * parallel and reproducibly.  All arrays are host arrays of doubles, complex = (re, im).
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>

typedef double complex cplx;

static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* uniform in (0,1), 53 bits, never 0 or 1 */
static inline double u01(uint64_t seed, uint64_t ctr) {
    uint64_t r = mix64(mix64(seed) ^ mix64(ctr * 0xD1B54A32D192ED03ULL + 0x2545F4914F6CDD1DULL));
    return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* pair-th Box-Muller pair of stream `seed`: two independent standard normals */
static inline void gauss_pair(uint64_t seed, uint64_t pair, double *g0, double *g1) {
    double u1 = u01(seed, 2 * pair), u2 = u01(seed, 2 * pair + 1);
    double r = sqrt(-2.0 * log(u1));
    double a = 6.283185307179586476925286766559 * u2;
    *g0 = r * cos(a);
    *g1 = r * sin(a);
}

/* n-th standard normal of stream `seed` */
static inline double gauss(uint64_t seed, uint64_t n) {
    double g0, g1;
    gauss_pair(seed, n >> 1, &g0, &g1);
    return (n & 1) ? g1 : g0;
}

/* `per_site` (even) consecutive normals for each listed site: out[k][0..per_site) = normals per_site*sites[k] .. of the stream */
void wdin_gaussian_sites(double *out, const int64_t *sites, uint64_t nsites, uint64_t per_site, uint64_t seed) {
    const uint64_t pp = per_site / 2;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)nsites; k++)
        for (uint64_t q = 0; q < pp; q++)
            gauss_pair(seed, pp * (uint64_t)sites[k] + q, out + per_site * k + 2 * q, out + per_site * k + 2 * q + 1);
}

void wdin_gaussian(double *out, uint64_t n, uint64_t seed) {
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < (int64_t)((n + 1) / 2); p++) {
        double g0, g1;
        gauss_pair(seed, (uint64_t)p, &g0, &g1);
        out[2 * p] = g0;
        if ((uint64_t)(2 * p + 1) < n) out[2 * p + 1] = g1;
    }
}

static void gaussian_3x3(cplx g[3][3], uint64_t seed, uint64_t link) {
    for (int k = 0; k < 9; k++) {
        double re, im;
        gauss_pair(seed, 9 * link + k, &re, &im);
        g[k / 3][k % 3] = re + I * im;
    }
}

static cplx det3(cplx m[3][3]) {
    return m[0][0] * (m[1][1] * m[2][2] - m[1][2] * m[2][1]) -
           m[0][1] * (m[1][0] * m[2][2] - m[1][2] * m[2][0]) +
           m[0][2] * (m[1][0] * m[2][1] - m[1][1] * m[2][0]);
}

/* Haar SU(3): columns of a complex Gaussian matrix orthonormalised by modified Gram-Schmidt
 * (= QR with positive R diagonal, Haar on U(3)), then multiplied by exp(-i arg(det)/3). */
static void haar_link(double *o, uint64_t seed, uint64_t l) {
    {
        cplx g[3][3];
        gaussian_3x3(g, seed, l);
        for (int c = 0; c < 3; c++) {
            for (int p = 0; p < c; p++) {
                cplx dot = 0;
                for (int r = 0; r < 3; r++) dot += conj(g[r][p]) * g[r][c];
                for (int r = 0; r < 3; r++) g[r][c] -= dot * g[r][p];
            }
            double nrm = 0;
            for (int r = 0; r < 3; r++) nrm += creal(g[r][c]) * creal(g[r][c]) + cimag(g[r][c]) * cimag(g[r][c]);
            nrm = 1.0 / sqrt(nrm);
            for (int r = 0; r < 3; r++) g[r][c] *= nrm;
        }
        cplx d = det3(g);
        double th = atan2(cimag(d), creal(d)) / 3.0;
        cplx ph = cos(th) - I * sin(th);
        for (int k = 0; k < 9; k++) {
            cplx v = g[k / 3][k % 3] * ph;
            o[2 * k] = creal(v);
            o[2 * k + 1] = cimag(v);
        }
    }
}

void wdin_su3_haar(double *U, uint64_t nlinks, uint64_t seed) {
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)nlinks; l++) haar_link(U + 18 * l, seed, (uint64_t)l);
}

/* The same values for a LIST of sites of a gauge field (links 4*site .. 4*site+3 of the stream): U[k] receives the four
 * links of site sites[k], so a rank of a decomposed lattice draws its own part without generating the global field. */
void wdin_su3_haar_sites(double *U, const int64_t *sites, uint64_t nsites, uint64_t seed) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)nsites; k++)
        for (int mu = 0; mu < 4; mu++) haar_link(U + 18 * (4 * k + mu), seed, 4 * (uint64_t)sites[k] + mu);
}

static void matmul3(cplx c[3][3], cplx a[3][3], cplx b[3][3]) {
    cplx t[3][3];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[i][k] * b[k][j];
            t[i][j] = s;
        }
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c[i][j] = t[i][j];
}

/* U = exp(i*eps*H), H = (G+G^H)/2 - tr/3 with G complex Gaussian: scaling and squaring around a
 * degree-20 Taylor polynomial (argument norm scaled below 1/4). */
static void exp_link(double *o, uint64_t seed, uint64_t l, double eps) {
    {
        cplx g[3][3], a[3][3];
        gaussian_3x3(g, seed, l);
        cplx tr = 0;
        for (int i = 0; i < 3; i++) tr += creal(g[i][i]);
        double nrm = 0;
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                cplx h = 0.5 * (g[i][j] + conj(g[j][i]));
                if (i == j) h -= tr / 3.0;
                a[i][j] = I * eps * h;
                nrm += cabs(a[i][j]);
            }
        int s = 0;
        while (nrm > 0.25) { nrm *= 0.5; s++; }
        double sc = ldexp(1.0, -s);
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) a[i][j] *= sc;
        cplx e[3][3], term[3][3];
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) e[i][j] = term[i][j] = (i == j) ? 1.0 : 0.0;
        for (int k = 1; k <= 20; k++) {
            matmul3(term, term, a);
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) {
                    term[i][j] /= (double)k;
                    e[i][j] += term[i][j];
                }
        }
        for (int q = 0; q < s; q++) matmul3(e, e, e);
        for (int k = 0; k < 9; k++) {
            o[2 * k] = creal(e[k / 3][k % 3]);
            o[2 * k + 1] = cimag(e[k / 3][k % 3]);
        }
    }
}

void wdin_su3_exp(double *U, uint64_t nlinks, uint64_t seed, double eps) {
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)nlinks; l++) exp_link(U + 18 * l, seed, (uint64_t)l, eps);
}

void wdin_su3_exp_sites(double *U, const int64_t *sites, uint64_t nsites, uint64_t seed, double eps) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)nsites; k++)
        for (int mu = 0; mu < 4; mu++) exp_link(U + 18 * (4 * k + mu), seed, 4 * (uint64_t)sites[k] + mu, eps);
}

void wdin_su3_unit(double *U, uint64_t nlinks) {
#pragma omp parallel for schedule(static)
    for (int64_t l = 0; l < (int64_t)nlinks; l++) {
        double *o = U + 18 * l;
        for (int k = 0; k < 18; k++) o[k] = 0.0;
        o[0] = o[8] = o[16] = 1.0;
    }
}

/* Random self-coupling array in the 42-complex-per-site format (include/wd.h, R6):
 * entries 0..11 real diagonal = shift + scale*N(0,1) (imaginary part 0), entries 12..41 complex
 * off-diagonals scale*(N(0,1) + i N(0,1)).  An arbitrary Hermitian block-diagonal input, not a
 * clover term built from links. */
void wdin_selfcoupling_random(double *C, uint64_t nsites, uint64_t seed, double shift, double scale) {
#pragma omp parallel for schedule(static)
    for (int64_t x = 0; x < (int64_t)nsites; x++) {
        double *o = C + 84 * x;
        for (int k = 0; k < 42; k++) {
            double a = gauss(seed, 84 * (uint64_t)x + 2 * k), b = gauss(seed, 84 * (uint64_t)x + 2 * k + 1);
            if (k < 12) { o[2 * k] = shift + scale * a; o[2 * k + 1] = 0.0; }
            else        { o[2 * k] = scale * a;         o[2 * k + 1] = scale * b; }
        }
    }
}
