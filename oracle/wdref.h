/* oracle/wdref.h — CPU oracle for the Wilson(-clover) Dirac operator.  TEST INFRASTRUCTURE ONLY:
 * never included, linked or called by the CUDA library or any product path (see wdref.c header).
 *
 * All pointers are HOST pointers to doubles; complex = (re, im).  V = T*Z*Y*X, site index
 * i = ((t*Z+z)*Y+y)*X+x, directions mu = 0..3 = T,Z,Y,X, periodic in all four.
 *   U   [V][4][3][3][2]   forward links U_mu(x), row-major
 *   C   [V][42][2]        self-coupling D_sc incl. the (m0+4) diagonal (eq. 2.5)
 *   psi [nrhs][V][12][2]  component 3*spin+colour
 * Return 0 on success, negative on bad arguments.
 */
#ifndef WDREF_H
#define WDREF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* out = D in, eq. 1.13, a = 1.  C == NULL: pure Wilson, S = (m0+4) I.
 * C != NULL: S(x) is taken from C (m0 is then unused). */
int wdref_apply(int T, int Z, int Y, int X, double m0, const double *U, const double *C,
                double *out, const double *in, int nrhs);

/* C = the 42 stored entries of S(x), eq. 2.5 with Q of eq. 1.12. */
int wdref_build_clover(int T, int Z, int Y, int X, double m0, double csw, const double *U,
                       double *C);

/* S_out [V][12][12][2]: the full self-coupling matrix per site (to check its structure). */
int wdref_build_clover_full(int T, int Z, int Y, int X, double m0, double csw, const double *U,
                            double *S_out);

/* M_out [12V][12V][2] row-major: D as a dense matrix assembled from Kronecker products
 * (12V <= 6144).  csw != 0 builds S from U. */
int wdref_dense(int T, int Z, int Y, int X, double m0, double csw, const double *U, double *M_out);

/* g_out [4][4][2]: gamma_mu (R1). */
void wdref_gamma(int mu, double *g_out);

int wdref_num_threads(void);
void wdref_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
