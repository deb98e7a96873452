"""CPU oracle of restarted GMRES with right preconditioning M = I.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Follows Algorithm 1 of the paper line by line, in the paper's order and notation:

    1  x <- x0                                     3  while termination criterion not satisfied:
    4      r <- b - A x                            5      beta <- ||r||_2
    6      v_1 <- r / beta                         7      for j = 1..m:
    8          z_j <- M^-1 v_j  (M = I)            9          w <- A z_j
    10-12      for i = 1..j:  h_ij <- <w, v_i>;  w <- w - h_ij v_i          (modified Gram-Schmidt)
    14         h_{j+1,j} <- ||w||_2               15          v_{j+1} <- w / h_{j+1,j}
    18     y_m <- argmin_y || beta e_1 - H_m y ||_2
    19     x_m <- x + M^-1 V_m y_m                20      x <- x_m

Readings (R16-R18):
  R16  <w, v_i> is v_i^H w (conjugate-linear in v_i): the only reading for which line 11 makes w orthogonal to v_i.
  R17  Termination: ||b - A x|| < tol * ||b - A x_0||, tested where Algorithm 1 tests it — at the top
       of the restart loop, on the TRUE residual of line 4 — or `max_cycles` restart cycles done.
  R18  Early termination: if |h_{j+1,j}| < tol / 10 the Arnoldi loop stops after step j (near
       breakdown); the cycle's Krylov dimension is then j and lines 18-20 use H_j.
Line 18 is solved with a library routine (numpy.linalg.lstsq), no Givens recurrences: nothing here is shaped like
the CUDA path.  Vectors are complex128 numpy arrays of any shape; A is a callable.
"""
from __future__ import annotations

import numpy as np


def gmres(A, b, x0=None, m=10, tol=1e-10, max_cycles=50):
    """Returns (x, info).  info["resid"][k] = ||b - A x|| at the top of cycle k (k = 0: initial), one more entry
    for the final x; info["lsq_resid"][k] = min_y ||beta e_1 - H y|| of cycle k (the recurrence residual);
    info["H"] = list of the (j+1) x j Hessenberg matrices; info["kdim"] = Krylov dimension of each cycle."""
    b = np.asarray(b, dtype=np.complex128)
    x = np.zeros_like(b) if x0 is None else np.array(x0, dtype=np.complex128)      # line 1
    info = {"resid": [], "lsq_resid": [], "H": [], "kdim": [], "cycles": 0, "applies": 0}
    r0 = None
    while True:                                                                      # line 3
        r = b - A(x)                                                                 # line 4
        info["applies"] += 1
        beta = float(np.linalg.norm(r.ravel()))                                      # line 5
        info["resid"].append(beta)
        if r0 is None:
            r0 = beta
        if beta < tol * r0 or info["cycles"] >= max_cycles or beta == 0.0:           # R17
            break
        H = np.zeros((m + 1, m), dtype=np.complex128)                                # line 2
        V = [r / beta]                                                               # line 6
        kdim = m
        for j in range(m):                                                           # line 7
            z = V[j]                                                                 # line 8 (M = I)
            w = A(z)                                                                 # line 9
            info["applies"] += 1
            for i in range(j + 1):                                                   # line 10
                H[i, j] = np.vdot(V[i].ravel(), w.ravel())                           # line 11 (R16: v_i^H w)
                w = w - H[i, j] * V[i]                                               # line 12
            hn = float(np.linalg.norm(w.ravel()))                                    # line 14
            H[j + 1, j] = hn
            if hn < tol / 10.0:                                                      # R18
                kdim = j + 1
                break
            V.append(w / hn)                                                         # line 15
        Hk = H[: kdim + 1, :kdim]
        e1 = np.zeros(kdim + 1, dtype=np.complex128)
        e1[0] = beta
        y, *_ = np.linalg.lstsq(Hk, e1, rcond=None)                                  # line 18
        info["lsq_resid"].append(float(np.linalg.norm(e1 - Hk @ y)))
        for i in range(kdim):                                                        # line 19
            x = x + y[i] * V[i]                                                      # line 20
        info["H"].append(Hk.copy())
        info["kdim"].append(kdim)
        info["cycles"] += 1
    return x, info


def wilson_operator(dims, m0, U, C):
    """A(x) for the oracle's Wilson(-clover) operator: complex [V][12] in, complex [V][12] out."""
    from . import apply

    def A(x):
        xf = np.ascontiguousarray(x, dtype=np.complex128).view(np.float64).reshape(-1, 12, 2)
        return apply(dims, m0, U, C, xf).view(np.complex128)[..., 0]

    return A
