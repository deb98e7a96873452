"""Pins of the GMRES oracle (oracle/gmres.py, Algorithm 1 of the paper) against what the
mathematics fixes — none of them re-types its recurrences:

  G1  m = N on a 2^4 lattice: one cycle of GMRES(N) is a direct solve; compared with numpy.linalg.solve on the
      dense Kronecker-assembled operator (oracle.dense, itself pinned in test_oracle_pins.py).
  G2  the true residual ||b - A x_m|| (recomputed from x) equals the least-squares residual min ||beta e1 - H y||
      of the cycle that produced x_m; residuals never increase from cycle to cycle.
  G3  a normal matrix with k distinct eigenvalues: GMRES converges in exactly k steps, and with m > k the
      near-breakdown rule |h_{k+1,k}| < tol/10 ends the Arnoldi loop at j = k.
  G4  structure: H upper Hessenberg with real positive sub-diagonal; x0 = exact solution returns at once.
  G5  minimal-residual property: after one cycle, ||b - A x_m|| <= ||b - A (x0 + V c)|| for random c in the same
      Krylov space, built independently with numpy's QR of [r, Ar, ..., A^{m-1} r].
"""
import numpy as np
import pytest

import oracle
import wdinputs
from latticeutil import c
from oracle.gmres import gmres, wilson_operator


def _wilson(dims, seed, csw=1.0, m0=-0.4, eps=0.4):
    U = wdinputs.gauge_exp(dims, seed, eps)
    C = oracle.build_clover(dims, m0, csw, U) if csw else None
    return U, C, wilson_operator(dims, m0, U, C)


def test_G1_full_krylov_space_is_a_direct_solve():
    dims, m0, csw = (2, 2, 2, 2), -0.4, 1.0
    U, C, A = _wilson(dims, 701)
    N = 12 * 16
    b = c(wdinputs.spinor(dims, 702)[0])
    M = oracle.dense(dims, m0, csw, U)
    xs = np.linalg.solve(M, b.ravel()).reshape(b.shape)
    x, info = gmres(A, b, m=N, tol=1e-13, max_cycles=1)
    assert info["cycles"] == 1
    assert np.linalg.norm(x - xs) / np.linalg.norm(xs) < 1e-9
    assert info["resid"][-1] / info["resid"][0] < 1e-10


@pytest.mark.parametrize("m", [3, 8])
def test_G2_true_residual_equals_recurrence_residual_and_is_monotone(m):
    dims = (4, 4, 4, 4)
    U, C, A = _wilson(dims, 711)
    b = c(wdinputs.spinor(dims, 712)[0])
    x, info = gmres(A, b, m=m, tol=1e-8, max_cycles=6)
    res = info["resid"]
    assert len(res) == info["cycles"] + 1 and info["cycles"] >= 2
    for k in range(info["cycles"]):
        assert abs(res[k + 1] - info["lsq_resid"][k]) <= 1e-10 * res[0]  # ||b - A x_m|| = min ||beta e1 - H y||
        assert res[k + 1] <= res[k] * (1 + 1e-14)
    assert abs(np.linalg.norm((b - A(x)).ravel()) - res[-1]) <= 1e-12 * res[0]
    assert info["applies"] == info["cycles"] * (m + 1) + 1


def test_G3_k_distinct_eigenvalues_and_the_breakdown_rule():
    rng = np.random.default_rng(3)
    n, lam = 60, np.array([1.5 + 0.5j, -0.7 + 1.1j, 2.2 - 0.3j])
    d = lam[rng.integers(0, 3, size=n)]
    d[:3] = lam
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    M = Q @ np.diag(d) @ Q.conj().T  # normal, 3 distinct eigenvalues
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    x, info = gmres(lambda v: M @ v, b, m=3, tol=1e-12, max_cycles=1)
    assert np.linalg.norm(M @ x - b) / np.linalg.norm(b) < 1e-12
    x5, info5 = gmres(lambda v: M @ v, b, m=6, tol=1e-9, max_cycles=3)
    assert info5["kdim"][0] == 3 and info5["cycles"] == 1  # |h_43| < tol/10 stops the Arnoldi loop at j = 3
    assert np.linalg.norm(M @ x5 - b) / np.linalg.norm(b) < 1e-9
    # two steps are NOT enough: the residual polynomial of degree 2 cannot vanish on three eigenvalues
    x2, _ = gmres(lambda v: M @ v, b, m=2, tol=1e-12, max_cycles=1)
    assert np.linalg.norm(M @ x2 - b) / np.linalg.norm(b) > 1e-4


def test_G4_hessenberg_structure_and_exact_initial_guess():
    dims = (2, 4, 2, 4)
    U, C, A = _wilson(dims, 721)
    b = c(wdinputs.spinor(dims, 722)[0])
    x, info = gmres(A, b, m=6, tol=1e-30, max_cycles=2)
    for H in info["H"]:
        assert H.shape == (7, 6)
        assert np.abs(np.tril(H, -2)).max() == 0.0
        sub = np.diag(H, -1)
        assert np.abs(sub.imag).max() == 0.0 and (sub.real > 0).all()
    xs, inf2 = gmres(A, A(x), x0=x, m=6, tol=1e-10, max_cycles=5)
    assert inf2["cycles"] == 0 and np.array_equal(xs, x)


def test_G5_minimal_residual_over_the_krylov_space():
    dims = (4, 2, 4, 2)
    U, C, A = _wilson(dims, 731, csw=0.0)
    b = c(wdinputs.spinor(dims, 732)[0])
    m = 5
    x, info = gmres(A, b, m=m, tol=1e-30, max_cycles=1)
    rbest = np.linalg.norm((b - A(x)).ravel())
    K = [b]
    for _ in range(m - 1):
        K.append(A(K[-1]))
    Q, _ = np.linalg.qr(np.stack([k.ravel() for k in K], axis=1))
    AQ = np.stack([A(Q[:, i].reshape(b.shape)).ravel() for i in range(m)], axis=1)
    y, *_ = np.linalg.lstsq(AQ, b.ravel(), rcond=None)  # the minimiser, by a library routine
    assert abs(np.linalg.norm(b.ravel() - AQ @ y) - rbest) <= 1e-10 * np.linalg.norm(b.ravel())
    rng = np.random.default_rng(5)
    for _ in range(5):
        cvec = y + 1e-3 * (rng.normal(size=m) + 1j * rng.normal(size=m))
        assert np.linalg.norm(b.ravel() - AQ @ cvec) >= rbest * (1 - 1e-12)
