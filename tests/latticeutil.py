"""numpy helpers for the tests (lattice reshapes, shifts, independent restatement of DESIGN.md R1).

Nothing here is used by the oracle or by the CUDA library.
"""
import numpy as np

SIG1 = np.array([[0, 1], [1, 0]], dtype=complex)
SIG2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
SIG3 = np.array([[1, 0], [0, -1]], dtype=complex)


def gamma_r1(mu: int) -> np.ndarray:
    """DESIGN.md R1 restated with numpy blocks: gamma_mu = [[0, a], [a^H, 0]],
    a_T = 1, a_Z = i sigma_3, a_Y = i sigma_2, a_X = i sigma_1."""
    a = [np.eye(2, dtype=complex), 1j * SIG3, 1j * SIG2, 1j * SIG1][mu]
    z = np.zeros((2, 2), dtype=complex)
    return np.block([[z, a], [a.conj().T, z]])


GAMMA5 = np.diag([-1.0, -1.0, 1.0, 1.0]).astype(complex)


def c(a):
    """(…, 2) float64 -> (…) complex128 view."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a.view(np.complex128)[..., 0]


def f(a):
    """complex128 (…) -> float64 (…, 2) copy."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64).reshape(a.shape + (2,)).copy()


def spinor_lat(psi, dims):
    """[V][12][2] float -> complex [T][Z][Y][X][4][3]."""
    return c(psi).reshape(*dims, 4, 3)


def gauge_lat(U, dims):
    """[V][4][3][3][2] float -> complex [T][Z][Y][X][4][3][3]."""
    return c(U).reshape(*dims, 4, 3, 3)


def rel_l2(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def expand42(C):
    """[V][42][2] float -> complex [V][12][12] Hermitian block-diagonal (R6)."""
    Cc = c(C)
    V = Cc.shape[0]
    S = np.zeros((V, 12, 12), dtype=complex)
    for k in range(12):
        S[:, k, k] = Cc[:, k].real
    for b in range(2):
        k = 12 + 15 * b
        for r in range(6):
            for cc in range(r + 1, 6):
                S[:, 6 * b + r, 6 * b + cc] = Cc[:, k]
                S[:, 6 * b + cc, 6 * b + r] = Cc[:, k].conj()
                k += 1
    return S
