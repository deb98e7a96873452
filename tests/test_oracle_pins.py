"""Pins of the CPU oracle against what the paper and the mathematics fix.

The paper prints no worked numerical example (no input/output spinor anywhere in PAPER.md), so
the oracle is pinned by closed forms, invariants, brute force on tiny lattices and special cases
of eq. 1.13, chosen so that a dropped term, a wrong sign or index, a misplaced
dagger or a transposed operand fails at least one of them.  All CPU-only.
"""
import itertools

import numpy as np
import pytest

import oracle
import wdinputs
from latticeutil import GAMMA5, c, expand42, f, gamma_r1, gauge_lat, rel_l2, spinor_lat

TOL = 1e-13
DIRS = range(4)


def _shift(a, mu, s):
    """field(x) -> field(x + s*mu) on a lattice array whose first four axes are T,Z,Y,X."""
    return np.roll(a, -s, axis=mu)


# ------------------------------------------------------------------------- gamma matrices (R1)
def test_gamma_tables_match_reading_R1():
    for mu in DIRS:
        assert np.array_equal(oracle.gamma(mu), gamma_r1(mu))


def test_gamma_clifford_algebra_and_structure():
    g = [oracle.gamma(mu) for mu in DIRS]
    for mu in DIRS:
        assert np.allclose(g[mu], g[mu].conj().T)  # Hermitian (needed for eq. 1.10)
        for nu in DIRS:
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu))
        # exactly one entry per row, of modulus 1 (preprocessor "complex literals")
        assert np.all(np.count_nonzero(g[mu], axis=1) == 1)
        assert np.allclose(np.abs(g[mu][g[mu] != 0]), 1.0)
        # projectors (1 -+ gamma)/2 have rank 2: 6 of 12 entries
        for sgn in (+1, -1):
            assert np.linalg.matrix_rank(np.eye(4) + sgn * g[mu]) == 2
    # gamma_T couples spin 0<->2 and 1<->3 (Listing 4.2)
    assert g[0][0, 2] != 0 and g[0][1, 3] != 0
    # gamma5 diagonal; gamma_mu gamma_nu block diagonal in spins {0,1},{2,3} (42 = 12+2*15, :547)
    g5 = g[0] @ g[1] @ g[2] @ g[3]
    assert np.allclose(g5, GAMMA5)
    for mu, nu in itertools.product(DIRS, DIRS):
        p = g[mu] @ g[nu]
        assert np.allclose(p[:2, 2:], 0) and np.allclose(p[2:, :2], 0)


# ------------------------------------------------------------- P1 free field plane wave
@pytest.mark.parametrize("dims,k", [((4, 6, 2, 8), (1, 2, 1, 3)), ((2, 2, 2, 2), (1, 0, 1, 1)),
                                     ((3, 5, 4, 2), (2, 1, 3, 1))])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_P1_free_field_plane_wave_closed_form(dims, k, csw):
    m0 = -0.35
    U = wdinputs.gauge_unit(dims)
    p = np.array([2 * np.pi * k[mu] / dims[mu] for mu in DIRS])
    coords = np.stack(np.meshgrid(*[np.arange(n) for n in dims], indexing="ij"), axis=-1)
    phase = np.exp(1j * (coords @ p))  # [T][Z][Y][X]
    C = oracle.build_clover(dims, m0, csw, U) if csw else None
    rng = np.random.default_rng(5)
    # closed form, derived from eq. 1.13 with U = 1: M(p) = (m0+4-sum cos p) I + i sum sin p gamma
    Mp = (m0 + 4 - np.cos(p).sum()) * np.eye(4, dtype=complex)
    for mu in DIRS:
        Mp = Mp + 1j * np.sin(p[mu]) * gamma_r1(mu)
    Mfull = np.zeros((12, 12), dtype=complex)
    for j in range(12):
        u = np.zeros(12, dtype=complex)
        u[j] = 1.0
        psi = (phase[..., None] * u).reshape(-1, 12)
        out = c(oracle.apply(dims, m0, U, C, f(psi))).reshape(*dims, 12)
        w = out / phase[..., None]
        assert np.abs(w - w[0, 0, 0, 0]).max() < 1e-13  # plane-wave form is preserved
        Mfull[:, j] = w[0, 0, 0, 0]
    assert np.abs(Mfull - np.kron(Mp, np.eye(3))).max() < 1e-13
    # basis-independent part: eigenvalues (m0+4-sum cos) +- i sqrt(sum sin^2), each 6-fold
    ev = np.linalg.eigvals(Mfull)
    re, im = m0 + 4 - np.cos(p).sum(), np.sqrt((np.sin(p) ** 2).sum())
    assert np.abs(ev.real - re).max() < 1e-12
    assert np.abs(np.sort(ev.imag) - np.array([-im] * 6 + [im] * 6)).max() < 1e-12
    # and on a random spinor amplitude
    u = rng.normal(size=12) + 1j * rng.normal(size=12)
    psi = (phase[..., None] * u).reshape(-1, 12)
    out = c(oracle.apply(dims, m0, U, C, f(psi))).reshape(*dims, 12)
    assert rel_l2(out, phase[..., None] * (np.kron(Mp, np.eye(3)) @ u)) < TOL


# ------------------------------------------------------------- P2 gamma5-hermiticity
@pytest.mark.parametrize("csw", [0.0, 1.3])
@pytest.mark.parametrize("unitary", [True, False])
def test_P2_gamma5_hermiticity(csw, unitary):
    dims, m0 = (4, 2, 6, 4), -0.2
    V = wdinputs.volume(dims)
    if unitary:
        U = wdinputs.gauge_haar(dims, 11)
    else:  # holds for ANY complex 3x3 links (R11): U^H is used, never U^-1
        U = 0.6 * wdinputs.gaussian(V * 72, 12).reshape(V, 4, 3, 3, 2)
    C = oracle.build_clover(dims, m0, csw, U) if csw else None
    psi, phi = c(wdinputs.spinor(dims, 13)[0]), c(wdinputs.spinor(dims, 14)[0])
    g5 = np.kron(GAMMA5, np.eye(3))
    Dpsi = c(oracle.apply(dims, m0, U, C, f(psi)))
    g5Dg5phi = (c(oracle.apply(dims, m0, U, C, f(phi @ g5.T))) @ g5.T)
    lhs = np.vdot(phi, Dpsi)
    rhs = np.vdot(g5Dg5phi, psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-13


# ------------------------------------------------------------- P3 gauge covariance
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_P3_gauge_covariance(csw):
    dims, m0 = (4, 4, 2, 6), -0.4
    U = wdinputs.gauge_exp(dims, 21, 0.7)
    g = c(wdinputs.su3_field(dims, 22)).reshape(*dims, 3, 3)
    Ul = gauge_lat(U, dims)
    Ut = np.empty_like(Ul)
    for mu in DIRS:  # U'_mu(x) = g(x) U_mu(x) g(x+mu)^H
        gp = _shift(g, mu, +1)
        Ut[..., mu, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, Ul[..., mu, :, :], gp.conj())
    psi = spinor_lat(wdinputs.spinor(dims, 23)[0], dims)
    psit = np.einsum("...ab,...sb->...sa", g, psi)
    Uf, Utf = f(Ul.reshape(-1, 4, 3, 3)), f(Ut.reshape(-1, 4, 3, 3))
    C = oracle.build_clover(dims, m0, csw, Uf) if csw else None
    Ct = oracle.build_clover(dims, m0, csw, Utf) if csw else None
    out = spinor_lat(oracle.apply(dims, m0, Uf, C, f(psi.reshape(-1, 12))), dims)
    outt = spinor_lat(oracle.apply(dims, m0, Utf, Ct, f(psit.reshape(-1, 12))), dims)
    assert rel_l2(outt, np.einsum("...ab,...sb->...sa", g, out)) < TOL
    if csw:  # the clover term really contributes (the test is not vacuous)
        C0 = oracle.apply(dims, m0, Uf, None, f(psi.reshape(-1, 12)))
        assert rel_l2(c(C0).reshape(out.shape), out) > 1e-3


# ------------------------------------------------------------- P4 dense brute force
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (2, 4, 2, 4), (3, 2, 2, 2)])
@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_P4_dense_kronecker_assembly(dims, csw):
    m0 = -0.5
    V = wdinputs.volume(dims)
    U = wdinputs.gauge_haar(dims, 31)
    M = oracle.dense(dims, m0, csw, U)
    C = oracle.build_clover(dims, m0, csw, U) if csw else None
    psi = c(wdinputs.spinor(dims, 32, nrhs=3))
    ref = (M @ psi.reshape(3, 12 * V).T).T.reshape(3, V, 12)
    out = c(oracle.apply(dims, m0, U, C, f(psi)))
    assert rel_l2(out, ref) < TOL
    # the dense matrix itself is gamma5-Hermitian
    G5 = np.kron(np.eye(V), np.kron(GAMMA5, np.eye(3)))
    assert np.abs(G5 @ M @ G5 - M.conj().T).max() < 1e-13


def test_P4b_point_source_hand_check():
    """A delta source at x0 reaches x0-mu through U_mu(x0-mu) with (1-gamma_mu) and x0+mu through
    U_mu(x0)^H with (1+gamma_mu) — eq. 1.13 read off by hand, in numpy."""
    dims, m0 = (4, 4, 4, 4), -0.3
    V = wdinputs.volume(dims)
    Ul = gauge_lat(wdinputs.gauge_haar(dims, 41), dims)
    x0 = (1, 3, 0, 2)
    rng = np.random.default_rng(3)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    psi = np.zeros((*dims, 4, 3), dtype=complex)
    psi[x0] = u
    out = spinor_lat(oracle.apply(dims, m0, f(Ul.reshape(-1, 4, 3, 3)), None, f(psi.reshape(V, 12))), dims)
    expect = np.zeros_like(psi)
    expect[x0] += (m0 + 4) * u
    for mu in DIRS:
        xm = list(x0); xm[mu] = (xm[mu] - 1) % dims[mu]; xm = tuple(xm)
        xp = list(x0); xp[mu] = (xp[mu] + 1) % dims[mu]; xp = tuple(xp)
        g = gamma_r1(mu)
        expect[xm] += -0.5 * np.einsum("st,ab,tb->sa", np.eye(4) - g, Ul[xm][mu], u)
        expect[xp] += -0.5 * np.einsum("st,ab,tb->sa", np.eye(4) + g, Ul[x0][mu].conj().T, u)
    assert rel_l2(out, expect) < TOL


# ------------------------------------------------------------- P5 clover closed forms
@pytest.mark.parametrize("mu,nu", [(3, 2), (2, 3), (0, 1), (1, 3), (0, 3), (2, 1), (0, 2)])
def test_P5_constant_abelian_flux_closed_form(mu, nu):
    """U_nu(x) = diag(e^{i phi x_mu}, e^{-i phi x_mu}, 1), other links 1: every mu-nu plaquette of
    eq. 1.12 is diag(e^{i phi}, e^{-i phi}, 1), so eq. 2.5 gives
    S = (m0+4) I - (csw/2) i gamma_mu gamma_nu (x) diag(sin phi, -sin phi, 0)."""
    dims, m0, csw, kk = (4, 6, 4, 8), -0.4, 1.7, 1
    phi = 2 * np.pi * kk / dims[mu]
    Ul = gauge_lat(wdinputs.gauge_unit(dims), dims).copy()
    xm = np.arange(dims[mu]).reshape([-1 if a == mu else 1 for a in range(4)])
    xm = np.broadcast_to(xm, dims)
    Ul[..., nu, 0, 0] = np.exp(1j * phi * xm)
    Ul[..., nu, 1, 1] = np.exp(-1j * phi * xm)
    S = oracle.build_clover_full(dims, m0, csw, f(Ul.reshape(-1, 4, 3, 3)))
    expect = (m0 + 4) * np.eye(12) - (csw / 2) * 1j * np.kron(
        gamma_r1(mu) @ gamma_r1(nu), np.diag([np.sin(phi), -np.sin(phi), 0.0]))
    assert np.abs(S - expect[None]).max() < 1e-13
    assert abs(np.sin(phi)) > 0.1


def test_P5b_pure_gauge_field_has_no_clover_term():
    dims, m0 = (4, 2, 4, 6), -0.1
    g = c(wdinputs.su3_field(dims, 51)).reshape(*dims, 3, 3)
    Ul = np.empty((*dims, 4, 3, 3), dtype=complex)
    for mu in DIRS:  # U_mu(x) = g(x) g(x+mu)^H
        Ul[..., mu, :, :] = np.einsum("...ab,...cb->...ac", g, _shift(g, mu, +1).conj())
    S = oracle.build_clover_full(dims, m0, 1.0, f(Ul.reshape(-1, 4, 3, 3)))
    assert np.abs(S - (m0 + 4) * np.eye(12)[None]).max() < 1e-13


# ------------------------------------------------------------- P6 structure of S, 42-entry packing
def test_P6_selfcoupling_structure_and_packing():
    dims, m0, csw = (4, 4, 2, 4), -0.4, 1.0
    U = wdinputs.gauge_exp(dims, 61, 0.8)
    S = oracle.build_clover_full(dims, m0, csw, U)
    assert np.abs(S - S.conj().transpose(0, 2, 1)).max() < 1e-14          # Hermitian
    assert np.abs(S[:, :6, 6:]).max() == 0 and np.abs(S[:, 6:, :6]).max() == 0  # 42 = 12 + 2*15
    assert np.abs(S[:, :6, :6] - (m0 + 4) * np.eye(6)).max() > 1e-2       # non-trivial
    C = oracle.build_clover(dims, m0, csw, U)
    assert np.abs(expand42(C) - S).max() < 1e-14                          # order of the 42 (R6)
    assert np.abs(C[:, :12, 1]).max() == 0
    # apply through the stored 42 entries == full S psi + hopping part
    psi = wdinputs.spinor(dims, 62)[0]
    hop = c(oracle.apply(dims, m0, U, None, psi)) - (m0 + 4) * c(psi)
    ref = np.einsum("vij,vj->vi", S, c(psi)) + hop
    assert rel_l2(c(oracle.apply(dims, m0, U, C, psi)), ref) < TOL


def test_P6b_random_selfcoupling_all_42_entries_used():
    dims, m0 = (2, 4, 4, 2), -0.4
    U = wdinputs.gauge_haar(dims, 63)
    C = wdinputs.selfcoupling_random(dims, 64)
    psi = wdinputs.spinor(dims, 65)[0]
    hop = c(oracle.apply(dims, m0, U, None, psi)) - (m0 + 4) * c(psi)
    ref = np.einsum("vij,vj->vi", expand42(C), c(psi)) + hop
    assert rel_l2(c(oracle.apply(dims, m0, U, C, psi)), ref) < TOL


# ------------------------------------------------------------- P7 linearity, multi-RHS
def test_P7_linearity_and_multi_rhs():
    dims, m0, csw = (4, 4, 4, 2), -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 71)
    C = oracle.build_clover(dims, m0, csw, U)
    psis = wdinputs.spinor(dims, 72, nrhs=4)
    batch = oracle.apply(dims, m0, U, C, psis)
    for r in range(4):
        assert np.array_equal(batch[r], oracle.apply(dims, m0, U, C, psis[r]))
    a, b = 0.7 - 0.2j, -1.1 + 0.5j
    comb = f(a * c(psis[0]) + b * c(psis[1]))
    lin = a * c(batch[0]) + b * c(batch[1])
    assert rel_l2(c(oracle.apply(dims, m0, U, C, comb)), lin) < TOL


# ------------------------------------------------------------- P8 translation covariance
@pytest.mark.parametrize("mu", DIRS)
def test_P8_translation_covariance(mu):
    dims, m0, csw = (4, 2, 6, 4), -0.4, 1.0
    V = wdinputs.volume(dims)
    U = wdinputs.gauge_haar(dims, 81)
    psi = wdinputs.spinor(dims, 82)[0]
    out = oracle.apply(dims, m0, U, oracle.build_clover(dims, m0, csw, U), psi)
    Us = np.roll(U.reshape(*dims, 4, 3, 3, 2), 1, axis=mu).reshape(V, 4, 3, 3, 2)
    psis = np.roll(psi.reshape(*dims, 12, 2), 1, axis=mu).reshape(V, 12, 2)
    outs = oracle.apply(dims, m0, Us, oracle.build_clover(dims, m0, csw, Us), psis)
    assert rel_l2(outs.reshape(*dims, 12, 2), np.roll(out.reshape(*dims, 12, 2), 1, axis=mu)) < TOL


# ------------------------------------------------------------- P9 csw -> 0
def test_P9_identity_selfcoupling_reproduces_wilson():
    dims, m0 = (4, 4, 2, 2), -0.5
    V = wdinputs.volume(dims)
    U = wdinputs.gauge_haar(dims, 91)
    psi = wdinputs.spinor(dims, 92)[0]
    C = np.zeros((V, 42, 2))
    C[:, :12, 0] = m0 + 4
    assert rel_l2(oracle.apply(dims, m0, U, C, psi), oracle.apply(dims, m0, U, None, psi)) < 1e-15
    assert np.abs(oracle.build_clover(dims, m0, 0.0, U) - C).max() == 0


# ------------------------------------------------------------- input generators sanity
def test_inputs_are_what_the_recipe_says():
    dims = (4, 4, 4, 4)
    for U in (wdinputs.gauge_haar(dims, 1001), wdinputs.gauge_exp(dims, 1002, 0.3)):
        Ul = c(U).reshape(-1, 3, 3)
        assert np.abs(np.einsum("nab,ncb->nac", Ul, Ul.conj()) - np.eye(3)).max() < 1e-13
        assert np.abs(np.linalg.det(Ul) - 1).max() < 1e-13
    near = c(wdinputs.gauge_exp(dims, 1002, 0.3)).reshape(-1, 3, 3)
    assert np.abs(near - np.eye(3)).max() < 1.5  # near-unit field
    g = wdinputs.gaussian(200000, 7)
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01
    assert np.array_equal(wdinputs.spinor(dims, 5, nrhs=2)[1], wdinputs.spinor(dims, 6)[0])
