"""GPU parity of the domain-decomposed operator (csrc/wd_dd.cu + open-boundary mode of the fused kernels): 2, 4 and 8
sub-lattices on ONE device, the half-spinor faces exchanged through device buffers, compared with the oracle's
operator on the undivided global lattice (rel. L2 <= 1e-13).  Only one GPU is reachable per run, so this is how the
decomposition is proven; the rank arithmetic and the exchange order are covered on the CPU (test_decomposition.py)."""
import numpy as np
import pytest

import oracle
import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import rel_l2
from paper_2407_00041_b200.dd import EmulatedDecomposition
from test_gpu_parity import TOL, torch  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("gdims,grid", [
    ((8, 8, 8, 16), (2, 1, 1, 1)),    # T split in two (both neighbours are the same rank)
    ((16, 4, 8, 16), (4, 1, 1, 1)),   # T split in four
    ((8, 8, 8, 16), (2, 2, 1, 1)),    # T and Z (the 8-GPU plan of DESIGN.md at a small size)
    ((4, 8, 8, 32), (1, 2, 2, 2)),    # Z, Y and X
    ((8, 4, 8, 32), (2, 2, 2, 1)),    # eight sub-lattices
    ((6, 6, 4, 6), (2, 3, 1, 1)),     # odd local extents: only the linear LDG kernel fits
    ((2, 4, 4, 16), (2, 1, 1, 1)),    # local T extent 1: high and low face are the same sites
])
def test_decomposed_operator_matches_oracle_on_the_global_lattice(torch, gdims, grid):
    m0, csw, nrhs = -0.4, 1.0, 2
    U = wdinputs.gauge_haar(gdims, 801)
    psi = wdinputs.spinor(gdims, 802, nrhs=nrhs)
    C = oracle.build_clover(gdims, m0, csw, U)
    ref_c = oracle.apply(gdims, m0, U, C, psi)
    ref_w = oracle.apply(gdims, m0, U, None, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)  # S cut out of the oracle's global field
    try:
        kname = wd.wd_kernel_name(wd.wd_kernel_in_use(em.ops[0].h))
        assert rel_l2(em.apply(psi, nrhs), ref_c) <= TOL, kname
    finally:
        em.close()
    em = EmulatedDecomposition(torch, gdims, grid, m0, 0.0, U)  # pure Wilson
    try:
        assert rel_l2(em.apply(psi, nrhs), ref_w) <= TOL
    finally:
        em.close()


@pytest.mark.parametrize("kernel", ["tmw_2x4x16", "tma_2x4x16", "tmb_4x4x8", "tmb_2x8x8", "tile_1x4x4x16", "linear256"])
def test_every_kernel_family_supports_open_boundaries(torch, kernel):
    gdims, grid, m0, csw = (8, 8, 16, 32), (2, 2, 1, 2), -0.4, 1.0
    U = wdinputs.gauge_exp(gdims, 811, 0.5)
    psi = wdinputs.spinor(gdims, 812)
    C = wdinputs.selfcoupling_random(gdims, 813)
    ref = oracle.apply(gdims, m0, U, C, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)
    try:
        for op in em.ops:
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id(kernel))
        assert rel_l2(em.apply(psi), ref) <= TOL
    finally:
        em.close()


def test_local_clover_from_extended_links_and_state_rules(torch):
    """S of a sub-lattice built on the device from the links of the local lattice extended by one site, against the
    oracle's S of the global lattice; wd_build_clover is refused on a decomposed handle."""
    gdims, grid, m0, csw = (8, 8, 4, 16), (2, 2, 1, 1), -0.4, 1.0
    U = wdinputs.gauge_exp(gdims, 821, 0.4)
    psi = wdinputs.spinor(gdims, 822)
    C = oracle.build_clover(gdims, m0, csw, U)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U)  # C_global = None: local_clover path
    try:
        for r, op in enumerate(em.ops):
            Cl = np.empty((int(np.prod(em.decomp.local_dims)), 42, 2))
            wd.wd_get_clover(op.h, Cl)
            assert rel_l2(Cl, em.decomp.extract(C, r)) <= TOL
            with pytest.raises(wd.WDError) as e:
                wd.wd_build_clover(op.h)
            assert e.value.code == wd.WD_ESTATE
            assert wd.wd_dd_open_mask(op.h) == 0b0011 and wd.wd_dd_face_sites(op.h, 2) == 0
            with pytest.raises(wd.WDError):
                wd.wd_dd_pack(op.h, op.spinor(), 1, 2, op.spinor(), op.spinor())  # Y is not decomposed
        assert rel_l2(em.apply(psi), oracle.apply(gdims, m0, U, C, psi)) <= TOL
    finally:
        em.close()
    with pytest.raises(wd.WDError):
        wd.wd_create_local((8, 8, 8, 8), (3, 1, 1, 1), (0, 0, 0, 0), 0.0, 0.0)


def test_decomposed_bench_size_slab(torch, capsys):
    """The 8-GPU plan of the bench (64^4 cut 4 x 2 in T and Z: local 16 x 32 x 64 x 64) on one sub-lattice pair:
    a 32 x 32 x 64 x 64 global lattice cut (2, 1, 1, 1), default kernels, compared with the oracle on every site."""
    gdims, grid, m0, csw = (32, 32, 64, 64), (2, 1, 1, 1), -0.4, 1.0
    U = wdinputs.gauge_haar(gdims, 831)
    psi = wdinputs.spinor(gdims, 832)
    C = oracle.build_clover(gdims, m0, csw, U)
    ref = oracle.apply(gdims, m0, U, C, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)
    try:
        out = em.apply(psi)
        kname = wd.wd_kernel_name(wd.wd_kernel_in_use(em.ops[0].h))
    finally:
        em.close()
    err = rel_l2(out, ref)
    with capsys.disabled():
        print(f"\n[decomposed parity] global {'x'.join(map(str, gdims))} grid {grid} kernel {kname}: rel_l2 {err:.3e}", flush=True)
    assert err <= TOL
