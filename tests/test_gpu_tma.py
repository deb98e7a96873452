"""GPU parity of the TMA-staged T-marching kernels (wd_tma.cu) against the CPU oracle.

These kernels stage every operand through shared memory with cp.async.bulk.tensor and carry the
T-direction hops in registers across steps, so the cases below aim at what is specific to them:
tiles on every lattice boundary (periodic wrap of each face box), a lattice exactly one tile wide
(every face wraps onto the tile itself), T chunks of every length including 1 and T (prologue and
epilogue slices wrap around T), several work items per CTA (barrier phases carried across items),
and all three self-coupling modes.
"""
import numpy as np
import pytest

import oracle
import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import rel_l2
from test_gpu_parity import TOL, Op, torch  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


def tma_kernels(dims):
    out = []
    for k in range(wd.wd_kernel_count()):
        name = wd.wd_kernel_name(k)
        if name.startswith(("tma_", "tmb_", "tmw_", "tmq_")):
            b = [int(v) for v in name.split("_")[1].split("x")]
            if all(n % t == 0 for n, t in zip(dims[-3:], b)):
                out.append(k)
    return out


@pytest.mark.parametrize("dims", [(4, 2, 8, 16), (4, 2, 4, 16), (3, 4, 4, 16), (4, 4, 8, 32), (6, 8, 8, 16), (1, 4, 4, 8), (5, 8, 12, 24)])
def test_tma_kernels_match_oracle(torch, dims):
    m0, csw = -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 401)
    psi = wdinputs.spinor(dims, 402)
    C = wdinputs.selfcoupling_random(dims, 403)
    ref_c = oracle.apply(dims, m0, U, C, psi)
    ref_w = oracle.apply(dims, m0, U, None, psi)
    kids = tma_kernels(dims)
    assert kids
    for kid in kids:
        name = wd.wd_kernel_name(kid)
        with Op(torch, dims, m0, csw, U, C, kernel=kid) as op:
            err = rel_l2(op.apply(psi), ref_c)
            assert err <= TOL, (name, "clover", err)
        with Op(torch, dims, m0, 0.0, U, None, kernel=kid) as op:
            err = rel_l2(op.apply(psi), ref_w)
            assert err <= TOL, (name, "mass", err)
        with Op(torch, dims, m0, csw, U, C, kernel=kid, variant=1) as op:  # hopping kernel + S kernel
            err = rel_l2(op.apply(psi), ref_c)
            assert err <= TOL, (name, "unfused", err)


@pytest.mark.parametrize("tchunk", [1, 2, 3, 6, 12])
def test_tma_t_chunks_and_panels(torch, tchunk):
    dims, m0, csw = (12, 8, 16, 32), -0.4, 1.0
    U = wdinputs.gauge_exp(dims, 411, 0.5)
    psi = wdinputs.spinor(dims, 412)
    C = oracle.build_clover(dims, m0, csw, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    for kid in tma_kernels(dims):
        for zgroup in (0, 1, 2):
            with Op(torch, dims, m0, csw, U, C, kernel=kid, tchunk=tchunk, zgroup=zgroup) as op:
                out = op.apply(psi)
                assert rel_l2(out, ref) <= TOL, (wd.wd_kernel_name(kid), tchunk, zgroup)
                assert np.array_equal(op.apply(psi), out)  # deterministic


def test_tma_many_items_per_cta_and_multi_rhs(torch):
    """More work items than SMs (each CTA loops over several; barrier parities carry over), 3 RHS."""
    dims, m0, csw, nrhs = (4, 16, 32, 64), -0.4, 1.0, 3
    U = wdinputs.gauge_haar(dims, 421)
    psi = wdinputs.spinor(dims, 422, nrhs=nrhs)
    C = oracle.build_clover(dims, m0, csw, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    for kid in tma_kernels(dims):
        with Op(torch, dims, m0, csw, U, C, kernel=kid, tchunk=1) as op:
            assert rel_l2(op.apply(psi, nrhs), ref) <= TOL, wd.wd_kernel_name(kid)


@pytest.mark.parametrize("nrhs", [2, 4, 5, 12])
def test_quad_kernel_units_of_four_right_hand_sides(torch, nrhs):
    """tmq_*: one compute thread per (site, right-hand side), four right-hand sides per work item.  Full units, a partial
    last unit (its TMA boxes reach past the last right-hand side and are zero-filled; its threads must not store), every
    self-coupling mode, every right-hand side different."""
    dims, m0, csw = (6, 4, 8, 16), -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 431)
    psi = wdinputs.spinor(dims, 432, nrhs=nrhs)
    C = wdinputs.selfcoupling_random(dims, 433)
    ref_c = oracle.apply(dims, m0, U, C, psi)
    ref_w = oracle.apply(dims, m0, U, None, psi)
    kids = [k for k in tma_kernels(dims) if wd.wd_kernel_name(k).startswith("tmq_")]
    assert kids
    for kid in kids:
        for tchunk in (0, 1, 3):
            with Op(torch, dims, m0, csw, U, C, kernel=kid, tchunk=tchunk) as op:
                out = op.apply(psi, nrhs)
                for r in range(nrhs):
                    assert rel_l2(out[r], ref_c[r]) <= TOL, (wd.wd_kernel_name(kid), "clover", tchunk, r)
        with Op(torch, dims, m0, 0.0, U, None, kernel=kid) as op:
            assert rel_l2(op.apply(psi, nrhs), ref_w) <= TOL, (wd.wd_kernel_name(kid), "mass")


@pytest.mark.parametrize("nrhs", [1, 3, 4, 9, 12])
@pytest.mark.parametrize("dims", [(6, 4, 8, 16), (3, 2, 4, 8), (4, 6, 12, 24)])
def test_blocked_multi_rhs_layout(torch, dims, nrhs):
    """WD_OPT_RHS_BLOCK = 4: device spinors are double2 [unit][12][Vs][4]; pack / apply (tmqb_*) / unpack against the
    oracle for full and padded units, on lattices of one tile (every face wraps onto the tile itself) and of several,
    with clover term, mass term, T chunks of 1; every right-hand side different; bit-repeatable."""
    m0, csw = -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 451)
    psi = wdinputs.spinor(dims, 452, nrhs=nrhs).reshape(nrhs, -1, 12, 2)
    C = wdinputs.selfcoupling_random(dims, 453)
    ref_c = oracle.apply(dims, m0, U, C, psi).reshape(psi.shape)
    ref_w = oracle.apply(dims, m0, U, None, psi).reshape(psi.shape)
    for tchunk in (0, 1):
        with Op(torch, dims, m0, csw, U, C, rhs_block=4, tchunk=tchunk) as op:
            assert wd.wd_kernel_name(wd.wd_kernel_for(op.h, nrhs)).startswith("tmqb_")
            out = op.apply(psi, nrhs)
            for r in range(nrhs):
                assert rel_l2(out[r], ref_c[r]) <= TOL, ("clover", tchunk, r)
            assert np.array_equal(op.apply(psi, nrhs), out)
    with Op(torch, dims, m0, 0.0, U, None, rhs_block=4) as op:
        assert rel_l2(op.apply(psi, nrhs), ref_w) <= TOL, "mass"
        # the round trip through the blocked layout alone is exact
        d = op.dev_spinor(nrhs)
        wd.wd_pack_spinor(op.h, d, psi, nrhs)
        back = np.empty_like(psi)
        wd.wd_unpack_spinor(op.h, back, d, nrhs)
        assert np.array_equal(back, psi)


def test_blocked_layout_rules(torch):
    """What WD_OPT_RHS_BLOCK = 4 refuses: lattices its tile does not divide, kernels of the other layout, and the entry
    points that work on the plain layout."""
    with Op(torch, (4, 4, 4, 4), -0.4, 0.0) as op:
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, wd.WD_OPT_RHS_BLOCK, 4)
        assert wd.wd_get_option(op.h, wd.WD_OPT_RHS_BLOCK) == 1
    dims = (4, 2, 4, 8)
    U = wdinputs.gauge_haar(dims, 461)
    with Op(torch, dims, -0.4, 0.0, U) as op:
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id("tmqb_2x4x8"))  # plain handle, blocked kernel
        wd.wd_set_option(op.h, wd.WD_OPT_RHS_BLOCK, 4)
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id("tmb_4x4x8"))   # blocked handle, plain kernel
        psi = wdinputs.spinor(dims, 462)
        with pytest.raises(wd.WDError):
            wd.wd_apply_host(op.h, np.empty_like(psi), psi, 1)
        wd.wd_set_option(op.h, wd.WD_OPT_RHS_BLOCK, 1)
        out = np.empty_like(psi)
        wd.wd_apply_host(op.h, out, psi, 1)
        assert rel_l2(out, oracle.apply(dims, -0.4, U, None, psi)) <= TOL


@pytest.mark.parametrize("dims,csw", [((8, 4, 8, 16), 1.0), ((8, 4, 8, 16), 0.0), ((12, 8, 8, 32), 1.0), ((5, 4, 8, 16), 1.0)])
def test_apply_host_pipelined_over_t_chunks(torch, dims, csw):
    """wd_apply_host with a TMA kernel cuts the lattice into T chunks and overlaps upload, compute and download;
    each chunk is a launch restricted to a T range.  Against the oracle, and bit for bit against the serial path."""
    m0, nrhs = -0.4, 2
    U = wdinputs.gauge_haar(dims, 441)
    psi = wdinputs.spinor(dims, 442, nrhs=nrhs)
    C = oracle.build_clover(dims, m0, csw, U) if csw else None
    ref = oracle.apply(dims, m0, U, C, psi)
    # (lattices this small get the one-thread-per-site kernel automatically; the pipelined path needs a TMA kernel)
    with Op(torch, dims, m0, csw, U, C, kernel=wd.kernel_id("tmw_2x4x16" if csw else "tmb_2x4x16")) as op:
        assert wd.wd_kernel_name(wd.wd_kernel_in_use(op.h)).startswith(("tma_", "tmb_", "tmw_"))
        out = np.empty_like(psi)
        wd.wd_apply_host(op.h, out, psi, nrhs)
        assert rel_l2(out, ref) <= TOL
        pin_in = torch.from_numpy(psi).pin_memory()
        pin_out = torch.empty_like(pin_in).pin_memory()
        wd.wd_apply_host(op.h, pin_out, pin_in, nrhs)
        assert np.array_equal(pin_out.numpy(), out)
        wd.wd_set_option(op.h, wd.WD_OPT_HOST_PIPELINE, 0)
        ser = np.empty_like(psi)
        wd.wd_apply_host(op.h, ser, psi, nrhs)
        wd.wd_set_option(op.h, wd.WD_OPT_HOST_PIPELINE, 1)
        assert np.array_equal(ser, out)
        # the device path is untouched by the extra streams
        assert rel_l2(op.apply(psi, nrhs), ref) <= TOL
