"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bar: relative L2 error <= 1e-13 in FP64 (BASELINE.json north_star); where the
operation is a pure permutation (packers) the bar is bit-exact.

Run on a B200 with:  python -m pytest tests -m gpu
"""
import os

import numpy as np
import pytest

import oracle
import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import rel_l2

pytestmark = pytest.mark.gpu
TOL = 1e-13


@pytest.fixture(scope="module")
def torch():
    import torch as _torch

    if not _torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    _torch.cuda.init()
    return _torch


class Op:
    """Test helper: a handle plus torch-allocated device spinors (argument marshalling only)."""

    def __init__(self, torch, dims, m0, csw, U=None, C=None, build_clover=False, **opts):
        self.torch, self.dims, self.V = torch, dims, wdinputs.volume(dims)
        self.h = wd.wd_create(*dims, m0, csw)
        for k, v in opts.items():
            wd.wd_set_option(self.h, getattr(wd, "WD_OPT_" + k.upper()), v)
        wd.wd_set_stream(self.h, torch.cuda.current_stream().cuda_stream)
        if U is not None:
            wd.wd_load_gauge(self.h, U)
        if C is not None:
            wd.wd_load_clover(self.h, C)
        if build_clover:
            wd.wd_build_clover(self.h)

    def dev_spinor(self, nrhs=1):
        n = wd.wd_spinor_bytes(self.h, nrhs) // 8
        blk = wd.wd_get_option(self.h, wd.WD_OPT_RHS_BLOCK)  # blocked layout: units padded to blk right-hand sides
        assert n == -(-nrhs // blk) * blk * wd.wd_component_stride(self.h) * 24 and wd.wd_component_stride(self.h) >= self.V
        return self.torch.empty(n, dtype=self.torch.float64, device="cuda")

    def apply(self, psi, nrhs=1):
        """host canonical [nrhs][V][12][2] -> host canonical D psi, via pack / wd_apply / unpack."""
        psi = np.ascontiguousarray(psi, dtype=np.float64)
        din, dout = self.dev_spinor(nrhs), self.dev_spinor(nrhs)
        dout.fill_(float("nan"))
        wd.wd_pack_spinor(self.h, din, psi, nrhs)
        wd.wd_apply(self.h, dout, din, nrhs)
        wd.wd_synchronize(self.h)
        out = np.empty_like(psi)
        wd.wd_unpack_spinor(self.h, out, dout, nrhs)
        return out

    def close(self):
        if self.h:
            wd.wd_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()


def kernels_fitting(dims):
    out = []
    for k in range(wd.wd_kernel_count()):
        name = wd.wd_kernel_name(k)
        if name.startswith("linear"):
            out.append(k)
            continue
        if name.startswith("tmqb_"):  # written for the blocked multi-RHS layout (WD_OPT_RHS_BLOCK = 4): test_gpu_tma.py
            continue
        b = [int(v) for v in name.split("_")[1].split("x")]  # tile_TxZxYxX or tma_ZxYxX
        if all(n % t == 0 for n, t in zip(dims[-len(b):], b)):
            out.append(k)
    return out


# ---------------------------------------------------------------- BASELINE.json configs 1 and 2
def test_cfg1_4x4x4x4_wilson(torch):
    cfg = wdinputs.CONFIGS[1]
    dims = cfg["dims"]
    U = wdinputs.config_gauge(cfg)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    ref = oracle.apply(dims, cfg["m0"], U, None, psi)
    with Op(torch, dims, cfg["m0"], cfg["csw"], U) as op:
        assert rel_l2(op.apply(psi), ref) <= TOL


def test_cfg2_8x8x8x8_wilson_clover(torch):
    cfg = wdinputs.CONFIGS[2]
    dims = cfg["dims"]
    U = wdinputs.config_gauge(cfg)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U)
    ref = oracle.apply(dims, cfg["m0"], U, C, psi)
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, C) as op:  # S loaded from the host
        assert rel_l2(op.apply(psi), ref) <= TOL
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True) as op:  # S built on the device
        assert rel_l2(op.apply(psi), ref) <= TOL
        Cdev = np.empty_like(C)
        wd.wd_get_clover(op.h, Cdev)
        assert rel_l2(Cdev, C) <= TOL
        assert np.abs(Cdev[:, :12, 1]).max() == 0


# ---------------------------------------------------------------- every geometry, both variants
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (4, 8, 16, 64), (16, 4, 8, 32)])
def test_every_kernel_geometry_and_variant(torch, dims):
    m0, csw = -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 301)
    psi = wdinputs.spinor(dims, 302)
    C = wdinputs.selfcoupling_random(dims, 303)  # exercises all 42 entries independently
    ref_c = oracle.apply(dims, m0, U, C, psi)
    ref_w = oracle.apply(dims, m0, U, None, psi)
    kids = kernels_fitting(dims)
    assert len(kids) >= 5
    for kid in kids:
        for variant in (0, 1):
            with Op(torch, dims, m0, csw, U, C, kernel=kid, variant=variant) as op:
                assert wd.wd_kernel_in_use(op.h) == kid
                err = rel_l2(op.apply(psi), ref_c)
                assert err <= TOL, (wd.wd_kernel_name(kid), variant, err)
            with Op(torch, dims, m0, 0.0, U, None, kernel=kid, variant=variant) as op:
                err = rel_l2(op.apply(psi), ref_w)
                assert err <= TOL, (wd.wd_kernel_name(kid), variant, err)


@pytest.mark.parametrize("tchunk,zgroup", [(1, 1), (2, 2), (4, 1), (8, 0), (0, 2)])
def test_tiled_rasterisation_parameters(torch, tchunk, zgroup):
    dims, m0 = (8, 16, 8, 16), -0.4
    U = wdinputs.gauge_haar(dims, 311)
    psi = wdinputs.spinor(dims, 312)
    C = oracle.build_clover(dims, m0, 1.0, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    for name in ("tile_1x4x4x16",):
        if tchunk == 1 and name.startswith("tile_2"):
            continue
        with Op(torch, dims, m0, 1.0, U, C, kernel=wd.kernel_id(name), tchunk=tchunk, zgroup=zgroup) as op:
            assert rel_l2(op.apply(psi), ref) <= TOL, name


# ---------------------------------------------------------------- ragged / degenerate lattices
@pytest.mark.parametrize("dims", [(2, 2, 2, 2), (1, 1, 1, 1), (1, 2, 1, 3), (3, 5, 6, 7), (2, 4, 2, 4),
                                  (5, 3, 2, 33), (4, 4, 4, 65)])
def test_ragged_and_degenerate_extents(torch, dims):
    """n = 2 (x+mu == x-mu), n = 1, odd extents, a ragged last CTA: only the linear geometry fits."""
    m0, csw = -0.3, 1.2
    U = wdinputs.gauge_exp(dims, 321, 0.6)
    psi = wdinputs.spinor(dims, 322)
    C = oracle.build_clover(dims, m0, csw, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    with Op(torch, dims, m0, csw, U, build_clover=True) as op:
        assert wd.wd_kernel_name(wd.wd_kernel_in_use(op.h)).startswith("linear") or all(
            n % 4 == 0 for n in dims)
        assert rel_l2(op.apply(psi), ref) <= TOL
    with Op(torch, dims, m0, 0.0, U, kernel=0) as op:
        assert rel_l2(op.apply(psi), oracle.apply(dims, m0, U, None, psi)) <= TOL


# ---------------------------------------------------------------- multi-RHS
def test_multi_rhs_equals_repeated_single_rhs(torch):
    dims, m0, csw, nrhs = (8, 8, 8, 8), -0.4, 1.0, 5
    U = wdinputs.gauge_haar(dims, 331)
    psi = wdinputs.spinor(dims, 332, nrhs=nrhs)
    C = oracle.build_clover(dims, m0, csw, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    with Op(torch, dims, m0, csw, U, C) as op:
        out = op.apply(psi, nrhs)
        for r in range(nrhs):
            assert rel_l2(out[r], ref[r]) <= TOL
            single = op.apply(psi[r:r + 1])[0]
            if wd.wd_kernel_for(op.h, nrhs) == wd.wd_kernel_for(op.h, 1):
                assert np.array_equal(out[r], single)  # same kernel: same arithmetic, bit for bit
            else:  # the automatic choice differs for several right-hand sides: only the summation order may differ
                assert rel_l2(out[r], single) <= 1e-14


# ---------------------------------------------------------------- packers, host path, options
def test_pack_unpack_roundtrip_and_device_pack_bit_exact(torch):
    dims, m0, csw = (4, 8, 4, 20), -0.4, 1.0
    V = wdinputs.volume(dims)
    U = wdinputs.gauge_haar(dims, 341)
    psi = wdinputs.spinor(dims, 342, nrhs=2)
    C = wdinputs.selfcoupling_random(dims, 343)
    outs = []
    for device_pack in (0, 1):
        with Op(torch, dims, m0, csw, device_pack=device_pack) as op:
            wd.wd_load_gauge(op.h, U)
            wd.wd_load_clover(op.h, C)
            d = op.dev_spinor(2)
            wd.wd_pack_spinor(op.h, d, psi, 2)
            # the device image is the host packer's image, bit for bit
            img = np.empty((12, V, 2))
            wd.wd_layout_pack_host(wd.WD_FIELD_SPINOR, V, psi[1], img)
            Vs = wd.wd_component_stride(op.h)
            assert np.array_equal(d.cpu().numpy().reshape(2, 12, Vs, 2)[1, :, :V], img)
            back = np.empty_like(psi)
            wd.wd_unpack_spinor(op.h, back, d, 2)
            assert np.array_equal(back, psi)
            Cb = np.empty_like(C)
            wd.wd_get_clover(op.h, Cb)
            assert np.array_equal(Cb, C)
            outs.append(op.apply(psi, 2))
    assert np.array_equal(outs[0], outs[1])


def test_apply_host_matches_oracle(torch):
    dims, m0, csw = (8, 4, 8, 12), -0.4, 1.0
    U = wdinputs.gauge_haar(dims, 351)
    psi = wdinputs.spinor(dims, 352, nrhs=2)
    C = oracle.build_clover(dims, m0, csw, U)
    ref = oracle.apply(dims, m0, U, C, psi)
    with Op(torch, dims, m0, csw, U, C) as op:
        out = np.empty_like(psi)
        wd.wd_apply_host(op.h, out, psi, 2)
        assert rel_l2(out, ref) <= TOL
        pin_in = torch.from_numpy(psi).pin_memory()
        pin_out = torch.empty_like(pin_in).pin_memory()
        wd.wd_apply_host(op.h, pin_out, pin_in, 2)
        assert np.array_equal(pin_out.numpy(), out)


def test_non_default_stream_and_launch_count(torch):
    dims, m0 = (4, 4, 8, 16), -0.5
    U = wdinputs.gauge_haar(dims, 361)
    psi = wdinputs.spinor(dims, 362)
    ref = oracle.apply(dims, m0, U, None, psi)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        with Op(torch, dims, m0, 0.0, U) as op:
            n0 = wd.wd_launch_count(op.h)
            assert rel_l2(op.apply(psi), ref) <= TOL
            assert wd.wd_launch_count(op.h) == n0 + 1
            wd.wd_set_option(op.h, wd.WD_OPT_VARIANT, 1)
            assert rel_l2(op.apply(psi), ref) <= TOL
            assert wd.wd_launch_count(op.h) == n0 + 3


def test_error_reporting(torch):
    dims = (4, 4, 4, 4)
    U = wdinputs.gauge_haar(dims, 371)
    with Op(torch, dims, -0.4, 1.0) as op:
        a, b = op.dev_spinor(), op.dev_spinor()
        with pytest.raises(wd.WDError) as e:
            wd.wd_apply(op.h, a, b)
        assert e.value.code == wd.WD_ESTATE and "gauge" in str(e.value)
        with pytest.raises(wd.WDError) as e:
            wd.wd_build_clover(op.h)
        assert e.value.code == wd.WD_ESTATE
        wd.wd_load_gauge(op.h, U)
        with pytest.raises(wd.WDError) as e:
            wd.wd_apply(op.h, a, b)
        assert e.value.code == wd.WD_ESTATE and "self-coupling" in str(e.value)
        wd.wd_build_clover(op.h)
        wd.wd_apply(op.h, a, b)
        for bad in ((a, a, 1), (a, b, 0), (None, b, 1)):
            with pytest.raises(wd.WDError) as e:
                wd.wd_apply(op.h, *bad)
            assert e.value.code == wd.WD_EINVAL
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id("tile_1x4x4x16"))  # 16 does not divide 4
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, 99, 0)


def test_golden_fixture_on_gpu(torch):
    from test_golden import check_against_golden, golden_module

    mod = golden_module()
    U, psi, C, _, _ = mod.compute()
    with Op(torch, mod.DIMS, mod.M0, mod.CSW, U, build_clover=True) as op:
        out_c = op.apply(psi[None])[0]
    with Op(torch, mod.DIMS, mod.M0, 0.0, U) as op:
        out_w = op.apply(psi[None])[0]
    check_against_golden(out_c, out_w, psi, tol=1e-12)


# ---------------------------------------------------------------- linearity on the device, cfg 3 size
def test_cfg3_32x32x32x32_first_apply_and_repeatability(torch):
    cfg = wdinputs.CONFIGS[3]
    dims = cfg["dims"]
    U = wdinputs.config_gauge(cfg)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U)
    ref = oracle.apply(dims, cfg["m0"], U, C, psi)
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True) as op:
        out = op.apply(psi)
        assert rel_l2(out, ref) <= TOL
        assert np.array_equal(op.apply(psi), out)  # deterministic, no atomics
        for kid in kernels_fitting(dims):
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, kid)
            assert rel_l2(op.apply(psi), ref) <= TOL, wd.wd_kernel_name(kid)


# ---------------------------------------------------------------- R11, state handling
def gauge_gaussian(dims, seed):
    """General 3x3 complex links, NOT unitary (R11; as tests/test_oracle_pins.py P2): Re, Im ~ N(0, 1/2)."""
    V = wdinputs.volume(dims)
    return (wdinputs.gaussian(V * 72, seed) * 0.5).reshape(V, 4, 3, 3, 2)


@pytest.mark.parametrize("dims", [(4, 4, 8, 16), (3, 5, 6, 7)])
def test_non_unitary_links(torch, dims):
    """wd.h promises "general 3x3 complex" links (U and U^H are used, never U^-1): every kernel that fits, clover built
    on the device from those links and by the oracle, one and several right-hand sides."""
    m0, csw, nrhs = -0.4, 1.0, 3
    U = gauge_gaussian(dims, 381)
    psi = wdinputs.spinor(dims, 382, nrhs=nrhs)
    C = oracle.build_clover(dims, m0, csw, U)
    ref_c = oracle.apply(dims, m0, U, C, psi)
    ref_w = oracle.apply(dims, m0, U, None, psi)
    for kid in kernels_fitting(dims):
        with Op(torch, dims, m0, csw, U, build_clover=True, kernel=kid) as op:
            Cdev = np.empty_like(C)
            wd.wd_get_clover(op.h, Cdev)
            assert rel_l2(Cdev, C) <= TOL
            assert rel_l2(op.apply(psi, nrhs), ref_c) <= TOL, wd.wd_kernel_name(kid)
        with Op(torch, dims, m0, 0.0, U, kernel=kid) as op:
            assert rel_l2(op.apply(psi, nrhs), ref_w) <= TOL, wd.wd_kernel_name(kid)


def test_load_clover_on_a_csw0_handle(torch):
    """wd.h: wd_load_clover is allowed with csw == 0; the loaded S then replaces (m0+4) I."""
    dims, m0 = (4, 4, 8, 16), -0.4
    U = wdinputs.gauge_haar(dims, 385)
    psi = wdinputs.spinor(dims, 386)
    C = wdinputs.selfcoupling_random(dims, 387)
    with Op(torch, dims, m0, 0.0, U) as op:
        assert rel_l2(op.apply(psi), oracle.apply(dims, m0, U, None, psi)) <= TOL
        wd.wd_load_clover(op.h, C)
        assert rel_l2(op.apply(psi), oracle.apply(dims, m0, U, C, psi)) <= TOL
        assert rel_l2(op.apply(np.concatenate([psi, psi]), 2)[1], oracle.apply(dims, m0, U, C, psi)[0]) <= TOL


def test_reloading_the_gauge_field_invalidates_a_built_clover(torch):
    """A second wd_load_gauge must not leave S built from the previous links in use."""
    dims, m0, csw = (4, 4, 8, 16), -0.4, 1.0
    U1, U2 = wdinputs.gauge_haar(dims, 391), wdinputs.gauge_haar(dims, 392)
    psi = wdinputs.spinor(dims, 393)
    with Op(torch, dims, m0, csw, U1, build_clover=True) as op:
        ref1 = oracle.apply(dims, m0, U1, oracle.build_clover(dims, m0, csw, U1), psi)
        assert rel_l2(op.apply(psi), ref1) <= TOL
        wd.wd_load_gauge(op.h, U2)
        with pytest.raises(wd.WDError) as e:
            op.apply(psi)
        assert e.value.code == wd.WD_ESTATE
        wd.wd_build_clover(op.h)
        C2 = oracle.build_clover(dims, m0, csw, U2)
        assert rel_l2(op.apply(psi), oracle.apply(dims, m0, U2, C2, psi)) <= TOL
        # a field the caller supplied is the caller's: it survives a new gauge field
        wd.wd_load_clover(op.h, C2)
        wd.wd_load_gauge(op.h, U1)
        assert rel_l2(op.apply(psi), oracle.apply(dims, m0, U1, C2, psi)) <= TOL


# ---------------------------------------------------------------- full size, bench configuration
def _require_memory(torch, host_gb, dev_gb, what):
    """The full-size tests never shrink silently: WD_TEST_SMALL=1 asks for the reduced size explicitly (and the
    test says so in its output); otherwise too little memory is a FAILURE, not a fallback."""
    import psutil

    if os.environ.get("WD_TEST_SMALL"):
        return False
    free_host, free_dev = psutil.virtual_memory().available, torch.cuda.mem_get_info()[0]
    if free_host < host_gb * 1e9 or free_dev < dev_gb * 1e9:
        pytest.fail(f"{what}: needs {host_gb} GB of host and {dev_gb} GB of device memory, found "
                    f"{free_host / 1e9:.0f} / {free_dev / 1e9:.0f} GB (set WD_TEST_SMALL=1 to run the reduced size)")
    return True


def _report(capsys, text):
    with capsys.disabled():
        print("\n[full-size parity] " + text, flush=True)


def test_cfg4_full_size_whole_lattice(torch, capsys):
    """64^4 Wilson-clover in the launch configuration bench.py times (automatic kernel, S built on the device,
    device-side pack), compared with the oracle on EVERY site: rel. L2 and the worst component."""
    cfg = wdinputs.CONFIGS[4]
    full = _require_memory(torch, 45, 40, "cfg 4 (64^4)")
    dims = cfg["dims"] if full else (32, 32, 32, 64)
    U = wdinputs.config_gauge(cfg, dims)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True, device_pack=1) as op:
        kname = wd.wd_kernel_name(wd.wd_kernel_in_use(op.h))
        out = op.apply(psi)
    C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U)
    ref = oracle.apply(dims, cfg["m0"], U, C, psi)
    del U, C
    assert np.isfinite(out).all()
    err = rel_l2(out, ref)
    worst = float(np.abs(out - ref).max() / np.abs(ref).max())
    _report(capsys, f"lattice {'x'.join(map(str, dims))} nrhs 1 kernel {kname}: {out.size // 24} sites compared, "
                    f"rel_l2 {err:.3e}, worst component {worst:.3e}" + ("" if full else "  (WD_TEST_SMALL)"))
    assert err <= TOL and worst <= 1e-13


def test_cfg5_full_size_multi_rhs_whole_lattice(torch, capsys):
    """48^3 x 96 Wilson-clover with 12 right-hand sides in ONE wd_apply (the launch configurations bench.py --config 5
    times: S built on the device; the blocked multi-RHS layout with its kernel, and the plain layout with the automatic
    kernel), EVERY right-hand side compared with the oracle on EVERY site.  The host streams one unit of four right-hand
    sides at a time through the oracle."""
    cfg = wdinputs.CONFIGS[5]
    full = _require_memory(torch, 40, 100, "cfg 5 (48^3 x 96, 12 RHS)")
    dims, nrhs = (cfg["dims"], cfg["nrhs"]) if full else ((24, 16, 16, 48), 5)
    V = wdinputs.volume(dims)
    U = wdinputs.config_gauge(cfg, dims)
    units = [list(range(u, min(u + 4, nrhs))) for u in range(0, nrhs, 4)]
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True, device_pack=1) as op:
        Vs = wd.wd_component_stride(op.h)
        outs, knames = {}, {}
        for layout in (1, 4):
            wd.wd_set_option(op.h, wd.WD_OPT_RHS_BLOCK, layout)
            knames[layout] = wd.wd_kernel_name(wd.wd_kernel_for(op.h, nrhs))
            din, dout = op.dev_spinor(nrhs), op.dev_spinor(nrhs)
            dout.fill_(float("nan"))
            for rs in units:  # one unit at a time: generate, pack into its slots (a unit is contiguous in both layouts)
                psi_u = np.concatenate([wdinputs.spinor(dims, cfg["spinor_seed"] + r) for r in rs])
                wd.wd_pack_spinor(op.h, din[rs[0] * 24 * Vs:], psi_u, len(rs))
            wd.wd_apply(op.h, dout, din, nrhs)
            wd.wd_synchronize(op.h)
            outs[layout] = dout
            del din
        assert knames[4].startswith("tmqb_")
        C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U)
        errs, worsts = {1: [], 4: []}, {1: [], 4: []}
        for rs in units:
            ref = np.concatenate([oracle.apply(dims, cfg["m0"], U, C, wdinputs.spinor(dims, cfg["spinor_seed"] + r)) for r in rs])
            out_u = np.empty_like(ref)
            for layout in (1, 4):
                wd.wd_set_option(op.h, wd.WD_OPT_RHS_BLOCK, layout)
                wd.wd_unpack_spinor(op.h, out_u, outs[layout][rs[0] * 24 * Vs:], len(rs))
                assert np.isfinite(out_u).all(), (layout, rs)
                for k in range(len(rs)):
                    errs[layout].append(rel_l2(out_u[k], ref[k]))
                    worsts[layout].append(float(np.abs(out_u[k] - ref[k]).max() / np.abs(ref[k]).max()))
    for layout in (1, 4):
        _report(capsys, f"lattice {'x'.join(map(str, dims))} x{nrhs} kernel {knames[layout]} ({'blocked' if layout == 4 else 'plain'} layout): "
                        f"{nrhs} x {V} sites compared, max rel_l2 {max(errs[layout]):.3e}, worst component {max(worsts[layout]):.3e}"
                        + ("" if full else "  (WD_TEST_SMALL)"))
        assert len(errs[layout]) == nrhs and max(errs[layout]) <= TOL and max(worsts[layout]) <= 1e-13


# ---------------------------------------------------------------- two-row gauge storage (opt-in)
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (6, 4, 12, 32)])
def test_two_row_gauge_storage_on_su3_links(torch, dims):
    """WD_OPT_GAUGE_ROWS = 2: the fused TMA kernel reads rows 0, 1 of every link and rebuilds row 2 as the conjugate
    cross product — exact for SU(3) links up to rounding, so the 1e-13 bar holds on Haar and exp(i eps H) links; set
    before or after the gauge field is loaded; switching back restores the nine-entry path bit for bit."""
    m0, csw = -0.4, 1.0
    for U in (wdinputs.gauge_haar(dims, 901), wdinputs.gauge_exp(dims, 902, 0.5)):
        psi = wdinputs.spinor(dims, 903, nrhs=2)
        C = oracle.build_clover(dims, m0, csw, U)
        ref = oracle.apply(dims, m0, U, C, psi)
        with Op(torch, dims, m0, csw, U, C, kernel=wd.kernel_id("tma_2x4x16")) as op:
            full = op.apply(psi, 2)
            wd.wd_set_option(op.h, wd.WD_OPT_GAUGE_ROWS, 2)  # after the load
            two = op.apply(psi, 2)
            assert rel_l2(two, ref) <= TOL and not np.array_equal(two, full)
            wd.wd_set_option(op.h, wd.WD_OPT_GAUGE_ROWS, 3)
            assert np.array_equal(op.apply(psi, 2), full)
        with Op(torch, dims, m0, 0.0, gauge_rows=2, kernel=wd.kernel_id("tma_2x4x16")) as op:  # before the load, pure Wilson
            wd.wd_load_gauge(op.h, U)
            assert rel_l2(op.apply(psi, 2), oracle.apply(dims, m0, U, None, psi)) <= TOL
    with Op(torch, dims, m0, 0.0) as op:
        with pytest.raises(wd.WDError):
            wd.wd_set_option(op.h, wd.WD_OPT_GAUGE_ROWS, 1)
