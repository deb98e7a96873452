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
        assert n == nrhs * wd.wd_component_stride(self.h) * 24 and wd.wd_component_stride(self.h) >= self.V
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
    assert len(kids) >= 6
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
    for name in ("tile_1x4x4x16", "tile_2x4x4x8", "tile_1x4x4x8"):
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
    with Op(torch, dims, m0, 0.0, U, kernel=1) as op:
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


# ---------------------------------------------------------------- full size, bench configuration
def _full_size_dims():
    import psutil

    free_host = psutil.virtual_memory().available
    return (64, 64, 64, 64) if free_host > 40e9 and not os.environ.get("WD_TEST_SMALL") else (32, 32, 32, 64)


def test_cfg4_full_size_sampled_outputs(torch):
    """64^4 Wilson-clover in the launch configuration bench.py times (automatic kernel, S built on
    the device), checked on sampled sites the oracle computes one by one from (U, psi) alone."""
    cfg = wdinputs.CONFIGS[4]
    dims = _full_size_dims()
    if torch.cuda.mem_get_info()[0] < 40e9:
        dims = (32, 32, 32, 64)
    V = wdinputs.volume(dims)
    U = wdinputs.gauge_haar(dims, cfg["gauge"][1])
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    rng = np.random.default_rng(4)
    T, Z, Y, X = dims
    corners = [0, V - 1, X - 1, X, Y * X - 1, Z * Y * X - 1, Z * Y * X, (T - 1) * Z * Y * X, V - X, V // 2, V // 2 + X - 1]
    sites = np.unique(np.concatenate([np.array(corners), rng.integers(0, V, size=4000)])).astype(np.int64)
    ref = oracle.apply_sites(dims, cfg["m0"], cfg["csw"], U, psi[0], sites)
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True, device_pack=1) as op:
        del U
        out = op.apply(psi)[0]
        assert np.isfinite(out).all()
        assert rel_l2(out[sites], ref) <= TOL
        worst = np.abs(out[sites] - ref).max() / np.abs(ref).max()
        assert worst <= 1e-13


def test_cfg5_full_size_multi_rhs_sampled_outputs(torch):
    """48^3 x 96 Wilson-clover with 12 right-hand sides in ONE wd_apply (the launch configuration bench.py
    --config 5 times: automatic kernel, RHS-blocked item order, S built on the device), checked on sampled
    sites of every right-hand side that the oracle computes one by one from (U, psi_r) alone.  The host
    streams one RHS at a time through the oracle."""
    import psutil

    cfg = wdinputs.CONFIGS[5]
    dims, nrhs = cfg["dims"], cfg["nrhs"]
    if psutil.virtual_memory().available < 80e9 or torch.cuda.mem_get_info()[0] < 80e9 or os.environ.get("WD_TEST_SMALL"):
        dims, nrhs = (24, 16, 16, 48), 5
    V = wdinputs.volume(dims)
    T, Z, Y, X = dims
    U = wdinputs.gauge_haar(dims, cfg["gauge"][1])
    rng = np.random.default_rng(5)
    corners = [0, V - 1, X - 1, X, Y * X - 1, Z * Y * X - 1, Z * Y * X, (T - 1) * Z * Y * X, V - X, V // 2]
    sites = np.unique(np.concatenate([np.array(corners), rng.integers(0, V, size=600)])).astype(np.int64)
    with Op(torch, dims, cfg["m0"], cfg["csw"], U, build_clover=True, device_pack=1) as op:
        Vs = wd.wd_component_stride(op.h)
        din, dout = op.dev_spinor(nrhs), op.dev_spinor(nrhs)
        dout.fill_(float("nan"))
        refs = []
        for r in range(nrhs):  # one RHS at a time: generate, pack into its slot, keep only the sampled reference
            psi_r = wdinputs.spinor(dims, cfg["spinor_seed"] + r)
            wd.wd_pack_spinor(op.h, din[r * 24 * Vs:(r + 1) * 24 * Vs], psi_r, 1)
            refs.append(oracle.apply_sites(dims, cfg["m0"], cfg["csw"], U, psi_r[0], sites))
            del psi_r
        wd.wd_apply(op.h, dout, din, nrhs)
        wd.wd_synchronize(op.h)
        out_r = np.empty((1, V, 12, 2))
        for r in range(nrhs):
            wd.wd_unpack_spinor(op.h, out_r, dout[r * 24 * Vs:(r + 1) * 24 * Vs], 1)
            assert np.isfinite(out_r).all(), r
            assert rel_l2(out_r[0][sites], refs[r]) <= TOL, r
