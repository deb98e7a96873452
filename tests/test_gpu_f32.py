"""GPU parity of the FP32 variant (csrc/wd_f32.cu) against the FP64 oracle evaluated on the
SAME single-precision-rounded inputs, so that only the FP32 arithmetic of the kernel is measured.

Tolerance: every output component is a sum of at most 8*6 + 12 products of
O(1) numbers accumulated with FMA in FP32 (unit roundoff u = 2^-24 = 6e-8); worst case ~ 60 u = 3.6e-6 per component
relative to the component scale, ~ sqrt(60) u = 5e-7 typical; the L2 norm averages it to ~ 2e-7.  Bars written here:
relative L2 <= 1e-6, worst component <= 5e-6 of the largest reference component.
"""
import numpy as np
import pytest

import oracle
import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import rel_l2
from test_gpu_parity import Op, torch  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu
TOL32, WORST32 = 1e-6, 5e-6


def r32(a):
    return np.ascontiguousarray(a, dtype=np.float32).astype(np.float64)


def apply_f32(torch, op, psi, nrhs):
    """host canonical FP64 psi -> device FP64 layout -> FP32 layout -> wd_apply_f32 -> back, all conversions on device"""
    d64, o64 = op.dev_spinor(nrhs), op.dev_spinor(nrhs)
    n32 = wd.wd_spinor_bytes_f32(op.h, nrhs) // 4
    assert n32 == d64.numel()  # same element count, half the bytes
    d32 = torch.empty(n32, dtype=torch.float32, device="cuda")
    o32 = torch.full((n32,), float("nan"), dtype=torch.float32, device="cuda")
    wd.wd_pack_spinor(op.h, d64, psi, nrhs)
    wd.wd_convert_spinor(op.h, d32, d64, nrhs, True)
    wd.wd_apply_f32(op.h, o32, d32, nrhs)
    wd.wd_convert_spinor(op.h, o64, o32, nrhs, False)
    wd.wd_synchronize(op.h)
    out = np.empty_like(psi)
    wd.wd_unpack_spinor(op.h, out, o64, nrhs)
    return out


@pytest.mark.parametrize("f32_kernel", [0, 1])
@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (4, 4, 8, 32), (5, 2, 4, 16), (3, 5, 6, 7), (2, 2, 2, 2)])
def test_fp32_operator_matches_the_oracle_on_rounded_inputs(torch, dims, f32_kernel):
    """f32_kernel 0: automatic (the TMA kernel on 8-byte elements where its tile fits, else the LDG kernels); 1: LDG."""
    m0, csw, nrhs = -0.4, 1.0, 3
    U = wdinputs.gauge_exp(dims, 911, 0.5)
    psi = wdinputs.spinor(dims, 912, nrhs=nrhs)
    C = oracle.build_clover(dims, m0, csw, U)
    ref_c = oracle.apply(dims, m0, r32(U), r32(C), r32(psi))
    ref_w = oracle.apply(dims, m0, r32(U), None, r32(psi))
    with Op(torch, dims, m0, csw, U, build_clover=True) as op:
        a, b = op.dev_spinor(), op.dev_spinor()
        with pytest.raises(wd.WDError) as e:
            wd.wd_apply_f32(op.h, a, b, 1)
        assert e.value.code == wd.WD_ESTATE
        wd.wd_enable_f32(op.h)
        wd.wd_set_option(op.h, wd.WD_OPT_F32_KERNEL, f32_kernel)
        out = apply_f32(torch, op, psi, nrhs)
        assert np.isfinite(out).all()
        assert rel_l2(out, ref_c) <= TOL32
        assert np.abs(out - ref_c).max() <= WORST32 * np.abs(ref_c).max()
        # it IS single precision: the FP64 path is a million times closer to the unrounded reference
        assert rel_l2(out, ref_c) > 1e-9
        with pytest.raises(wd.WDError):
            wd.wd_apply_f32(op.h, a, a, 1)
    with Op(torch, dims, m0, 0.0, U, f32_kernel=f32_kernel) as op:
        wd.wd_enable_f32(op.h)
        out = apply_f32(torch, op, psi, nrhs)
        assert rel_l2(out, ref_w) <= TOL32 and np.abs(out - ref_w).max() <= WORST32 * np.abs(ref_w).max()


def test_convert_is_ieee_rounding_and_open_boundaries_work_in_fp32(torch):
    dims = (4, 4, 4, 16)
    psi = wdinputs.spinor(dims, 921)
    with Op(torch, dims, -0.4, 0.0, wdinputs.gauge_haar(dims, 922)) as op:
        d64, b64 = op.dev_spinor(), op.dev_spinor()
        d32 = torch.empty(d64.numel(), dtype=torch.float32, device="cuda")
        wd.wd_pack_spinor(op.h, d64, psi, 1)
        wd.wd_convert_spinor(op.h, d32, d64, 1, True)
        wd.wd_convert_spinor(op.h, b64, d32, 1, False)
        back = np.empty_like(psi)
        wd.wd_unpack_spinor(op.h, back, b64, 1)
        assert np.array_equal(back, r32(psi))


def test_fp32_copies_go_stale_when_the_fp64_fields_change(torch):
    """wd_enable_f32 copies the links and S as they are; after wd_load_gauge / wd_load_clover / wd_build_clover the copies
    describe the OLD operator, so wd_apply_f32 and wd_gmres_mixed refuse (WD_ESTATE) until wd_enable_f32 is called again."""
    dims, m0, csw = (4, 4, 8, 16), -0.2, 1.0
    U1, U2 = wdinputs.gauge_exp(dims, 921, 0.5), wdinputs.gauge_exp(dims, 922, 0.5)
    psi = wdinputs.spinor(dims, 923)
    with Op(torch, dims, m0, csw, U1, build_clover=True) as op:
        wd.wd_enable_f32(op.h)
        out1 = apply_f32(torch, op, psi, 1)
        wd.wd_load_gauge(op.h, U2)
        wd.wd_build_clover(op.h)
        n32 = wd.wd_spinor_bytes_f32(op.h, 1) // 4
        a, b = torch.zeros(n32, dtype=torch.float32, device="cuda"), torch.zeros(n32, dtype=torch.float32, device="cuda")
        with pytest.raises(wd.WDError) as e:
            wd.wd_apply_f32(op.h, a, b, 1)
        assert e.value.code == wd.WD_ESTATE and "stale" in str(e.value)
        x, y = op.dev_spinor(), op.dev_spinor()
        x.zero_()
        wd.wd_pack_spinor(op.h, y, psi, 1)
        with pytest.raises(wd.WDError) as e:
            wd.wd_gmres_mixed(op.h, x, y, 4, 2, 1e-6)
        assert e.value.code == wd.WD_ESTATE
        wd.wd_enable_f32(op.h)
        out2 = apply_f32(torch, op, psi, 1)
        C2 = oracle.build_clover(dims, m0, csw, U2)
        assert rel_l2(out2, oracle.apply(dims, m0, r32(U2), r32(C2), r32(psi))) <= TOL32
        assert rel_l2(out1, out2) > 1e-2  # it really is another operator
