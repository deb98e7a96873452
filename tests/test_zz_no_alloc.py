"""wd_inner_product_static (include/wd.h, "an entry point that allocates nothing").

Some users of libwd cannot let the library call cudaMalloc at the moment they need an inner product or a norm: a
solver running under PyTorch, whose caching allocator already owns nearly all of the GPU's memory; an iteration loop
between two operator applications, where cudaMalloc / cudaFree would stall the whole device.  For them the library has
one reduction whose scratch (per-block partial sums and completion counters) is a fixed 65 792-byte array inside the
library image instead of cudaMalloc'ed memory: at most 64 right-hand sides per call, every call on a device shares the
array, and the first call on a device looks the array's device address up.

The GPU test checks it against the path that existed before — the reductions inside wd_gmres, whose scratch is
cudaMalloc'ed — on two calls in a row, so that a call which relied on a freshly zeroed array, or was upset by what the
previous call left in it, fails.  This file is named test_zz_* so that pytest collects it last: under `pytest -x` a
failure here hides no other test.  It passes alone in a fresh process (its first call is then the one that does the
per-device set-up) and after the other tests.
"""
import ctypes

import numpy as np
import pytest

import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import c

TOL = 1e-13  # the parity bar of tests/test_gpu_parity.py (relative, FP64)
MAX_NRHS = 64  # the limit include/wd.h states


def test_sizes_beyond_the_scratch_array_are_refused_with_a_clear_error():
    """Argument errors are found before any CUDA call, so this runs without a GPU."""
    L = wd.lib()
    fake = ctypes.c_void_p(256)  # never dereferenced: the call is refused first
    assert L.wd_inner_product_static(fake, fake, 16, 16, MAX_NRHS + 1, fake, None) == wd.WD_EINVAL
    text = wd.wd_last_error(None)
    assert "wd_inner_product_static" in text and "65" in text and "maximum of 64" in text and "split the call" in text
    assert L.wd_inner_product_static(None, fake, 16, 16, 1, fake, None) == wd.WD_EINVAL
    assert L.wd_inner_product_static(fake, fake, 16, 8, 1, fake, None) == wd.WD_EINVAL  # Vs < V
    assert L.wd_inner_product_static(fake, fake, 16, 16, 0, fake, None) == wd.WD_EINVAL
    assert L.wd_inner_product_static(ctypes.c_void_p(8), fake, 16, 16, 1, fake, None) == wd.WD_EINVAL  # misaligned
    with pytest.raises(wd.WDError):
        wd.wd_inner_product_static(256, 256, 16, 16, 1000, 256)


@pytest.mark.gpu
def test_static_scratch_inner_product_matches_the_reductions_of_wd_gmres_twice_in_a_row():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    from test_gpu_parity import Op

    # 6 x 10 x 12 x 20 = 14 400 sites: eight blocks per component with a ragged last one, odd against every tile
    dims, m0 = (6, 10, 12, 20), 0.2
    U = wdinputs.gauge_haar(dims, 4101)
    b = wdinputs.spinor(dims, 4102)
    with Op(torch, dims, m0, 0.0, U) as op:
        V, Vs = op.V, wd.wd_component_stride(op.h)
        stream = torch.cuda.current_stream().cuda_stream
        db, dx, dAb = op.dev_spinor(), op.dev_spinor(), op.dev_spinor()
        wd.wd_pack_spinor(op.h, db, b, 1)

        # --- the existing path: wd_gmres's own reductions (cudaMalloc'ed scratch) -------------------------------
        # ||b||: the residual norm of x_0 = 0 (Algorithm 1 lines 4-5; no cycle is run)
        dx.zero_()
        hist = np.full(1, np.nan)
        assert wd.wd_gmres(op.h, dx, db, 1, 0, 1e-10, hist) == 0
        norm_gmres = float(hist[0])
        # h_11 = v_1^H D v_1 with v_1 = b / ||b||: one cycle of GMRES(1) from x_0 = 0 (lines 6-11)
        dx.zero_()
        hist2 = np.full(2, np.nan)
        assert wd.wd_gmres(op.h, dx, db, 1, 1, 1e-10, hist2) == 1
        H = np.zeros((2, 2))
        kdim, _ = wd.wd_gmres_last_hessenberg(op.h, H)
        assert kdim == 1
        h11_gmres = complex(H[0, 0], H[0, 1])
        wd.wd_apply(op.h, dAb, db, 1)
        wd.wd_synchronize(op.h)

        # --- the new entry point, two calls in a row on one stream, different operands --------------------------
        res = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
        wd.wd_inner_product_static(db, db, V, Vs, 1, res[0:2], stream)   # <b, b>
        wd.wd_inner_product_static(db, dAb, V, Vs, 1, res[2:4], stream)  # <b, D b>
        torch.cuda.synchronize()
        r = res.cpu().numpy()
        bb, bAb = complex(r[0], r[1]), complex(r[2], r[3])

        assert abs(bb.imag) <= TOL * bb.real  # the two FMA-rounded cross terms of conj(b) b need not cancel to the last bit
        assert abs(np.sqrt(bb.real) - norm_gmres) <= TOL * norm_gmres
        # h_11 = <b, D b> / ||b||^2; the error scale of an inner product is ||b|| ||D b||, not |h_11|
        bc, Abc = c(b).ravel(), None
        out = np.empty_like(b)
        wd.wd_unpack_spinor(op.h, out, dAb, 1)
        Abc = c(out).ravel()
        scale = np.linalg.norm(bc) * np.linalg.norm(Abc)
        assert abs(bAb - h11_gmres * bb.real) <= TOL * scale
        # and against the definition, summed by numpy on the host
        assert abs(bb - np.vdot(bc, bc)) <= TOL * abs(np.vdot(bc, bc))
        assert abs(bAb - np.vdot(bc, Abc)) <= TOL * scale

        # --- two more calls in a row: several right-hand sides after a single one, then the first call again -------
        nrhs = 3
        psi = wdinputs.spinor(dims, 4103, nrhs)
        da, dbb = op.dev_spinor(nrhs), op.dev_spinor(nrhs)
        wd.wd_pack_spinor(op.h, da, psi, nrhs)
        wd.wd_apply(op.h, dbb, da, nrhs)
        res3 = torch.full((2 * nrhs,), float("nan"), dtype=torch.float64, device="cuda")
        again = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
        wd.wd_inner_product_static(da, dbb, V, Vs, nrhs, res3, stream)
        wd.wd_inner_product_static(db, db, V, Vs, 1, again, stream)
        torch.cuda.synchronize()
        outm = np.empty_like(psi)
        wd.wd_unpack_spinor(op.h, outm, dbb, nrhs)
        got = res3.cpu().numpy().view(np.complex128)
        for k in range(nrhs):
            a_k, b_k = c(psi[k]).ravel(), c(outm[k]).ravel()
            assert abs(got[k] - np.vdot(a_k, b_k)) <= TOL * np.linalg.norm(a_k) * np.linalg.norm(b_k)
            # one right-hand side at a time gives the same number: the partial sums of different right-hand sides do not mix
            one = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
            off = k * 12 * Vs * 2
            wd.wd_inner_product_static(da[off:], dbb[off:], V, Vs, 1, one, stream)
            torch.cuda.synchronize()
            assert abs(complex(*one.cpu().numpy()) - got[k]) <= TOL * np.linalg.norm(a_k) * np.linalg.norm(b_k)
        assert np.array_equal(again.cpu().numpy(), r[0:2])  # same input, same grid, fixed summation order: same bits
