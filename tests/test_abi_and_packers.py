"""CPU-only checks of the boundary: libwd.so loads, exports every symbol include/wd.h declares, the
Python binding mirrors the header, argument errors are reported without a GPU, and the host
packer (step a0) is the permutation DESIGN.md "Data layout in HBM" states.  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2407_00041_b200 as wd
import wdinputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(header="wd.h", prefix="wd_"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(" + prefix + r"[a-z_0-9]+)\s*\(", text)))


def test_every_header_under_include_is_covered():
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["wd.h", "wd_bench.h"]


def test_bench_library_exports_every_declared_symbol_and_is_not_the_product():
    from paper_2407_00041_b200 import benchlib

    names = declared_functions("wd_bench.h", "wdb_")
    assert names == sorted(benchlib.SIGNATURES) and len(names) >= 2
    B = ctypes.CDLL(benchlib.LIB_PATH)
    L = ctypes.CDLL(wd.LIB_PATH)
    for n in names:
        assert hasattr(B, n), f"libwdbench.so does not export {n}"
        assert not hasattr(L, n), f"libwd.so must not export the bench helper {n}"


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert len(names) >= 20 and "wd_apply" in names and "wd_create" in names
    L = ctypes.CDLL(wd.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"libwd.so does not export {n}"


def test_binding_mirrors_header():
    assert sorted(wd.SIGNATURES) == declared_functions()
    for n in wd.SIGNATURES:
        assert callable(getattr(wd, n)), n


def test_version_and_kernel_registry():
    assert "sm_100a" in wd.wd_version()
    n = wd.wd_kernel_count()
    assert n >= 2
    names = [wd.wd_kernel_name(k) for k in range(n)]
    assert names[0].startswith("linear") and len(set(names)) == n
    assert wd.wd_kernel_name(n) is None and wd.wd_kernel_name(-1) is None


def test_argument_errors_need_no_gpu():
    h = ctypes.c_void_p()
    L = wd.lib()
    assert L.wd_create(None, 4, 4, 4, 4, -0.5, 0.0) == wd.WD_EINVAL
    assert L.wd_create(ctypes.byref(h), 4, 0, 4, 4, -0.5, 0.0) == wd.WD_EINVAL
    assert "extent" in wd.wd_last_error(None)
    assert L.wd_apply(None, None, None, 1) == wd.WD_EINVAL
    assert L.wd_spinor_bytes(None, 1) == 0
    assert L.wd_layout_bytes(7, 10) == 0
    with pytest.raises(wd.WDError):
        wd.wd_create(4, 4, -1, 4, 0.0, 0.0)


@pytest.mark.parametrize("V", [1, 63, 64, 65, 1000])
def test_host_packer_is_the_stated_permutation(V):
    rng = np.random.default_rng(V)
    # spinor: [V][12] -> [12][V]; gauge: [V][36] -> [36][V]
    for field, nc in ((wd.WD_FIELD_SPINOR, 12), (wd.WD_FIELD_GAUGE, 36)):
        a = rng.normal(size=(V, nc, 2))
        packed = np.empty((nc, V, 2))
        assert wd.wd_layout_bytes(field, V) == packed.nbytes
        wd.wd_layout_pack_host(field, V, a, packed)
        assert np.array_equal(packed, a.transpose(1, 0, 2))
        back = np.empty_like(a)
        wd.wd_layout_unpack_host(field, V, packed, back)
        assert np.array_equal(back, a)
    # one unit of the blocked multi-RHS layout (WD_OPT_RHS_BLOCK = 4): [4][V][12] -> [12][V][4]
    a = rng.normal(size=(4, V, 12, 2))
    packed = np.empty((12, V, 4, 2))
    assert wd.wd_layout_bytes(wd.WD_FIELD_SPINOR_BLOCK4, V) == packed.nbytes == 4 * V * 192
    wd.wd_layout_pack_host(wd.WD_FIELD_SPINOR_BLOCK4, V, a, packed)
    assert np.array_equal(packed, a.transpose(2, 1, 0, 3))
    back = np.empty_like(a)
    wd.wd_layout_unpack_host(wd.WD_FIELD_SPINOR_BLOCK4, V, packed, back)
    assert np.array_equal(back, a)
    # self-coupling: 42 canonical -> 36 slots, 18 per chirality block (3 real-diagonal pairs, then
    # the block's 15 strict-upper entries), block A first
    C = wdinputs.selfcoupling_random((1, 1, 1, V), 77)
    packed = np.empty((36, V, 2))
    assert wd.wd_layout_bytes(wd.WD_FIELD_CLOVER, V) == packed.nbytes == V * 576
    wd.wd_layout_pack_host(wd.WD_FIELD_CLOVER, V, C, packed)
    for b in range(2):
        for j in range(3):
            q = 3 * b + j
            assert np.array_equal(packed[18 * b + j, :, 0], C[:, 2 * q, 0])
            assert np.array_equal(packed[18 * b + j, :, 1], C[:, 2 * q + 1, 0])
        assert np.array_equal(packed[18 * b + 3:18 * b + 18], C[:, 12 + 15 * b:27 + 15 * b].transpose(1, 0, 2))
    back = np.empty_like(C)
    wd.wd_layout_unpack_host(wd.WD_FIELD_CLOVER, V, packed, back)
    assert np.array_equal(back, C)


def test_no_cpu_fallback_in_product_path():
    """The package never imports the oracle, and the oracle never imports the package."""
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2407_00041_b200")):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(root, fn)).read()
                assert "wdref" not in txt and "import oracle" not in txt and "from oracle" not in txt, fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "import paper_2407_00041_b200" not in txt and "libwd.so" not in txt and "include/wd.h" not in txt, fn
