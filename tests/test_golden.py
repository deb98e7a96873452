"""The oracle reproduces the stored fixture (written by tests/golden/make_golden.py from oracle/ only)."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def load_golden():
    rows = []
    with open(os.path.join(HERE, "golden", "wilson_clover_2x4x2x4.txt")) as fh:
        for line in fh:
            if line.startswith("#"):
                continue
            kind, s, k, re, im = line.split()
            rows.append((kind, int(s), int(k), float(re), float(im)))
    return rows


def golden_module():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def check_against_golden(out_c, out_w, psi, tol=1e-12):
    for kind, s, k, re, im in load_golden():
        if kind.startswith("norm2"):
            continue
        arr = out_c if kind == "clover" else out_w
        assert abs(arr[s, k, 0] - re) <= tol * max(1.0, abs(re)), (kind, s, k)
        assert abs(arr[s, k, 1] - im) <= tol * max(1.0, abs(im)), (kind, s, k)


def test_oracle_reproduces_golden():
    mod = golden_module()
    U, psi, C, out_c, out_w = mod.compute()
    check_against_golden(out_c, out_w, psi)
    rows = [r for r in load_golden() if r[0].startswith("norm2")]
    vals = [float((out_c ** 2).sum()), float((out_w ** 2).sum()), float((psi ** 2).sum())]
    for r, v in zip(rows, vals):
        assert abs(r[3] - v) <= 1e-12 * v
