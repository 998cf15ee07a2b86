"""C-ABI surface checks that need no GPU: the library builds, loads, exports every symbol
include/orb.h declares, and its argument checks answer with the documented codes."""
import ctypes as C
import os
import re

import pytest

from paper_1908_02219_b200 import binding as B
from paper_1908_02219_b200 import build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build_mod.build()
    return B.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "orb.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(orb_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(L):
    names = declared_symbols()
    assert set(names) == set(B.SYMBOLS), (names, B.SYMBOLS)
    for n in names:
        assert getattr(L, n) is not None


def test_version_and_strerror(L):
    assert L.orb_version() == 100
    assert L.orb_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert L.orb_strerror(code) not in (b"ok", b"unknown status")
    assert L.orb_strerror(-99) == b"unknown status"


def test_struct_layout_matches_header():
    assert C.sizeof(B.GridDesc) == 64     # 3*i32 (+pad) + 5*f64 + 2*i32
    assert C.sizeof(B.NlPolicy) == 32


def test_argument_checks_without_device(L):
    h = C.c_void_p()
    assert L.orb_grid_create(None, C.byref(h)) == B.ORB_E_INVAL
    bad = B.GridDesc(2, 32, 16, 1.0, 0.3, 1.0, 1 / 180, 1.0, 1, 0)
    assert L.orb_grid_create(C.byref(bad), C.byref(h)) == B.ORB_E_INVAL      # ns < 4
    bad = B.GridDesc(16, 32, 16, 1.0, 1.3, 1.0, 1 / 180, 1.0, 1, 0)
    assert L.orb_grid_create(C.byref(bad), C.byref(h)) == B.ORB_E_INVAL      # a >= r0
    assert L.orb_grid_destroy(None) == B.ORB_OK
    assert L.orb_markers_bind(None, 0, None, None, None, None, None, None, 0) == B.ORB_E_INVAL
    assert L.orb_deposit(None, None, None, None, None) == B.ORB_E_INVAL


def test_no_cpu_fallback(L):
    """Without a CUDA device the library refuses to create a grid (ORB_E_CUDA): no CPU path."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = C.c_void_p()
    ok = B.GridDesc(16, 32, 16, 1.0, 0.3, 1.0, 1 / 180, 1.0, 1, 0)
    assert L.orb_grid_create(C.byref(ok), C.byref(h)) == B.ORB_E_CUDA
    with pytest.raises(B.OrbError):
        B.Grid(16, 32, 16)


def test_product_does_not_import_oracle():
    """The package never imports, links or executes anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1908_02219_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "orb_oracle" not in text and "liborb_oracle" not in text, f


@pytest.mark.parametrize("ns", [4, 5, 7, 16, 128])
def test_radial_spline_table_matches_scipy(L, ns):
    """Host logic of the tile kernel: the polynomial pieces of the clamped cubic B-splines
    (orb_spline_table_radial) evaluated by Horner equal scipy's BSpline design matrix on the same
    open knot vector, in every cell including the four end cells; and they sum to one."""
    import numpy as np
    from scipy import interpolate
    tab = B.spline_table_radial(ns)
    assert tab.shape == (ns, 4, 4)
    T = np.array([0.0] * 3 + list(range(ns + 1)) + [float(ns)] * 3)
    rng = np.random.default_rng(ns)
    for c in list(range(min(ns, 4))) + list(range(max(ns - 4, 0), ns)) + [ns // 2]:
        for t in list(rng.uniform(0, 1, 8)) + [0.0, 0.5, 1.0 - 1e-12]:
            x = c + t
            t = x - c   # the in-cell coordinate scipy actually sees
            row = interpolate.BSpline.design_matrix(np.array([min(x, ns)]), T, 3).toarray()[0]
            got = np.zeros(ns + 3)
            for a in range(4):
                k = tab[c, a]
                got[c + a] = ((k[3] * t + k[2]) * t + k[1]) * t + k[0]
            np.testing.assert_allclose(got, row, rtol=0, atol=5e-15)
            assert abs(got.sum() - 1.0) < 5e-15
    # interior cells hold the cardinal pieces exactly
    if ns >= 8:
        want = np.array([[1 / 6, -0.5, 0.5, -1 / 6], [2 / 3, 0, -1, 0.5], [1 / 6, 0.5, 0.5, -0.5],
                         [0, 0, 0, 1 / 6]])
        np.testing.assert_allclose(tab[ns // 2], want, rtol=0, atol=1e-15)
