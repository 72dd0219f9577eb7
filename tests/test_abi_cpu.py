"""Host-side checks that need no GPU: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/fdtd_b200.h declares; host-only entry points behave."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from conftest import ROOT, golden
from paper_2606_06910_b200 import build as fbuild


@pytest.fixture(scope="module")
def lib():
    path = fbuild.build()
    return C.CDLL(path)


def _declared():
    src = open(os.path.join(ROOT, "include", "fdtd_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fdtd_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared()
    assert "fdtd_create" in names and "fdtd_step" in names and "fdtd_get_field" in names
    assert "fdtd_set_model" in names and "fdtd_destroy" in names
    for n in names:
        assert hasattr(lib, n), n
    from paper_2606_06910_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_coefficient_table_bit_exact(lib):
    out = np.zeros(4, np.float32)
    assert lib.fdtd_coeffs(C.c_void_p(out.ctypes.data)) == 0
    assert list(out.view(np.uint32)) == [int(b, 16) for b in golden("coefficients.txt")["bits"]]


def test_workspace_bytes_and_validation():
    from paper_2606_06910_b200 import binding as B
    p = B.make_params((256,) * 3, (16,) * 6, cpml_alpha_max=0.1)
    n = B.fdtd_workspace_bytes(p)
    vol = 288 ** 3 * 4
    psi = 12 * 20 * 288 * 288 * 4                 # 6 variables x 2 faces, <= 20 planes each (16 + staggering + x rounding)
    assert 5 * vol < n < 5 * vol + psi + (1 << 25)      # 4 fields + Kc + slab-local psi + tables / wavelets
    # slab-local psi: far below the paper's six extra full-volume arrays
    assert n < 6 * vol
    bad = B.make_params((0, 8, 8))
    assert B.fdtd_workspace_bytes(bad) == 0 and "n_interior" in B.last_error()
    bad = B.make_params((32,) * 3, (8,) * 6, decomp=(1, 2, 2), ghost=4, substeps=2)          # g < 4 m
    assert B.fdtd_workspace_bytes(bad) == 0 and "ghost" in B.last_error()
    ok = B.make_params((32,) * 3, decomp=(2, 1, 1), ghost=8, substeps=2)                     # an x cut (block-xy)
    assert B.fdtd_workspace_bytes(ok) > 0
    bad = B.make_params((32,) * 3, decomp=(2, 1, 1), ghost=6, substeps=1)                    # ... needs float4-aligned ghosts
    assert B.fdtd_workspace_bytes(bad) == 0 and "multiples of 4" in B.last_error()
    bad = B.make_params((24,) * 3, (8,) * 6, decomp=(2, 1, 1), ghost=8, substeps=2)         # ... and room beside the x layers
    assert B.fdtd_workspace_bytes(bad) == 0
    bad = B.make_params((32,) * 3, dt=0.0)
    assert B.fdtd_workspace_bytes(bad) == 0
    ok = B.make_params((512,) * 3, (20,) * 6, cpml_alpha_max=0.1, decomp=(1, 2, 2), ghost=16, substeps=4)
    assert B.fdtd_workspace_bytes(ok) > 5 * 552 * 292 * 292 * 4 * 4


def test_create_fails_loudly_without_workspace():
    from paper_2606_06910_b200 import binding as B
    p = B.make_params((16,) * 3)
    h = B.lib.fdtd_create(C.byref(p))
    assert not h and "workspace" in B.last_error()
