"""CPU-side checks of the C-ABI boundary: libpcamm.so builds for sm_100a, loads without a GPU and
exports every symbol include/pcamm.h declares; the host-only entry points behave; the product
fails loudly (never falls back) when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1004_0014_b200 as pc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "pcamm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pcamm_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = pc.lib()
    names = _declared()
    assert sorted(pc.SYMBOLS) == names
    for n in names:
        assert getattr(lib, n) is not None


def test_default_opts_and_struct_layout():
    o = pc.pcamm_opts()
    pc.lib().pcamm_default_opts(C.byref(o))
    d = pc.Opts()
    for f, _ in pc.pcamm_opts._fields_:
        assert getattr(o, f) == pytest.approx(getattr(d, f)), f
    assert C.sizeof(pc.pcamm_geometry) == 24 * 4
    assert C.sizeof(pc.pcamm_opts) == 10 * 4
    assert C.sizeof(pc.pcamm_info) == 8 + 4 * 8 + 4 * 8


def test_invalid_arguments_are_reported_without_a_gpu():
    lib = pc.lib()
    h = C.c_void_p()
    assert lib.pcamm_model_create(None, None, None, None, 0, None, None, C.byref(h)) == pc.E_INVALID
    assert "NULL" in pc.last_error()
    assert lib.pcamm_warp(None, None, None, None) == pc.E_INVALID
    assert lib.pcamm_reconstruct(None, None, C.c_float(0), None, None, None, None, None, None, None) == pc.E_INVALID
    assert pc.launch_count() >= 0
    x = (C.c_float * 4)()
    assert lib.pcamm_pca_fit(C.c_int64(4), 3, 2, None, -1, x, x, None, None, None, None) == pc.E_INVALID
    assert lib.pcamm_pca_fit(C.c_int64(4), 1, 1, x, -1, x, x, None, None, None, None) == pc.E_INVALID    # N < 2
    assert lib.pcamm_pca_fit(C.c_int64(4), 3, 3, x, -1, x, x, None, None, None, None) == pc.E_INVALID    # K > N - 1
    assert "K outside" in pc.last_error()


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU box")
    z = torch.zeros(8)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pc.Model(nx=2, ny=2, nz=2, hx=1, hy=1, hz=1, K=1, nu=2, nv=2, pu=1, pv=1, f0=z, mean_dvf=z, eig_dvf=z)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1004_0014_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
