"""Host-side checks of the C ABI (no GPU needed): libocn.so builds, loads, exports every symbol include/ocn.h
declares, validates arguments before touching the device, and fails loudly (no CPU fallback) without one."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def Bd():
    from paper_2502_14148_b200 import build
    build.build()
    from paper_2502_14148_b200 import binding
    binding.lib()
    return binding


def _declared():
    src = open(os.path.join(ROOT, "include", "ocn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ocn_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(Bd):
    names = _declared()
    assert {"ocn_grid_create", "ocn_fill_halos", "ocn_compute_tendencies", "ocn_rk3_substage"} <= set(names)
    L = C.CDLL(Bd.LIBPATH)
    for n in names:
        assert hasattr(L, n), "libocn.so does not export %s" % n
    assert sorted(Bd.EXPORTS) == names, "binding.EXPORTS and include/ocn.h disagree"


def test_struct_layouts_match_header(Bd):
    # ocn_params: 8 ints, 7 doubles, 2 pointers, 1 + 8 doubles, 1 int (+ 4 bytes tail padding); ocn_fields: 3 + 8 pointers
    assert C.sizeof(Bd.ocn_fields) == 11 * 8
    assert C.sizeof(Bd.ocn_params) == 8 * 4 + 7 * 8 + 2 * 8 + 9 * 8 + 8
    assert C.sizeof(Bd.ocn_layout) == 7 * 8 + 4 * 4
    assert Bd.ocn_version() == "0.1" or re.match(r"\d+\.\d+", Bd.ocn_version())


def test_argument_errors_are_detected_before_the_device_is_touched(Bd):
    L = Bd.lib()
    h = C.c_void_p()
    topo = (C.c_int * 3)(0, 0, 1)
    bad = [
        dict(Nx=0, Ny=4, Nz=4, halo=3, dx=1.0, dy=1.0, dz=1.0, topo=(0, 0, 1)),      # N < 1
        dict(Nx=8, Ny=8, Nz=8, halo=0, dx=1.0, dy=1.0, dz=1.0, topo=(0, 0, 1)),      # halo < 1
        dict(Nx=8, Ny=8, Nz=8, halo=3, dx=0.0, dy=1.0, dz=1.0, topo=(0, 0, 1)),      # spacing <= 0
        dict(Nx=8, Ny=8, Nz=8, halo=3, dx=1.0, dy=1.0, dz=-1.0, topo=(0, 0, 1)),
        dict(Nx=2, Ny=8, Nz=8, halo=3, dx=1.0, dy=1.0, dz=1.0, topo=(0, 0, 1)),      # N < halo
        dict(Nx=8, Ny=8, Nz=4, halo=3, dx=1.0, dy=1.0, dz=1.0, topo=(0, 0, 2)),      # Flat axis with N != 1
        dict(Nx=8, Ny=8, Nz=8, halo=3, dx=1.0, dy=1.0, dz=1.0, topo=(0, 7, 1)),      # unknown topology
    ]
    for b in bad:
        t = (C.c_int * 3)(*b["topo"])
        rc = L.ocn_grid_create(C.byref(h), b["Nx"], b["Ny"], b["Nz"], b["halo"], b["dx"], b["dy"], None, b["dz"], t, 0)
        assert rc == Bd.OCN_ERR_INVALID, b
        assert L.ocn_last_error() and len(L.ocn_last_error()) > 0
        assert not h.value
    assert L.ocn_grid_create(None, 8, 8, 8, 3, 1.0, 1.0, None, 1.0, topo, 0) == Bd.OCN_ERR_INVALID
    assert L.ocn_grid_create(C.byref(h), 8, 8, 8, 3, 1.0, 1.0, None, 1.0, topo, 5) == Bd.OCN_ERR_INVALID
    # NULL handles on the compute calls
    assert L.ocn_fill_halos(None, None, None, None) == Bd.OCN_ERR_INVALID
    assert L.ocn_compute_w(None, None, None) == Bd.OCN_ERR_INVALID
    assert L.ocn_compute_tendencies(None, None, None, None, None, None) == Bd.OCN_ERR_INVALID
    assert L.ocn_rk3_substage(None, None, 1, 0.1, None, None, None, None) == Bd.OCN_ERR_INVALID
    assert L.ocn_rk3_substage(None, None, 4, 0.1, None, None, None, None) == Bd.OCN_ERR_INVALID
    assert L.ocn_grid_destroy(None) == Bd.OCN_OK


def test_no_cpu_fallback_without_a_device(Bd):
    """on a box without a GPU a valid grid_create must FAIL with OCN_ERR_CUDA (it never computes on the host)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(Bd.OcnError) as e:
        Bd.ocn_grid_create(8, 8, 8, 3, 1.0, 1.0, None, 1.0, (0, 0, 1), "f64")
    assert e.value.code == Bd.OCN_ERR_CUDA


def test_product_does_not_import_the_oracle():
    pk = os.path.join(ROOT, "paper_2502_14148_b200")
    for root, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(root, f)).read()
                assert "ocnref" not in s and "from oracle" not in s and "import oracle" not in s, f
    s = open(os.path.join(ROOT, "oracle", "ocnref.py")).read() + open(os.path.join(ROOT, "oracle", "ocnref.cpp")).read()
    assert "paper_2502_14148_b200 import" not in s and "libocn.so" not in s and "ocn.h" not in s.replace("include/ocn.h", "")
