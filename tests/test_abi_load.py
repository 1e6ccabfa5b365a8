"""CPU checks of the boundary: the C-ABI libraries build, load and export every symbol include/grpic.h
declares; host-side argument validation that needs no device.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    from paper_2511_17701_b200 import build
    return build.build()


def _declared():
    src = open(os.path.join(ROOT, "include", "grpic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(grpic_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    d = _declared()
    for name in ("grpic_create", "grpic_interp_push", "grpic_deposit", "grpic_sort", "grpic_step", "grpic_destroy"):
        assert name in d


@pytest.mark.parametrize("prec,nbytes", [("f32", 4), ("f64", 8)])
def test_library_loads_and_exports_every_declared_symbol(libs, prec, nbytes):
    lib = C.CDLL(libs[prec])
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in grpic.h but not exported by libgrpic_{prec}.so"
    assert lib.grpic_real_bytes() == nbytes
    assert lib.grpic_tile_size() > 0


def test_binding_lists_the_same_symbols(libs):
    from paper_2511_17701_b200 import grpic
    assert sorted(grpic.EXPORTS) == _declared()


def test_create_validates_arguments_and_never_falls_back(libs):
    import torch
    from paper_2511_17701_b200 import grpic
    lib = grpic.load("f64")
    h = C.c_void_p()
    g = grpic._Grid(0, 8, 2, 1)
    assert lib.grpic_create(C.byref(g), 0.9, 1.0, 20.0, C.byref(h)) == grpic.GRPIC_EINVAL
    assert b"n1" in lib.grpic_last_error(None)
    g = grpic._Grid(8, 8, 0, 1)
    assert lib.grpic_create(C.byref(g), 0.9, 1.0, 20.0, C.byref(h)) == grpic.GRPIC_EINVAL
    g = grpic._Grid(8, 8, 2, 2)          # r_map: 1 = A.3 (log r), 0 = A.2 (uniform r); anything else is refused
    assert lib.grpic_create(C.byref(g), 0.9, 1.0, 20.0, C.byref(h)) == grpic.GRPIC_EINVAL
    g = grpic._Grid(8, 8, 2, 1)
    assert lib.grpic_create(C.byref(g), 0.9, 20.0, 1.0, C.byref(h)) == grpic.GRPIC_EINVAL
    assert lib.grpic_create(C.byref(g), 1.5, 1.0, 20.0, C.byref(h)) == grpic.GRPIC_EINVAL
    if not torch.cuda.is_available():
        # no device: the product path fails loudly instead of computing on the CPU
        assert lib.grpic_create(C.byref(g), 0.9, 1.0, 20.0, C.byref(h)) == grpic.GRPIC_ECUDA
        with pytest.raises(grpic.GrpicError):
            grpic.Context(8, 8, 0.9, 1.0, 20.0, precision="f64")


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2511_17701_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "grpic_oracle" not in txt, f
