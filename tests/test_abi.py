"""CPU-side checks of the C-ABI boundary: the library builds, loads without a GPU and exports every symbol that
include/cs.h declares; argument validation that needs no device."""
import ctypes as C
import os
import re

import numpy as np

import paper_2604_08463_b200 as cs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "cs.h")).read()
    return sorted(set(re.findall(r"CS_API[^;(]*?\b(cs_\w+)\s*\(", src)))


def test_header_declares_the_four_north_star_calls():
    names = _declared()
    for must in ("cs_build_sed_tables", "cs_spectral_like_grad", "cs_component_maps", "cs_optimize"):
        assert must in names


def test_library_exports_every_declared_symbol():
    L = cs.lib()
    names = _declared()
    assert len(names) >= 18
    for n in names:
        assert getattr(L, n) is not None
    assert sorted(cs.EXPORTS) == names


def test_error_strings_and_version():
    assert cs.lib().cs_version() >= 1
    for code in (0, -1, -2, -3, -4, -5, -6):
        assert cs.strerror(code) not in ("", "unknown error")
    assert cs.strerror(-99) == "unknown error"


def test_create_rejects_bad_models_without_touching_a_device():
    L = cs.lib()
    h = C.c_void_p()
    f = np.array([40.0, 50.0], dtype=np.float64)
    m = cs.binding.CsModel(2, f.ctypes.data_as(C.POINTER(C.c_double)), 353.0, 23.0, 2.7255, 0, 768)
    assert L.cs_create(C.byref(h), C.byref(m)) == cs.EINVAL and not h.value
    f = np.array([40.0, 50.0, -1.0], dtype=np.float64)
    m = cs.binding.CsModel(3, f.ctypes.data_as(C.POINTER(C.c_double)), 353.0, 23.0, 2.7255, 0, 768)
    assert L.cs_create(C.byref(h), C.byref(m)) == cs.EINVAL
    m = cs.binding.CsModel(3, f.ctypes.data_as(C.POINTER(C.c_double)), 353.0, 23.0, 2.7255, 7, 768)
    assert L.cs_create(C.byref(h), C.byref(m)) == cs.EINVAL
    assert L.cs_create(None, C.byref(m)) == cs.EINVAL
    assert L.cs_destroy(None) == cs.EINVAL
    assert L.cs_check(None, None) == cs.EINVAL


def test_opt_defaults_follow_design_R13():
    o = cs.opt_defaults()
    assert (o.iters, o.ls_max) == (200, 8)
    assert (o.lr, o.beta1, o.beta2, o.eps, o.ls_c1) == (0.02, 0.9, 0.999, 1e-16, 1e-4)
    assert (o.safe_lo, o.safe_hi) == (1e-15, 1e15)
    assert o.ls_noise == 1e-7 and o.topk == 0.0


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2604_08463_b200")
    for dp, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "cs_oracle" not in txt, fn
