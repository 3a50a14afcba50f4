"""The C-ABI library builds, loads and exports every symbol include/mg.h declares (no GPU needed),
and the product package never reaches into oracle/ (and vice versa)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "mg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+)?(?:int|void|long long|char\s*\*|const char\s*\*)\s*\*?\s*(\w+)\s*\(", text, flags=re.M)
    return sorted(set(names))


def test_library_exports_every_declared_symbol():
    from paper_2401_06755_b200 import _build, binding
    lib = ctypes.CDLL(_build.build())
    declared = _declared_functions()
    assert {"mg_create", "mg_apply_operator", "mg_smooth", "mg_vcycle", "mg_solve", "vof_residual"} <= set(declared)
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared
    for name in declared:
        assert hasattr(binding, name), "binding lacks %s" % name


def test_compute_calls_fail_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        return
    import pytest
    from paper_2401_06755_b200 import _build
    lib = ctypes.CDLL(_build.build())
    lib.mg_last_error.restype = ctypes.c_char_p

    class G(ctypes.Structure):
        _fields_ = [("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
                    ("hx", ctypes.c_double), ("hy", ctypes.c_double), ("hz", ctypes.c_double)]
    h = ctypes.c_void_p()
    bc = (ctypes.c_int * 6)(1, 1, 1, 1, 1, 1)
    rc = lib.mg_create(ctypes.byref(h), ctypes.byref(G(8, 8, 8, .1, .1, .1)), 2, bc, 0, None)
    assert rc == -3 and not h.value and lib.mg_last_error()          # MG_ECUDA, no CPU fallback
    assert lib.mg_create(ctypes.byref(h), ctypes.byref(G(9, 8, 8, .1, .1, .1)), 2, bc, 0, None) == -2   # MG_ESHAPE
    assert lib.mg_create(ctypes.byref(h), ctypes.byref(G(2048, 1024, 1024, .1, .1, .1)), 2, bc, 0, None) == -2   # > 2^31 - 1 points
    assert b"2^31" in lib.mg_last_error()
    with pytest.raises(Exception):
        import paper_2401_06755_b200 as m
        m.mg_create((8, 8, 8, 0.1), 2, (1,) * 6)


def test_oracle_and_product_share_no_code():
    pkg = os.path.join(ROOT, "paper_2401_06755_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert not re.search(r"#include\s+[\"<][^\">]*oracle", text), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2401_06755_b200", text, flags=re.M), f
            assert not re.search(r"#include\s+[\"<][^\">]*(csrc|mg\.h)", text), f
