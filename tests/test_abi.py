"""Host-side checks of the C-ABI library (no GPU, no compute calls): it builds, loads, exports every symbol
include/te_jk.h declares, and rejects bad arguments before touching the device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    import paper_2406_14920_b200 as te
    return te.lib()


def declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "te_jk.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(te_[a-z0-9_]+)\s*\(", hdr)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("te_basis_create", "te_shellpair_build", "te_build_jk", "te_eri_block"):
        assert name in syms


def test_library_exports_every_declared_symbol(L):
    for name in declared_symbols():
        assert hasattr(L, name), name


def test_unsupported_l_and_bad_arguments_fail_loudly(L):
    xyz = np.zeros((1, 3))
    sa = np.zeros(1, dtype=np.int32)
    npr = np.ones(1, dtype=np.int32)
    ex = np.ones(1)
    co = np.ones(1)
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
    h = C.c_void_p()

    def create(l, expo=ex, natoms=1):
        sl = np.array([l], dtype=np.int32)
        return L.te_basis_create(natoms, xyz.ctypes.data_as(dp), 1, sa.ctypes.data_as(ip), sl.ctypes.data_as(ip),
                                 npr.ctypes.data_as(ip), expo.ctypes.data_as(dp), co.ctypes.data_as(dp), C.byref(h))
    assert create(4) == -2                      # TE_ERR_UNSUPPORTED_L
    assert b"l = 4" in L.te_last_error()
    assert create(-1) == -1                     # TE_ERR_BAD_ARG
    assert create(0, expo=np.array([-1.0])) == -1
    assert create(0, natoms=0) == -1
    assert h.value is None
    assert L.te_shellpair_build(None, 1e-12, C.byref(h)) == -1
    assert L.te_build_jk(None, None, None, None, 0.0, None) == -1
    assert L.te_eri_block(None, 1, None, None, None) == -1
    assert L.te_boys(1, None, 13, None) == -1
    assert L.te_pairs_info(None, None, None) == -1


def test_python_binding_mirrors_c_names():
    import paper_2406_14920_b200 as te
    for name in ("te_basis_create", "te_shellpair_build", "te_build_jk", "te_eri_block", "te_boys"):
        assert callable(getattr(te, name))


def test_product_does_not_import_oracle():
    """The product path shares nothing with the oracle (and has no CPU fallback)."""
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2406_14920_b200")):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "te_oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "te_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2406_14920_b200" not in txt.replace("(paper_2406_14920_b200/csrc)", "").replace(
        "(paper_2406_14920_b200)", "")
