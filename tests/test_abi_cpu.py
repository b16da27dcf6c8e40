"""CPU-side checks of the boundary: the library builds, loads and exports every symbol md.h declares;
argument errors are reported before any device work (-m "not gpu")."""
import ctypes as C
import os
import re

import paper_1610_03343_b200 as md

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "md.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = md.load()
    names = declared_symbols()
    assert "md_build_neighbors" in names and "md_tersoff_force" in names
    assert "md_sw_force" in names and "md_velocity_verlet_step" in names
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(md.EXPORTS) == names
    assert "sm_100a" in md.md_version()


def test_binding_has_the_same_names_as_the_header():
    for name in declared_symbols():
        assert callable(getattr(md, name)), name


def test_argument_errors_are_synchronous_and_need_no_device():
    lib = md.load()
    h = C.c_void_p(0)
    assert lib.md_neighbors_create(C.byref(h), C.c_int64(10), C.c_int(0)) == md.MD_ERR_ARG
    assert lib.md_neighbors_create(C.byref(h), C.c_int64(-1), C.c_int(8)) == md.MD_ERR_ARG
    assert lib.md_neighbors_create(None, C.c_int64(1), C.c_int(8)) == md.MD_ERR_ARG
    assert lib.md_neighbors_create(C.byref(h), C.c_int64(10 ** 9), C.c_int(64)) == md.MD_ERR_ARG
    assert lib.md_neighbors_destroy(None) == md.MD_ERR_ARG
    box = (C.c_double * 3)(10.0, 10.0, 10.0)
    assert lib.md_velocity_verlet_step(C.c_int(2), C.c_int64(0), None, None, None, None, None, None, None,
                                       C.c_double(1.0), C.c_double(1.0), box, None) == md.MD_ERR_ARG
    assert lib.md_velocity_verlet_step(C.c_int(0), C.c_int64(4), None, None, None, None, None, None, None,
                                       C.c_double(1.0), C.c_double(1.0), box, None) == md.MD_ERR_ARG
    assert lib.md_build_neighbors(None, C.c_int64(0), None, None, None, box, C.c_double(3.0), None) == md.MD_ERR_ARG
    assert lib.md_probe_fp64_peak(C.c_int(0), None, None) == md.MD_ERR_ARG


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1610_03343_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in text and "from oracle" not in text, fn
                assert "md_oracle" not in text, fn
