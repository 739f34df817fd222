"""The C-ABI library loads on a machine without a GPU, exports every symbol include/ljmd.h
declares, and validates arguments before touching the device."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def b():
    from paper_0709_3225_b200 import build
    build.build()
    from paper_0709_3225_b200 import binding
    return binding


def declared_functions():
    src = open(os.path.join(ROOT, "include", "ljmd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+)?(?:int|int64_t|char\s*\*|void)\s*\*?\s*(\w+)\s*\(", src, flags=re.M)
    return sorted(set(n for n in names if not n.startswith("md_alloc_fn") and not n.startswith("md_free_fn")))


def test_header_declares_the_six_named_calls():
    names = declared_functions()
    for must in ("md_create", "md_set_state", "md_step", "md_get_forces", "md_get_energies", "rand48_fill"):
        assert must in names


def test_library_exports_every_declared_symbol(b):
    lib = ctypes.CDLL(b.LIB_PATH)
    names = declared_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), "libljmd_b200.so does not export %s" % n
    assert set(b._SIGS) == set(names)


def test_strerror(b):
    assert b.md_strerror(0) == "MD_OK"
    for code in range(-6, 0):
        assert b.md_strerror(code).startswith("MD_E")
    assert "unknown" in b.md_strerror(-99)


@pytest.mark.parametrize("args", [
    (0, 10.0, 2.5, 1.0, 1.0, 0.005, 1), (-5, 10.0, 2.5, 1.0, 1.0, 0.005, 1),
    (100, 0.0, 2.5, 1.0, 1.0, 0.005, 1), (100, 10.0, -1.0, 1.0, 1.0, 0.005, 1),
    (100, 10.0, 2.5, -1.0, 1.0, 0.005, 1), (100, 10.0, 2.5, 1.0, 0.0, 0.005, 1),
    (100, 10.0, 2.5, 1.0, 1.0, 0.0, 1), (100, 10.0, 2.5, 1.0, 1.0, 0.005, 3),
    (100, 10.0, 2.5, 1.0, 1.0, 0.005, -1),
    (100, 4.9, 2.5, 1.0, 1.0, 0.005, 1),            # rc > L/2: minimum image invalid
    (100, float("nan"), 2.5, 1.0, 1.0, 0.005, 1),
])
def test_md_create_rejects_bad_arguments_without_a_device(b, args):
    with pytest.raises(b.MDError) as e:
        b.md_create(*args)
    assert e.value.code == b.MD_EINVAL


def test_null_handles_and_pointers(b):
    lib = ctypes.CDLL(b.LIB_PATH)
    assert b._lib.md_create(None, 10, 10.0, 2.5, 1.0, 1.0, 0.005, 1) == b.MD_EINVAL
    assert b._lib.md_destroy(None) == b.MD_OK
    for fn, args in [("md_set_state", (None, None, None)), ("md_get_state", (None, None, None)),
                     ("md_compute_forces", (None, 0)), ("md_step", (None, 1, 0)),
                     ("md_get_forces", (None, None)), ("md_get_energies", (None, None, None, None))]:
        assert getattr(b._lib, fn)(*args) == b.MD_EINVAL, fn


def test_rand48_argument_validation(b):
    seeds = np.array([1, 2], dtype=np.uint64)
    out = np.zeros(8, dtype=np.uint32)
    assert b._lib.rand48_fill(seeds.ctypes.data, 2, 4, 7, out.ctypes.data) == b.MD_EINVAL     # kind
    assert b._lib.rand48_fill(seeds.ctypes.data, -1, 4, 0, out.ctypes.data) == b.MD_EINVAL
    assert b._lib.rand48_fill(seeds.ctypes.data, 2, -4, 0, out.ctypes.data) == b.MD_EINVAL
    assert b._lib.rand48_fill(None, 2, 4, 0, out.ctypes.data) == b.MD_EINVAL
    assert b._lib.rand48_fill(seeds.ctypes.data, 2, 4, 0, None) == b.MD_EINVAL
    assert b._lib.rand48_fill(seeds.ctypes.data, 0, 4, 0, out.ctypes.data) == b.MD_OK         # nothing to do
    bad = np.array([1 << 48], dtype=np.uint64)
    assert b._lib.rand48_fill(bad.ctypes.data, 1, 4, 0, out.ctypes.data) == b.MD_EINVAL       # seed > 48 bits


def test_no_cpu_fallback_without_device(b):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(b.MDError) as e:
        b.md_create(100, 10.0, 2.5, 1.0, 1.0, 0.005, 1)
    assert e.value.code == b.MD_ECUDA
    seeds = np.array([1], dtype=np.uint64)
    out = np.zeros(4, dtype=np.uint32)
    assert b._lib.rand48_fill(seeds.ctypes.data, 1, 4, 0, out.ctypes.data) == b.MD_ECUDA


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_0709_3225_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), f
                assert "ljmd_oracle" not in txt, f
