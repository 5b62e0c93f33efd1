"""CPU-side checks of the C-ABI boundary: libdvx.so builds, loads and exports every function include/dvx.h declares;
the Python binding declares the same names; the product path refuses to run without a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "dvx.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = set(re.findall(r"\b(dvx_[a-z_0-9]+)\s*\(", text))
    return sorted(n for n in names if not n.endswith("_fn"))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2606_23031_b200 import build
    return build.build()


def test_header_declares_the_hot_path_calls():
    names = _declared()
    for must in ("dvx_create", "dvx_octree_create", "dvx_render", "dvx_backward", "dvx_render_host", "dvx_backward_host",
                 "dvx_debug_tile_list", "dvx_sort_pairs"):
        assert must in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared():
        assert hasattr(lib, name), "libdvx.so does not export %s" % name


def test_binding_lists_the_same_names(lib_path):
    import paper_2606_23031_b200 as dvx
    assert sorted(dvx.EXPORTS) == _declared()
    dvx.load()


def test_no_cpu_fallback(lib_path):
    import torch
    import paper_2606_23031_b200 as dvx
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError):
        dvx.Context(0)
    # and the C entry point itself refuses without a device
    lib = dvx.load()
    h = ctypes.c_void_p()
    rc = lib.dvx_create(0, None, dvx.binding.ALLOC_FN(0), dvx.binding.FREE_FN(0), None, ctypes.byref(h))
    assert rc == -4 and not h.value


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_23031_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("dvx_oracle", "oracle") or f == "__never__", "%s mentions the oracle" % f
