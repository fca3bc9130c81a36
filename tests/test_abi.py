"""Host-side checks of the boundary (no compute calls without a GPU): libbt.so loads, exports every symbol
include/bt.h declares, the binding's struct layout matches the header, and -- on a box without a CUDA device --
the product path fails loudly instead of falling back to anything."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2208_02382_b200 as bt

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = open(os.path.join(ROOT, "include", "bt.h")).read()


def declared_functions():
    body = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    return sorted(set(re.findall(r"\b(bt_[a-z0-9_]+)\s*\(", body)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for required in ("bt_beam_create", "bt_lattice_set", "bt_track", "bt_deposit_cic", "bt_gather_kick"):
        assert required in names


def test_library_exports_every_declared_symbol():
    L = ctypes.CDLL(bt.LIB_PATH)
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), "libbt.so does not export %s" % n
    assert sorted(bt.EXPORTS) == names, "binding and header disagree"


def test_element_struct_layout_matches_header():
    assert bt.ELEMENT_DTYPE.itemsize == 64
    assert bt.ELEMENT_DTYPE.fields["type"][1] == 0 and bt.ELEMENT_DTYPE.fields["nslice"][1] == 4
    assert bt.ELEMENT_DTYPE.fields["ds"][1] == 8 and bt.ELEMENT_DTYPE.fields["p"][1] == 16
    arr = bt.pack_lattice([("quad", 1.0, 25, -1.0), ("dipedge", 0.0, 1, 0.05, 10.0, 0.02, 0.5)])
    assert arr[0]["type"] == 1 and arr[0]["nslice"] == 25 and arr[0]["p"][0] == -1.0
    assert arr[1]["type"] == 3 and list(arr[1]["p"][:4]) == [0.05, 10.0, 0.02, 0.5]
    for name, val in (("BT_DRIFT", 0), ("BT_QUAD", 1), ("BT_SBEND", 2), ("BT_DIPEDGE", 3), ("BT_MULTIPOLE", 4), ("BT_SHORTRF", 5)):
        assert re.search(r"%s\s*=\s*%d" % (name, val), HEADER) and getattr(bt, name) == val


def test_version_and_error_string():
    assert bt.version() == int(re.search(r"#define BT_VERSION (\d+)", HEADER).group(1))
    assert bt.lib.bt_beam_set_ref(None, 1.0, 1.0, 1.0) == bt.BT_ERR_INVALID
    assert b"NULL" in bt.lib.bt_last_error()
    out = ctypes.c_void_p()
    assert bt.lib.bt_beam_create(ctypes.byref(out), 0, None, None) == bt.BT_ERR_INVALID      # n <= 0, before any CUDA call
    assert bt.lib.bt_grid_create(ctypes.byref(out), 1, 4, 4, (ctypes.c_double * 3)(), (ctypes.c_double * 3)(1, 1, 1)) == bt.BT_ERR_INVALID


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(bt.BtError) as ei:
        bt.Beam(16, storage="library", stream=0)
    assert ei.value.code == bt.BT_ERR_CUDA
    with pytest.raises(bt.BtError):
        bt.Grid((4, 4, 4), (0, 0, 0), (1, 1, 1))
    with pytest.raises(bt.BtError):
        bt.calib_fp64(1.0, stream=0)


def test_product_does_not_import_the_oracle():
    """Neither side imports, includes or loads the other."""
    pkg = os.path.join(ROOT, "paper_2208_02382_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert not re.search(r"#include\s*[<\"][^>\"]*oracle", src), f
                assert "libbt_oracle" not in src and "bt_oracle" not in src, f
    for f in ("__init__.py", "build.py", "bt_oracle.c"):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert not re.search(r"^\s*(from|import)\s+paper_2208_02382_b200", src, flags=re.M), f
        assert not re.search(r"#include\s*[<\"][^>\"]*(bt\.h|bt_internal|csrc)", src), f
        assert "libbt.so" not in src, f
