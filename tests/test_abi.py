"""The C-ABI library loads and exports every symbol include/bh.h declares (no GPU, no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import load_library
    return load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "bh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bh_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_1106_1900_b200 import SYMBOLS
    names = _declared()
    assert names == sorted(SYMBOLS)
    for n in names:
        assert hasattr(lib, n), n


def test_host_only_entry_points(lib):
    from paper_1106_1900_b200 import workspace_bytes
    b1, b2 = workspace_bytes(1 << 14), workspace_bytes(1 << 20)
    assert 0 < b1 < b2 and b2 < 3 * 2 ** 30        # ~2.1 KB per particle at the default capacities (1.3 KB of it the interaction lists)
    assert workspace_bytes(0) == 0 and workspace_bytes(1 << 20, nleaf=65) == 0 and workspace_bytes(1 << 20, ncrit=65) == 0
    # a tighter cell capacity shrinks the workspace
    assert workspace_bytes(1 << 20, max_cells=1 << 19) < b2
    assert lib.bh_status_string(0) == b"ok" and b"workspace" in lib.bh_status_string(-2)
    # null handles are rejected, not dereferenced
    assert lib.bh_tree_build(None, None) == -1 and lib.bh_destroy(None) == -1
    h = ctypes.c_void_p()
    assert lib.bh_create(ctypes.byref(h), 1 << 10, None, None, 0) == -1


def test_product_and_oracle_do_not_import_each_other():
    import glob
    imp_oracle = re.compile(r"^\s*(import\s+oracle|from\s+oracle\b|#include.*oracle)", re.M)
    imp_product = re.compile(r"^\s*(import\s+paper_1106_1900_b200|from\s+paper_1106_1900_b200\b|#include.*(csrc|bh\.h|bh_internal))", re.M)
    for f in glob.glob(os.path.join(ROOT, "paper_1106_1900_b200", "**", "*"), recursive=True):
        if f.endswith((".py", ".cu", ".cuh")):
            assert not imp_oracle.search(open(f).read()), f
    for f in glob.glob(os.path.join(ROOT, "oracle", "*")):
        if f.endswith((".py", ".cpp")):
            assert not imp_product.search(open(f).read()), f
