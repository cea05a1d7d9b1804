"""The C-ABI library loads (no GPU needed) and exports every symbol include/ff.h declares."""
import ctypes
import os
import re

import paper_1212_2934_b200 as ff

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "ff.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ff_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    L = ff.lib()
    names = _declared()
    assert set(names) == set(ff.SYMBOLS), (names, ff.SYMBOLS)
    for n in names:
        assert hasattr(L, n), n


def test_host_side_argument_checks_without_gpu():
    L = ff.lib()
    assert L.ff_workspace_bytes(0) == 0 and L.ff_workspace_bytes(-5) == 0
    assert L.ff_workspace_bytes(1 << 29) == 0                       # beyond FF_MAX_N
    b1, b2 = L.ff_workspace_bytes(4096), L.ff_workspace_bytes(8192)
    assert 0 < b1 < b2 and b1 % 256 == 0
    h = ctypes.c_void_p()
    assert L.ff_create(ctypes.byref(h), 0, 0.5, None, 0) == ff.FF_ERR_INVALID_ARG
    assert L.ff_create(ctypes.byref(h), 16, -1.0, None, 0) == ff.FF_ERR_INVALID_ARG
    assert L.ff_create(ctypes.byref(h), 16, float("nan"), None, 0) == ff.FF_ERR_INVALID_ARG
    assert L.ff_create(ctypes.byref(h), 16, 0.5, None, 0) == ff.FF_ERR_WORKSPACE
    assert L.ff_create(ctypes.byref(h), 16, 0.5, ctypes.c_void_p(256), 16) == ff.FF_ERR_WORKSPACE
    assert L.ff_create(ctypes.byref(h), 16, 0.5, ctypes.c_void_p(257), 1 << 30) == ff.FF_ERR_WORKSPACE
    assert L.ff_destroy(None) == ff.FF_ERR_INVALID_ARG
    assert L.ff_build_tree(None, None, 1) == ff.FF_ERR_INVALID_ARG
    assert L.ff_error_string(ff.FF_ERR_NO_TREE).decode().startswith("no tree")
    assert "check" in L.ff_error_string(ff.FF_ERR_CHECK).decode()
    assert ctypes.sizeof(ff.ff_step_params) == 96 and ctypes.sizeof(ff.ff_tree_view) == 136


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1212_2934_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ff_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1212_2934_b200 import" not in src and "import paper_1212_2934_b200" not in src
            assert "csrc" not in src.replace("paper_1212_2934_b200/csrc (the CUDA path)", "")


def test_checked_library_builds_and_exports_the_same_symbols():
    """libff_checked.so (-DFF_CHECKED: device-side index and bound checks in every kernel) is the same ABI."""
    from paper_1212_2934_b200 import build
    L = ctypes.CDLL(build.build(checked=True))
    for n in _declared():
        assert hasattr(L, n), n
