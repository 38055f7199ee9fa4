"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/ic.h declares; argument
validation that needs no device.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_2301_11735_b200 as p
    return p


def declared_functions():
    text = open(os.path.join(ROOT, "include", "ic.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ic_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = declared_functions()
    for must in ["ic_create", "ic_sweep", "ic_observables", "ic_state", "ic_set_state", "ic_sweep_trace",
                 "ic_reset_observables", "ic_debug_recompute", "ic_destroy", "ic_strerror", "ic_workspace_bytes"]:
        assert must in names


def test_library_exports_every_declared_symbol(pkg):
    raw = C.CDLL(pkg.LIB_PATH)
    for name in declared_functions():
        assert hasattr(raw, name), f"{name} declared in include/ic.h but not exported"
        assert name in pkg.EXPORTS, f"{name} has no Python binding"
    assert set(pkg.EXPORTS) == set(declared_functions())


def test_library_is_built_in_tree(pkg):
    assert os.path.dirname(pkg.LIB_PATH) == os.path.join(ROOT, "paper_2301_11735_b200")


def test_workspace_bytes_and_size_errors(pkg):
    lib = pkg.lib
    assert lib.ic_workspace_bytes(16384, 1, 8) >= 16384 * 16384
    assert lib.ic_workspace_bytes(16384, 1, 2) >= 16384 * 16384 // 4
    assert lib.ic_workspace_bytes(64, 64, 8) >= 64 * 64 * 64
    for bad in [(0, 1, 8), (3, 1, 8), (48, 1, 8), (2, 1, 8), (64, 0, 8), (64, 1, 4), (131072, 1, 8)]:
        assert lib.ic_workspace_bytes(*bad) == 0
    h = C.c_void_p()
    assert lib.ic_create(None, 64, 0.1, 0, 0, 0, 1, 1, 8, None, 0, None) == pkg.IC_ERR_NULL
    assert lib.ic_create(C.byref(h), 48, 0.1, 0, 0, 0, 1, 1, 8, None, 0, None) == pkg.IC_ERR_SIZE
    assert lib.ic_create(C.byref(h), 64, 1.5, 0, 0, 0, 1, 1, 8, None, 0, None) == pkg.IC_ERR_PARAM
    assert lib.ic_create(C.byref(h), 64, float("nan"), 0, 0, 0, 1, 1, 8, None, 0, None) == pkg.IC_ERR_PARAM
    assert lib.ic_create(C.byref(h), 64, 0.1, 0, 0, 0, 1, 1, 8, None, 0, None) == pkg.IC_ERR_WORKSPACE
    assert lib.ic_create(C.byref(h), 64, 0.1, 0, 0, 0, 1, 1, 8, C.c_void_p(256), 16, None) == pkg.IC_ERR_WORKSPACE
    assert lib.ic_create(C.byref(h), 64, 0.1, 0, 0, 0, 1, 1, 8, C.c_void_p(257), 1 << 30, None) == pkg.IC_ERR_WORKSPACE
    assert h.value is None
    for code in range(0, -8, -1):
        assert len(lib.ic_strerror(code)) > 0
    assert lib.ic_sweep(None, None, 1) == pkg.IC_ERR_NULL
    assert lib.ic_sweep_count(None) == -1


def test_no_cpu_path_without_device(pkg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(RuntimeError):
        pkg.Sim(16, 0.25, 0.5, 1.0, 1.0, seed=1)


def test_product_does_not_touch_the_oracle():
    """The product path shares nothing with oracle/: no import, include or link in either direction."""
    pk = os.path.join(ROOT, "paper_2301_11735_b200")
    for dp, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dp, f)).read()
                assert "oracle" not in src.replace("no CPU", ""), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2301_11735_b200" not in src and "libic_b200" not in src
            assert "#include \"ic.h\"" not in src and "ic_common" not in src
