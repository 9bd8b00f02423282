"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol that
include/hydro.h declares, and its argument validation / workspace arithmetic behave as documented."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1604_03360_b200 import build
    path = build.build()
    lib = ctypes.CDLL(path)
    lib.hydro_create.argtypes = [ctypes.POINTER(ctypes.c_void_p)] + [ctypes.c_int] * 3 + [ctypes.c_double, ctypes.c_int]
    lib.hydro_set_option.argtypes = [ctypes.c_void_p, ctypes.c_char_p, ctypes.c_double]
    lib.hydro_workspace_bytes.argtypes = [ctypes.c_void_p]
    lib.hydro_workspace_bytes.restype = ctypes.c_size_t
    lib.hydro_bind_workspace.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
    lib.hydro_step.argtypes = [ctypes.c_void_p, ctypes.c_double, ctypes.c_int]
    lib.hydro_last_error.argtypes = [ctypes.c_void_p]
    lib.hydro_last_error.restype = ctypes.c_char_p
    lib.hydro_destroy.argtypes = [ctypes.c_void_p]
    lib.hydro_destroy.restype = None
    return lib


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "hydro.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hydro_[a-zA-Z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert len(names) >= 18, names
    for n in names:
        assert hasattr(L, n), "libhydro_b200.so does not export %s" % n


def test_binding_lists_the_same_symbols():
    src = open(os.path.join(ROOT, "paper_1604_03360_b200", "binding.py")).read()
    listed = set(re.findall(r'"(hydro_[a-z_A-Z0-9]+)"', src))
    assert listed == set(declared_symbols())


def test_create_validates_arguments(L):
    h = ctypes.c_void_p()
    assert L.hydro_create(ctypes.byref(h), 0, 4, 4, 0.1, 0) == -1
    assert L.hydro_create(ctypes.byref(h), 8, 8, 8, -1.0, 0) == -1
    assert L.hydro_create(ctypes.byref(h), 8, 8, 8, 0.1, 3) == -1
    assert L.hydro_create(ctypes.byref(h), 8, 2, 8, 0.1, 0) == -1      # active axis shorter than g = 3
    assert L.hydro_create(None, 8, 8, 8, 0.1, 0) == -1
    assert L.hydro_create(ctypes.byref(h), 400, 1, 1, 0.005, 0) == 0   # the shock tube shape
    L.hydro_destroy(h)


@pytest.mark.parametrize("scheme,g", [(0, 3), (1, 4), (2, 2)])
def test_workspace_size_follows_the_padded_layout(L, scheme, g):
    h = ctypes.c_void_p()
    n = (20, 12, 9)
    assert L.hydro_create(ctypes.byref(h), n[0], n[1], n[2], 0.1, scheme) == 0
    for prec, es in ((0, 8), (1, 4)):
        assert L.hydro_set_option(h, b"precision", float(prec)) == 0
        sx = -(-(n[0] + 2 * g) // (16 // es)) * (16 // es)
        vol = sx * (n[1] + 2 * g) * (n[2] + 2 * g)
        fs = -(-vol // (256 // es)) * (256 // es)
        # three states: the marching kernels keep no primitive arrays ...
        assert L.hydro_set_option(h, b"kernel", 0.0) == 0
        assert L.hydro_workspace_bytes(h) == 256 + 3 * 5 * fs * es
        # ... the generic kernel keeps one set of seven
        assert L.hydro_set_option(h, b"kernel", 1.0) == 0
        assert L.hydro_workspace_bytes(h) == 256 + (3 * 5 + 7) * fs * es
    L.hydro_destroy(h)


def test_options_and_call_order(L):
    h = ctypes.c_void_p()
    assert L.hydro_create(ctypes.byref(h), 16, 16, 16, 0.1, 0) == 0
    assert L.hydro_set_option(h, b"bc_x", 1.0) == 0
    assert L.hydro_set_option(h, b"bc_y", 7.0) == -1
    assert L.hydro_set_option(h, b"weno_eps", 0.0) == -1
    assert L.hydro_set_option(h, b"no_such_option", 1.0) == -1
    assert b"no_such_option" in L.hydro_last_error(h)
    # stepping without a workspace is refused, not executed on the host
    assert L.hydro_step(h, 0.01, 1) == -2
    assert L.hydro_bind_workspace(h, ctypes.c_void_p(0x1001), 1 << 30) == -1     # misaligned
    assert L.hydro_bind_workspace(h, ctypes.c_void_p(0x1000), 16) == -2          # too small
    L.hydro_destroy(h)


def test_binding_refuses_to_run_without_the_library(tmp_path, monkeypatch):
    """The product path fails loudly when the CUDA library is missing (no CPU fallback)."""
    import importlib
    import sys
    sys.modules.pop("paper_1604_03360_b200.binding", None)
    import os.path as osp
    real = osp.exists
    monkeypatch.setattr(osp, "exists", lambda p: False if str(p).endswith("libhydro_b200.so") else real(p))
    with pytest.raises(ImportError):
        importlib.import_module("paper_1604_03360_b200.binding")
    sys.modules.pop("paper_1604_03360_b200.binding", None)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1604_03360_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "hydro_oracle" not in text, f
