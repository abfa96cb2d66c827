"""Host-side checks of the C ABI that need no GPU: the library builds, loads, exports every
symbol include/pty.h declares, and validates dims / sizes the workspace on the host."""
import ctypes as C
import os
import re

import pytest


@pytest.fixture(scope="module")
def lib(repo_root):
    from paper_2505_07814_b200 import build
    path = build.build()
    assert os.path.exists(path)
    return C.CDLL(path)


def declared_functions(repo_root):
    text = open(os.path.join(repo_root, "include", "pty.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pty_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib, repo_root):
    names = declared_functions(repo_root)
    assert {"pty_forward_loss", "pty_backward", "pty_step", "pty_create", "pty_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/pty.h but not exported by libpty.so"


def test_binding_lists_the_same_exports(repo_root):
    src = open(os.path.join(repo_root, "paper_2505_07814_b200", "binding.py")).read()
    for n in declared_functions(repo_root):
        assert f'"{n}"' in src


def test_workspace_bytes_and_dim_validation(lib):
    from paper_2505_07814_b200.binding import pty_dims
    lib.pty_last_error.restype = C.c_char_p
    out = C.c_size_t(0)
    d = pty_dims(6, 1088, 1088, 12, 128, 64, 5.0, 0.0197, 0.1, 0, 0)
    assert lib.pty_workspace_bytes(C.byref(d), C.byref(out)) == 0
    waves = 64 * 12 * (6 + 1) * 128 * 128 * 8            # incident waves + far field
    assert waves < out.value < waves * 1.1 and out.value % 256 == 0
    d2 = pty_dims(6, 1088, 1088, 12, 128, 64, 5.0, 0.0197, 0.1, 1, 0)
    out2 = C.c_size_t(0)
    assert lib.pty_workspace_bytes(C.byref(d2), C.byref(out2)) == 0
    assert out2.value > out.value                          # kept spectra for the tilt gradient
    for bad, code in ((pty_dims(1, 160, 160, 1, 96, 4, 1, 0.02, 0.1, 0, 0), -2),     # unsupported N
                      (pty_dims(1, 100, 160, 1, 128, 4, 1, 0.02, 0.1, 0, 0), -2),    # window > object
                      (pty_dims(0, 160, 160, 1, 64, 4, 1, 0.02, 0.1, 0, 0), -1),
                      (pty_dims(1, 160, 160, 1, 64, 4, 1, 0.02, 0.1, 3, 0), -1)):
        assert lib.pty_workspace_bytes(C.byref(bad), C.byref(out)) == code
        assert lib.pty_last_error(None) != b""
    assert lib.pty_workspace_bytes(None, C.byref(out)) == -1


def test_no_oracle_import_in_product(repo_root):
    """The product package never references the oracle (it is test infrastructure)."""
    pkg = os.path.join(repo_root, "paper_2505_07814_b200")
    for root, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(root, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b|#include.*oracle|import_module\(.oracle", text, re.M), f
