"""The C-ABI library builds for sm_100a here (no GPU needed), loads, and exports every symbol include/tmw.h
declares; argument validation that happens before any CUDA call is checked too. No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2201_09004_b200 import build, tmw
    build.build()
    return tmw.load()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "tmw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tmw_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    from paper_2201_09004_b200 import tmw
    names = declared_symbols()
    assert set(names) == set(tmw.EXPORTS), (names, tmw.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_binary_targets_sm_100a():
    import subprocess
    from paper_2201_09004_b200 import tmw
    out = subprocess.run(["cuobjdump", "--list-elf", tmw.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out, out


def test_argument_validation_before_any_cuda_call(lib):
    from paper_2201_09004_b200 import tmw
    h = ctypes.c_void_p()
    g = np.zeros(8, dtype=np.float64)
    m = tmw.tmw_complex(0.1, 0.0)
    assert lib.tmw_create(None, 4, 4, g.ctypes.data, m, 0.0, None) == tmw.EINVAL
    assert lib.tmw_create(ctypes.byref(h), 4, 4, None, m, 0.0, None) == tmw.EINVAL
    for L, T in ((3, 4), (4, 7), (2, 2), (0, 4)):
        assert lib.tmw_create(ctypes.byref(h), L, T, g.ctypes.data, m, 0.0, None) == tmw.EINVAL
        assert h.value is None
        assert b"even" in lib.tmw_last_error(None)
    opt = tmw.make_options(reconstruct=13)
    assert lib.tmw_create(ctypes.byref(h), 4, 4, g.ctypes.data, m, 0.0, ctypes.byref(opt)) == tmw.EINVAL
    assert lib.tmw_create(ctypes.byref(h), 4, 4, g.ctypes.data, tmw.tmw_complex(float("nan"), 0.0), 0.0, None) == tmw.EINVAL
    # null context
    assert lib.tmw_apply(None, 0, 0, 0, None, None) == tmw.EINVAL
    assert lib.tmw_solve(None, None, None, 1e-10, None) == tmw.EINVAL
    assert lib.tmw_apply_multi(None, 0, 0, 0, 2, None, None) == tmw.EINVAL
    assert lib.tmw_apply_schur_multi(None, 0, 0, 2, None, None) == tmw.EINVAL
    assert lib.tmw_apply_schur_static(None, 0, 0, None, None) == tmw.EINVAL
    assert lib.tmw_solve_multi(None, 2, None, None, 1e-10, None) == tmw.EINVAL
    assert lib.tmw_cheb_apply(None, 1, (ctypes.c_double * 1)(1.0), 1.0, 0.0, None, None) == tmw.EINVAL
    bad = tmw.make_options(reconstruct=12, solver=7)  # unknown solver
    assert lib.tmw_create(ctypes.byref(h), 4, 4, g.ctypes.data, m, 0.0, ctypes.byref(bad)) == tmw.EINVAL
    # an options struct laid out by another version of the header: refused by its size, before anything is read from it
    for size in (0, ctypes.sizeof(tmw.tmw_options) - 4, ctypes.sizeof(tmw.tmw_options) + 8):
        other = tmw.make_options()
        other.struct_size = size
        assert lib.tmw_create(ctypes.byref(h), 4, 4, g.ctypes.data, m, 0.0, ctypes.byref(other)) == tmw.EINVAL
        assert b"struct_size" in lib.tmw_last_error(None)
    assert lib.tmw_spinor_bytes(None, 0) == 0
    assert lib.tmw_launch_count(None) == 0
    lib.tmw_destroy(None)


def test_no_fallback_when_library_missing(monkeypatch):
    from paper_2201_09004_b200 import tmw
    monkeypatch.setattr(tmw, "_lib", None)
    monkeypatch.setattr(tmw, "LIB_PATH", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        tmw.load()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2201_09004_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", text, flags=re.M), f
                assert "tmw_oracle" not in text and "liboracle" not in text, f
