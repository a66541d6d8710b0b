"""No-GPU checks of the boundary: the C-ABI library builds, loads, and exports every symbol include/splitsolve.h
declares (no compute calls), and the host-side argument logic that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1812_01396_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "splitsolve.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ss_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("ss_create", "ss_set_hamiltonian", "ss_solve", "ss_transmission", "ss_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in splitsolve.h but not exported"


def test_binding_covers_every_declared_symbol(libpath):
    from paper_1812_01396_b200 import binding
    assert sorted(binding.SIGNATURES) == declared_symbols()
    binding.load()


def test_pure_host_queries(libpath):
    from paper_1812_01396_b200 import binding
    lib = binding.load()
    assert lib.ss_strerror(0) == b"ok"
    assert lib.ss_strerror(4) == b"exactly zero pivot"
    assert binding.workspace_bytes(1, 16, 1, 1) == 0            # nb >= 2 (reading c19)
    # C4 fits a 180 GB B200 together with H, S (25.2 GB): SURVEY.md §8(d)
    assert binding.workspace_bytes(24, 4096, 4, 512) < 120e9
    assert binding.workspace_bytes(8, 16, 4, 4) > 0
    # argument checks that never touch the device
    h = ctypes.c_void_p()
    assert lib.ss_create(1, 16, 1, ctypes.byref(h)) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_create(4, 5000, 1, ctypes.byref(h)) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_create(4, 16, 0, ctypes.byref(h)) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_destroy(None) == binding.SS_OK
    assert lib.ss_set_option(None, b"nb_lu", 64) == binding.SS_ERR_INVALID_ARG


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_1812_01396_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.load()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1812_01396_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+(paper_1812_01396_b200|ctypes)\b", src, flags=re.M), f
