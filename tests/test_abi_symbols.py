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
    assert lib.ss_set_option(None, b"stream_groups", 2) == binding.SS_ERR_INVALID_ARG


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


def test_host_side_argument_logic_without_a_device(libpath):
    """Calls that must answer from host logic alone (no CUDA work): argument validation, closed forms, strings."""
    from ctypes import byref, c_void_p
    from paper_1812_01396_b200 import binding
    lib = binding.load()
    h = c_void_p()
    # nb >= 2, 1 <= bs <= 4096, n_energy >= 1 (include/splitsolve.h "Limits"); rejected before any CUDA call
    for nb, bs, ne in ((1, 8, 1), (2, 0, 1), (2, 4097, 1), (2, 8, 0)):
        assert lib.ss_create(nb, bs, ne, byref(h)) == binding.SS_ERR_INVALID_ARG
        assert not h.value
    assert lib.ss_create(2, 8, 1, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_destroy(None) == binding.SS_OK
    assert lib.ss_solve(None, None, None, None, None, None, 0, None, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_transmission(None, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_set_option(None, b"stream_groups", 2) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_strerror(binding.SS_OK) == b"ok" and lib.ss_strerror(binding.SS_ERR_SINGULAR) == b"exactly zero pivot"
    assert lib.ss_workspace_bytes(1, 8, 1, 1) == 0 and lib.ss_workspace_bytes(2, 8, 1, -1) == 0
    # workspace grows with every size argument and is dominated by the 2 (nb+1) bs^2 slots per energy
    w = lib.ss_workspace_bytes(32, 2048, 8, 256)
    assert w >= 8 * 2 * 33 * 2048 * 2048 * 16
    assert lib.ss_workspace_bytes(32, 2048, 8, 512) > w and lib.ss_workspace_bytes(33, 2048, 8, 256) > w
    assert w < 100e9                                   # config C3 fits a B200
    assert lib.ss_workspace_bytes(24, 4096, 4, 512) < 100e9
    assert lib.ss_flops(None, 1) == 0.0 and lib.ss_flops_sweep(None) == 0.0
    d = binding.get_default_gemm_variant()
    assert lib.ss_set_default_gemm_variant(-1) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_set_default_gemm_variant(len(binding.GEMM_VARIANTS)) == binding.SS_ERR_INVALID_ARG
    assert binding.get_default_gemm_variant() == d
    assert lib.ss_zgemm_batched(-1, 1, 1, 1.0, None, 1, 0, None, 1, 0, 0.0, None, 1, 0, 1, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_zgetrf_batched(0, 0, None, 0, 0, None, None, 1, None, 0, None) == binding.SS_ERR_INVALID_ARG
    # a C sum plane cannot be honoured by the 4M kernel: refused before anything is launched (fake non-NULL pointers)
    try:
        assert lib.ss_set_default_gemm_variant(0) == binding.SS_OK
        assert lib.ss_zgemm_batched_sums(8, 8, 8, 1.0, 4096, None, 8, 64, 4096, None, 8, 64, 0.0, 4096, 4096, 8, 64, 1, None) \
            == binding.SS_ERR_INVALID_ARG
    finally:
        lib.ss_set_default_gemm_variant(d)
    # the no-allocation LU: the size limit is host arithmetic and comes before any device access
    assert lib.ss_zgesv_batched_noalloc(1024, 4, 4096, 1028, 0, 4096, 4, 0, 4096, 4096, 2, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_zgesv_batched_noalloc(0, 0, None, 0, 0, None, 0, 0, None, None, 1, None) == binding.SS_ERR_INVALID_ARG
    assert lib.ss_lu_workspace_bytes(0, 1) == 0 and lib.ss_lu_workspace_bytes(300, 2) >= 2 * 2 * 3 * 128 * 128 * 16
    assert lib.ss_lu_workspace_bytes(300, 4) > lib.ss_lu_workspace_bytes(300, 2) > lib.ss_lu_workspace_bytes(100, 2)


def test_closed_form_flop_counts_match_survey_table():
    """F_sweep = (160/3 nb - 32) bs^3; per-energy totals 0.505 / 16.0 / 97.4 TFLOP for C2-C4.
    (ss_flops needs a handle, hence a device; the same closed form is restated here against the table.)"""
    def f_sweep(nb, bs):
        return (160.0 / 3.0 * nb - 32.0) * bs ** 3

    def f_total(nb, bs, m):
        return f_sweep(nb, bs) + (32 + 64 / 3) * bs ** 3 + 32 * bs * bs * m + 16 * nb * bs * bs * m + 64 * bs ** 3 + 8 * bs * bs
    assert abs(f_sweep(64, 512) / 1e12 - 0.454) < 5e-4
    assert abs(f_sweep(32, 2048) / 1e12 - 14.4) < 5e-2
    assert abs(f_sweep(24, 4096) / 1e12 - 85.8) < 5e-2
    assert abs(f_total(64, 512, 128) / 1e12 - 0.505) < 1e-3
    assert abs(f_total(32, 2048, 256) / 1e12 - 16.0) < 5e-2
    assert abs(f_total(24, 4096, 512) / 1e12 - 97.4) < 5e-2


def test_library_links_no_vendor_math_library(libpath):
    """north_star: "no cuBLAS/cuSOLVER on the hot path" -- the shared library depends on the CUDA runtime only (statically
    linked by nvcc), not on cuBLAS, cuSOLVER, cuFFT, NCCL or torch."""
    import subprocess
    out = subprocess.run(["ldd", libpath], capture_output=True, text=True).stdout.lower()
    for name in ("cublas", "cusolver", "cufft", "nccl", "torch", "c10"):
        assert name not in out, name
