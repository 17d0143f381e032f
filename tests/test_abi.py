"""The C-ABI library builds (nvcc cross-compiles without a GPU), loads, and exports every symbol that
include/etics.h declares.  Argument errors are reported synchronously, before any CUDA call, so the error
paths can be exercised without a device.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "etics.h")


@pytest.fixture(scope="module")
def libetics():
    from paper_1406_4254_b200 import build
    path = build.build()
    return C.CDLL(path)


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(etics_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for name in ("etics_scf_coeffs", "etics_scf_force", "etics_mex_force"):
        assert name in syms


def test_library_exports_every_declared_symbol(libetics):
    syms = declared_symbols()
    assert len(syms) >= 10
    for name in syms:
        assert hasattr(libetics, name), f"libetics.so does not export {name}"


def test_binding_lists_every_declared_symbol():
    from paper_1406_4254_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    for name in binding.EXPORTS:
        if name != "etics_status_string":
            assert hasattr(binding, name), f"binding lacks {name}"


def test_status_strings(libetics):
    libetics.etics_status_string.restype = C.c_char_p
    libetics.etics_status_string.argtypes = [C.c_int]
    assert libetics.etics_status_string(0) == b"ETICS_OK"
    for code in (-1, -2, -3, -4, -5, -6):
        assert libetics.etics_status_string(code).startswith(b"ETICS_ERR_")
    assert b"unknown" in libetics.etics_status_string(-99)


def test_argument_errors_are_synchronous(libetics):
    vp, ll, i, sz = C.c_void_p, C.c_longlong, C.c_int, C.c_size_t
    f = libetics.etics_scf_coeffs
    f.restype = i
    f.argtypes = [vp, vp, ll, i, i, vp, vp, vp, sz, vp]
    ok = 0x1000  # aligned dummy address; never dereferenced on the error paths
    assert f(ok, ok, 0, 10, 6, ok, ok, ok, 1 << 30, None) == -1          # N < 1
    assert f(ok, ok, 1 << 31, 10, 6, ok, ok, ok, 1 << 30, None) == -1    # N >= 2^31
    assert f(ok, ok, 100, -1, 6, ok, ok, ok, 1 << 30, None) == -1        # nmax < 0
    assert f(ok, ok, 100, 10, 11, ok, ok, ok, 1 << 30, None) == -2       # lmax beyond limit
    assert f(ok, ok, 100, 33, 6, ok, ok, ok, 1 << 30, None) == -2        # nmax beyond limit
    assert f(None, ok, 100, 10, 6, ok, ok, ok, 1 << 30, None) == -1      # null pointer
    assert f(ok + 8, ok, 100, 10, 6, ok, ok, ok, 1 << 30, None) == -3    # misaligned
    assert f(ok, ok, 100, 10, 6, ok, ok, ok, 8, None) == -4              # workspace too small
    g = libetics.etics_mex_force
    g.restype = i
    g.argtypes = [vp, vp, ll, i, vp, vp, vp, sz, vp]
    assert g(ok, ok, 0, 6, ok, ok, ok, 1 << 30, None) == -1
    assert g(ok, ok, 100, 11, ok, ok, ok, 1 << 30, None) == -2
    assert g(ok, ok, 100, 6, ok, ok, ok, 16, None) == -4
    h = libetics.etics_scf_force
    h.restype = i
    h.argtypes = [vp, ll, i, i, vp, vp, vp, vp, vp, sz, vp]
    assert h(ok, 100, 10, 6, None, ok, ok, ok, None, 0, None) == -1
    assert h(ok, 100, 10, 6, ok, ok, ok + 4, ok, None, 0, None) == -3


def test_workspace_sizes(libetics):
    f = libetics.etics_workspace_bytes
    f.restype = C.c_size_t
    f.argtypes = [C.c_int, C.c_longlong, C.c_int, C.c_int]
    for which in (0, 1, 2):
        for n in (1, 10_000, 1_000_000, 100_000_000):
            b = f(which, n, 10, 6)
            assert b >= 256 and b % 256 == 0
    assert f(4, 1000, 10, 6) == 0
    assert f(0, 0, 10, 6) == 0
    assert f(2, 1000, 10, 11) == 0
    # MEX workspace grows with N (sort double-buffers + sorted records), SCF coefficient workspace is bounded
    assert f(2, 100_000_000, 0, 8) > f(2, 1_000_000, 0, 8)
    assert f(0, 100_000_000, 10, 6) < (1 << 26)
    # the N = 10^8 configuration (BASELINE.json config 5) fits one B200 with its I/O arrays (6.4 GB)
    assert f(2, 100_000_000, 0, 8) + 64 * 100_000_000 < 150 * (1 << 30)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1406_4254_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
                assert "etics_oracle" not in src, fn
