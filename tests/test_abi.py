"""CPU-only checks of the C-ABI boundary: the library builds/loads, exports every function that
include/gsvox.h declares, and its host-side argument checking and workspace arithmetic work.
No kernel is launched here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as g
    g.build()
    import paper_2503_22139_b200 as p
    return p


def declared_functions(header="gsvox.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gsvox_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_agree(pkg):
    names = declared_functions()
    assert "gsvox_preprocess" in names and "gsvox_forward" in names and "gsvox_backward" in names
    assert sorted(pkg.EXPORTS) == names


def test_library_exports_every_declared_symbol(pkg):
    L = C.CDLL(pkg.LIB_PATH)
    for name in declared_functions():
        assert getattr(L, name) is not None
    assert pkg.lib().gsvox_version() >= 100


def test_probe_library_is_separate_from_the_product_library(pkg):
    """include/gsvox_probe.h (bench-only microbenchmarks) lives in libgsvox_probe.so, not in libgsvox.so."""
    names = declared_functions("gsvox_probe.h")
    assert names == sorted(pkg.PROBE_EXPORTS) == ["gsvox_probe_peaks"]
    P = pkg.probe_lib()
    for name in names:
        assert getattr(P, name) is not None
    with pytest.raises(AttributeError):
        getattr(C.CDLL(pkg.LIB_PATH), "gsvox_probe_peaks")


def test_library_is_sm100a_only_and_uses_no_tensor_cores(pkg):
    """The path is not a dense contraction (north_star): the cubin must target sm_100a."""
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", pkg.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out and not re.search(r"sm_(?!100a)\d+", out)


def test_workspace_bytes_and_argument_checks(pkg):
    L = pkg.lib()
    n = C.c_size_t(0)
    g = pkg.make_grid((0, 0, 0), (1, 1, 1), (256, 256, 256))
    assert L.gsvox_workspace_bytes(500000, 1, C.byref(g), 16_000_000, C.byref(n)) == 0
    # records 64 B + aux 32 B + accumulators 48 B per Gaussian, 4 B per key, 8 B per (brick, class) bin,
    # 8 B per hot-brick segment (one per 512 keys of capacity)
    expect = 500000 * (64 + 32 + 48) + 16_000_000 * 4 + 32768 * 17 * 8 + (16_000_000 // 512 + 1) * 8
    assert expect <= n.value <= expect + 8192
    bad = pkg.make_grid((0, 0, 0), (1, 0, 1), (8, 8, 8))
    assert L.gsvox_workspace_bytes(10, 1, C.byref(bad), 10, C.byref(n)) == -1
    bad = pkg.make_grid((0, 0, 0), (1, 1, 1), (8, 0, 8))
    assert L.gsvox_workspace_bytes(10, 1, C.byref(bad), 10, C.byref(n)) == -1
    assert L.gsvox_workspace_bytes(10, 97, C.byref(g), 10, C.byref(n)) == -1      # GSVOX_MAX_CHANNELS = 96
    assert L.gsvox_workspace_bytes(-1, 1, C.byref(g), 10, C.byref(n)) == -1
    big = pkg.make_grid((0, 0, 0), (1, 1, 1), (40000, 8, 8))
    assert L.gsvox_workspace_bytes(10, 1, C.byref(big), 10, C.byref(n)) == -5
    h = C.c_void_p(None)
    assert L.gsvox_plan_create(10, 1, C.byref(g), 10, None, 0, C.byref(h)) == -2       # no workspace
    assert L.gsvox_preprocess(None, None, None, None, 0, None) == -1
    assert L.gsvox_forward(None, None, 1, None, None) == -1
    for code in (0, -1, -2, -3, -4, -5):
        assert L.gsvox_error_string(code).decode() not in ("", "unknown error")
    assert L.gsvox_error_string(-99).decode() == "unknown error"


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg_dir = os.path.join(ROOT, "paper_2503_22139_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "gsvox_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            # the oracle may NAME the product package in prose (its header says who may import what); it may not
            # load it: no import, no ctypes/dlopen of the product library
            assert "libgsvox.so" not in text and "binding" not in text, f
            assert not re.search(r"^\s*(import|from)\s+paper_2503_22139_b200\b", text, flags=re.M), f
