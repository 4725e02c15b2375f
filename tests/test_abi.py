"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/pic.h declares; pure-host entry points behave (no kernel is launched here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1603_02886_b200 import build
    build.build()
    import paper_1603_02886_b200 as B
    return B


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "pic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pic_[a-z_]+)\s*\(", src)))


def test_header_declares_the_contract():
    syms = declared_symbols()
    for name in ("pic_sort", "pic_deposit", "pic_push", "pic_step", "pic_workspace_bytes", "pic_strerror"):
        assert name in syms


def test_library_exports_every_declared_symbol(B):
    L = ctypes.CDLL(B.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(L, name), name
    assert sorted(B.EXPORTS) == declared_symbols()


def test_binding_has_the_same_names(B):
    for name in declared_symbols():
        if name != "pic_strerror":
            assert callable(getattr(B, name)), name


def test_workspace_bytes_and_validation_on_host(B):
    g = B.Grid(3, (128, 128, 128), (1.0, 1.0, 1.0), 3, "f32")
    n = 100_000_000
    b = B.pic_workspace_bytes(g, n)
    assert b % 256 == 0 and b >= 32 * n                     # movers' key and index arrays, one key per position, record scratch
    assert b < 36 * n + 64 * 2 ** 20
    assert B.pic_step_host_bytes(g, n) > b + 14 * 4 * n
    assert B.pic_workspace_bytes(g, 0) > 0
    for bad in (B.Grid(1, (8,), (1.0,), 1, "f32"), B.Grid(2, (8, 8), (1.0, 1.0), 0, "f32"),
                B.Grid(2, (8, 3), (1.0, 1.0), 3, "f64"), B.Grid(2, (8, 8), (1.0, -1.0), 1, "f64"),
                B.Grid(3, (2048, 2048, 1024), (1.0, 1.0, 1.0), 1, "f32")):
        with pytest.raises(B.PicError, match="invalid argument"):
            B.pic_workspace_bytes(bad, 10)
    with pytest.raises(B.PicError):
        B.pic_workspace_bytes(g, -1)
    with pytest.raises(B.PicError):
        B.pic_workspace_bytes(g, 2 ** 30)
    assert B.lib().pic_strerror(0) == b"ok"
    assert b"workspace" in B.lib().pic_strerror(-3)


def test_missing_library_fails_loudly(B, monkeypatch):
    import paper_1603_02886_b200 as mod
    monkeypatch.setattr(mod, "_lib", None)
    monkeypatch.setattr(mod, "LIB_PATH", "/nonexistent/libpic_b200.so")
    with pytest.raises(mod.PicError, match="no CPU fallback"):
        mod.pic_workspace_bytes(mod.Grid(2, (8, 8), (1.0, 1.0), 1, "f32"), 10)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1603_02886_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                s = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in s and "from oracle" not in s and "pic_ref" not in s, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1603_02886_b200" not in s and "csrc" not in s, f


def test_host_only_entry_points_of_the_next_rows(B):
    """Pure host computations of the NEXT rows: bucket counts, workspace sizes, argument validation (no kernel runs)."""
    g = B.Grid(3, (128, 128, 128), (1.0, 1.0, 1.0), 3, "f32")
    assert B.pic_bucket_count(g, (1, 1, 1)) == 128 ** 3
    assert B.pic_bucket_count(g, (4, 4, 4)) == 32 ** 3
    assert B.pic_bucket_count(g, (5, 128, 3)) == 26 * 1 * 43          # ragged last buckets
    for bad in ((0, 1, 1), (1, 129, 1), (1, 1, -2)):
        with pytest.raises(B.PicError, match="invalid argument"):
            B.pic_bucket_count(g, bad)
    C = 128 ** 3
    assert B.pic_field_solve_bytes(g) >= 2 * 16 * C                   # two complex-double grids
    n = 1_000_000
    base = B.pic_workspace_bytes(g, n)
    assert B.pic_step_selfconsistent_bytes(g, n) == base + B.pic_field_solve_bytes(g)
    assert B.pic_deposit_replicated_bytes(g, n) == base + 64 * 8 * C  # 4^3 local-grid nodes per cell, double
    g2 = B.Grid(2, (64, 32), (1.0, 1.0), 1, "f64")
    assert B.pic_deposit_replicated_bytes(g2, 10) == B.pic_workspace_bytes(g2, 10) + 4 * 8 * 64 * 32
    with pytest.raises(B.PicError):
        B.pic_deposit_replicated_bytes(g, 2 ** 30)
