"""CPU-side checks of the C-ABI boundary: libhardkv.so loads, exports every symbol include/hardkv.h
declares, and its host-only entry points (no GPU needed) validate their arguments."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__
    __graft_entry__.build()
    from paper_2606_28831_b200 import hardkv
    return hardkv


def declared_functions():
    src = open(os.path.join(ROOT, "include", "hardkv.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hardkv_[a-z_]+)\s*\(", src)))


def test_header_symbols_exported(lib):
    names = declared_functions()
    assert len(names) >= 12 and set(names) == set(lib.EXPORTS)
    so = C.CDLL(os.path.join(ROOT, "paper_2606_28831_b200", "libhardkv.so"))
    for n in names:
        assert hasattr(so, n), n


def test_struct_layout_matches_header(lib):
    assert C.sizeof(lib.Config) == 16 * 4
    assert C.sizeof(lib.StateStruct) == 32 * C.sizeof(C.c_void_p)


def test_host_only_validation(lib):
    ok = lib.Config(2, 32, 8, 128, 16, 4096, 4, 128, 1024, 256, 0, lib.BF16, 0.0)
    n = C.c_size_t()
    assert lib.lib.hardkv_workspace_bytes(C.byref(ok), C.byref(n)) == 0 and n.value > 0 and n.value % 256 == 0
    bad_g = lib.Config(2, 24, 8, 128, 16, 4096, 4, 128, 1024, 256, 0, lib.BF16, 0.0)       # G = 3
    assert lib.lib.hardkv_workspace_bytes(C.byref(bad_g), C.byref(n)) == 2
    bad_page = lib.Config(2, 32, 8, 128, 32, 4096, 4, 128, 1024, 256, 0, lib.BF16, 0.0)
    assert lib.lib.hardkv_workspace_bytes(C.byref(bad_page), C.byref(n)) == 2
    bad_ctx = lib.Config(2, 32, 8, 128, 16, 4100, 4, 128, 1024, 256, 0, lib.BF16, 0.0)
    assert lib.lib.hardkv_workspace_bytes(C.byref(bad_ctx), C.byref(n)) == 1
    even_pool = lib.Config(2, 32, 8, 128, 16, 4096, 4, 128, 1024, 256, 0, lib.BF16, 0.0, 6)  # SNAPKV window must be odd
    assert lib.lib.hardkv_workspace_bytes(C.byref(even_pool), C.byref(n)) == 1
    pooled = lib.Config(2, 32, 8, 128, 16, 4096, 4, 128, 1024, 256, 0, lib.BF16, 0.0, 7)
    m = C.c_size_t()
    assert lib.lib.hardkv_workspace_bytes(C.byref(pooled), C.byref(m)) == 0 and m.value >= n.value + 2 * 32 * 4096 * 4
    ctx = C.c_void_p()
    assert lib.lib.hardkv_create(C.byref(ok), None, 0, C.byref(ctx)) == 3                   # no workspace
    assert b"workspace" in lib.lib.hardkv_status_string(3)
    assert lib.lib.hardkv_append_kv(None, None, None, None, None) == 1
