"""CPU-only checks of the C-ABI library: it loads without a GPU, exports every symbol that
include/bh.h declares, and its host-side argument validation works.  No compute calls."""
import ctypes as C
import os
import re

import pytest

from paper_1912_04197_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "bh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(bh_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = binding.lib()
    names = _declared()
    assert len(names) >= 20
    for name in names:
        assert hasattr(L, name), f"{name} declared in include/bh.h but not exported"
    assert set(names) == set(binding.EXPORTS)
    assert b"sm_100a" in L.bh_version()


def test_workspace_bytes_host_logic():
    wb = binding.bh_workspace_bytes
    assert wb(0, 16) == 0 and wb(1024, 0) == 0 and wb(1024, 16, 33) == 0 and wb(1024, 16, -1) == 0 and wb((1 << 30) + 1, 16) == 0
    a, b, c = wb(1024, 8), wb(1 << 20, 16), wb(1 << 22, 32)
    assert 0 < a < b < c
    assert b < 1 << 30                      # N=1M fits in well under 1 GiB
    assert c < 4 << 30
    assert wb(1 << 20, 16, 32) == b         # group_size 0 means 32
    assert wb(1 << 20, 16, 1) == b          # any W in 1..32 (the group arrays are sized for one body per group)
    assert wb(1 << 20, 1) > b               # smaller leaves -> larger node bound


def test_create_rejects_bad_arguments_without_gpu():
    L = binding.lib()
    ctx = C.c_void_p()
    assert L.bh_create(C.byref(ctx), 1024, 8, 0, None, 0, None) == binding.BH_ERR_INVALID_ARG
    assert L.bh_create(C.byref(ctx), 0, 8, 0, 256, 1 << 20, None) == binding.BH_ERR_INVALID_ARG
    assert L.bh_create(C.byref(ctx), 1024, 8, 0, 256 + 8, 1 << 30, None) == binding.BH_ERR_INVALID_ARG   # misaligned
    assert L.bh_create(C.byref(ctx), 1024, 8, 0, 256, 16, None) == binding.BH_ERR_CAPACITY               # too small
    assert ctx.value is None
    assert L.bh_build(None, None, None, 5) == binding.BH_ERR_INVALID_ARG
    assert L.bh_set_group_cell(None, 64) == binding.BH_ERR_INVALID_ARG
    assert b"workspace" in L.bh_last_error(None)


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libbh.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lib()


def test_profile_rows_match_the_kernel_sources():
    """profiles/r03_roofline.csv carries a fingerprint of each kernel's sources at its ncu capture; bench.py marks a row
    stale when the sources have changed since.  No committed row may be stale: a kernel edit needs a new capture."""
    import csv

    import bench
    with open(bench.PROFILE_CSV) as f:
        rows = list(csv.DictReader(f))
    assert len(rows) >= 10
    for r in rows:
        assert bench.source_sha1(r["source_files"]) == r["source_sha1"], (r["kernel"], r["config"], r["commit"])
    assert bench.profile_row("walk_kernel", "c4")["stale"] is False
    assert bench.profile_row("walk_kernel", "c9") is None

