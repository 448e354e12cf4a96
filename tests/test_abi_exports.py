"""-m "not gpu": the C-ABI library builds (nvcc cross-compiles), loads, and exports every symbol
include/concordia.h declares.  No compute call is made."""
import ctypes
import os
import re

import paper_2606_23521_b200 as cc

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "concordia.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cc_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    lib = cc.load_library()
    decl = _declared_symbols()
    assert len(decl) >= 20
    for name in decl:
        assert hasattr(lib, name), name
    assert sorted(cc.EXPORTS) == decl


def test_struct_sizes_match_header():
    assert ctypes.sizeof(cc.binding.cc_result) == 64
    assert ctypes.sizeof(cc.binding.cc_task) == 64
    assert ctypes.sizeof(cc.binding.cc_config) == 24
    assert ctypes.sizeof(cc.binding.cc_region_desc) == 56


def test_pure_host_entry_points():
    """cc_workspace_bytes / cc_apply_scratch_bytes are host arithmetic and need no GPU."""
    lib = cc.load_library()
    assert lib.cc_workspace_bytes(0, 4096) == 0
    assert lib.cc_workspace_bytes(4096, 100) == 0            # page size not a multiple of 16
    assert lib.cc_workspace_bytes(4096 + 8, 4096) == 0       # size not a multiple of 16
    w = lib.cc_workspace_bytes(8 << 30, 65536)
    assert 0 < w < (8 << 20)
    assert lib.cc_workspace_bytes(64 << 30, 4096) < (640 << 20)      # ~32 B per page: < 1 % of the region
    assert lib.cc_apply_scratch_bytes(0) == 0
    assert lib.cc_apply_scratch_bytes(10100) < (1 << 20)


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_23521_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "concordia_oracle" not in text, f
