"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/sparse_sv.h declares (no compute calls without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared(header="sparse_sv.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sv_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_mandated_calls():
    d = _declared()
    for name in ("sv_create", "sv_apply_gate", "sv_truncate", "sv_norm", "sv_top"):
        assert name in d


def test_library_exports_every_declared_symbol():
    from paper_2607_07816_b200 import build
    lib = ctypes.CDLL(build.build())
    for name in _declared() + _declared("sparse_sv_test.h"):
        assert hasattr(lib, name), name


def test_binding_lists_every_declared_symbol():
    import importlib
    eng = importlib.import_module("paper_2607_07816_b200.engine")
    assert sorted(eng.EXPORTS) == _declared()
    assert sorted(eng.TEST_EXPORTS) == _declared("sparse_sv_test.h")
    assert eng.lib.sv_arena_bytes(1 << 20) >= (1 << 20) * 48


def test_no_oracle_import_in_product():
    pkg = os.path.join(ROOT, "paper_2607_07816_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "sv_oracle" not in txt, f
