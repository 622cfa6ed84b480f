"""CPU-side checks of the boundary: libtaiga.so builds, loads, and exports every symbol that
include/taiga.h declares (no compute calls without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "taiga.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(taiga_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2506_15812_b200 import build as tb
    lib = ctypes.CDLL(tb.build())
    names = _declared()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_same_entry_points():
    from paper_2506_15812_b200 import taiga
    assert sorted(taiga.EXPORTS) == _declared()


def test_null_arguments_are_rejected_without_a_device():
    from paper_2506_15812_b200 import build as tb
    lib = ctypes.CDLL(tb.build())
    assert lib.taiga_create(None, 0, None) == -1
    assert lib.taiga_destroy(None) == -1
    assert lib.taiga_load_field(None, None, None) == -1
    lib.taiga_last_error.restype = ctypes.c_char_p
    assert lib.taiga_last_error(None) == b"null context"


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_2506_15812_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("the CPU oracle", "").replace("CPU oracle", "") \
                    or f == "workloads.py" or f == "__init__.py", f
