"""The C-ABI library loads and exports every symbol include/sap.h declares (no compute calls: no GPU needed)."""
import ctypes
import os
import re

from paper_2606_30460_b200 import _lib

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "sap.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sap_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported_and_bound():
    names = declared_symbols()
    assert len(names) >= 20
    L = ctypes.CDLL(_lib.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in sap.h but not exported"
        assert n in _lib.SIGNATURES, f"{n} has no ctypes signature in the binding"
    assert sorted(_lib.SIGNATURES) == names


def test_strerror_and_launch_count_without_gpu():
    L = _lib.lib()
    assert L.sap_strerror(0) == b"ok"
    assert b"divisible" in L.sap_strerror(3)
    assert L.sap_launch_count() >= 0


def test_item_struct_is_ten_int32():
    assert ctypes.sizeof(_lib.SapItem) == 40
