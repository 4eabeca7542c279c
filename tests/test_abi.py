"""The C-ABI library loads and exports every symbol include/hcc.h declares (no compute
calls: this runs without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "hcc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"HCC_API\s+[\w\s\*]*?\b(hcc_\w+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_2305_16652_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert len(names) >= 25
    for n in names:
        assert hasattr(lib, n), n


def test_binding_covers_the_header():
    import paper_2305_16652_b200 as h
    assert h.EXPORTS == _declared()
    assert h.version() >= 100
    assert h.lib().hcc_last_error() == b"" or isinstance(h.lib().hcc_last_error(), bytes)


def test_host_side_argument_checks_need_no_gpu():
    import paper_2305_16652_b200 as h
    need = ctypes.c_uint64()
    assert h.lib().hcc_sort_workspace_bytes(1 << 20, 32, ctypes.byref(need)) == 0
    assert need.value >= (1 << 20) * 8
    assert h.lib().hcc_sort_workspace_bytes(1 << 20, 48, ctypes.byref(need)) == -1
    assert b"container_bits" in h.lib().hcc_last_error()
    assert h.lib().hcc_sort_workspace_bytes(1 << 31, 32, ctypes.byref(need)) == -5


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2305_16652_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".c")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "oracle/" not in text and "hcc_oracle" not in text, f
