"""The C-ABI library loads and exports every symbol include/aceapex.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_every_declared_symbol_is_exported():
    from paper_2606_18900_b200 import build
    path = build.build_cuda()
    hdr = open(os.path.join(ROOT, "include", "aceapex.h")).read()
    names = sorted(set(re.findall(r"\b(aceapex_[a-z0-9_]+)\s*\(", hdr)))
    assert len(names) >= 15
    lib = ctypes.CDLL(path)
    for n in names:
        assert hasattr(lib, n), n
    lib.aceapex_strerror.restype = ctypes.c_char_p
    assert lib.aceapex_strerror(0) == b"ok"
    assert lib.aceapex_open(None, 0, None, None) == -9          # E_ARG, no CUDA call made


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_18900_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".c", ".h")):
                text = open(os.path.join(d, f), errors="ignore").read()
                assert "acx_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f
