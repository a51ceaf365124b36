"""The C-ABI library builds (nvcc cross-compiles without a GPU), loads, and exports every symbol that
include/picsarqed.h declares.  No compute calls here (no GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    with open(os.path.join(ROOT, "include", "picsarqed.h")) as f:
        return sorted(set(re.findall(r"\b(picsarqed_[a-z_0-9]+)\s*\(", f.read())))


def test_library_exports_every_declared_symbol():
    import paper_2110_00256_b200 as q
    lib = ctypes.CDLL(q.build())
    names = _declared()
    assert len(names) >= 15
    for name in names:
        assert hasattr(lib, name), name
    assert lib.picsarqed_version() & 1


def test_binding_covers_the_header():
    from paper_2110_00256_b200 import binding
    assert sorted(binding._SIGNATURES) == _declared()


def test_no_cpu_fallback():
    import pytest
    import torch
    import paper_2110_00256_b200 as q
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(q.PicsarQedError):
        q.Context(0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2110_00256_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                with open(os.path.join(dirpath, f)) as fh:
                    text = fh.read()
                assert "import oracle" not in text and "from oracle" not in text and "picsarqed_oracle" not in text, f
