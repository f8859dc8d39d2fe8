"""CPU-only: the C-ABI library builds, loads, and exports every symbol include/dwf.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "dwf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dwf_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2103_05034_b200 import build as dwf_build
    from paper_2103_05034_b200 import exported_symbols
    lib = ctypes.CDLL(dwf_build.build())
    names = _declared()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), f"{n} declared in dwf.h but not exported"
    assert names == exported_symbols()            # the Python binding marshals exactly the declared calls


def test_binding_has_no_cpu_fallback():
    """The product path must fail loudly without a GPU: no oracle import, no CPU path."""
    import torch
    import paper_2103_05034_b200 as pkg
    src = open(os.path.join(ROOT, "paper_2103_05034_b200", "dwf.py")).read()
    assert "oracle" not in src
    if not torch.cuda.is_available():
        import pytest
        with pytest.raises(pkg.DwfError):
            pkg.Dwf((4, 4, 4, 4), 8, 1.8, 0.01, pkg.DWF_F64)
