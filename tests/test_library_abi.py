"""CPU checks of the boundary: libpawfe.so loads and exports every symbol include/pawfe.h declares; the
product fails loudly without a GPU (no CPU fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_26037_b200 import build
    build.build()
    from paper_2604_26037_b200 import load_library
    return load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "pawfe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pawfe_[A-Za-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    from paper_2604_26037_b200 import SYMBOLS
    declared = _declared_symbols()
    assert declared == sorted(SYMBOLS)
    for s in declared:
        assert hasattr(lib, s), s


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2604_26037_b200 import Context, PawfeError
    with pytest.raises(PawfeError):
        Context(0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2604_26037_b200")
    for root, _d, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(root, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "oracle/" not in src.replace("under oracle/", ""), f
