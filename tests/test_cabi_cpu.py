"""CPU-side checks of the boundary: the library builds/loads and exports every symbol include/rpa_b200.h declares;
without a GPU the product path fails loudly (no fallback)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rpa_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rpa_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2405_20258_b200 as rpa
    lib = rpa.load_library()
    syms = declared_symbols()
    assert "rpa_create" in syms and "rpa_correlation_energy" in syms and len(syms) >= 12
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in rpa_b200.h but not exported"
    assert sorted(rpa.EXPORTED_SYMBOLS) == syms


def test_no_cpu_fallback():
    import torch
    import paper_2405_20258_b200 as rpa
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(rpa.RpaError) as ei:
        rpa.rpa_create([1, 0, 0, 0, 1, 0, 0, 0, 1], [8, 8, 8], [[0, 0, 0]], [1.0], [[0, 0, 0]])
    assert ei.value.code == -3


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2405_20258_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{f} mentions the oracle"
    osrc = open(os.path.join(ROOT, "oracle", "rpa_oracle.py")).read()
    assert "import paper_2405_20258_b200" not in osrc and "from paper_2405_20258_b200" not in osrc
