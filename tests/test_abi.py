"""The C-ABI library loads and exports every symbol include/*.h declare (no compute calls: no GPU here)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include"))) if f.endswith(".h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gc_[a-z0-9_]+)\s*\(", src)) - {"gc_alloc_fn", "gc_free_fn"})


def test_library_exports_every_declared_symbol():
    from paper_1901_06798_b200 import build, binding
    build.build()
    lib = binding.lib()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "missing symbol " + n
    assert sorted(binding.SYMBOLS) == names


def test_no_cpu_fallback_without_gpu():
    import torch
    from paper_1901_06798_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Context(coord=0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1901_06798_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "gco" not in txt.replace("gco_", "gco_") or "oracle" not in txt or f == "binding.py", f
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert '#include "gco' not in txt and "oracle/" not in txt.replace("Shares nothing with oracle/", ""), f
