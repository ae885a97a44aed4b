"""CPU-side checks of the boundary: the in-tree C-ABI library loads and exports every symbol
include/bem.h declares; no compute call is made (there is no CPU fallback to call)."""
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "bem.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(bem_[a-z0-9_]+)\s*\(", txt)))


def test_header_symbols_are_exported():
    from paper_1905_01341_b200.build import build
    lib_path = build()
    import paper_1905_01341_b200 as bem
    lib = bem.load_library()
    declared = _declared()
    assert sorted(bem.EXPORTS) == declared
    nm = subprocess.run(["nm", "-D", "--defined-only", lib_path], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (bem_[a-z0-9_]+)", nm))
    assert set(declared) <= exported
    for name in declared:
        assert getattr(lib, name) is not None


def test_library_is_sm100a_and_has_no_torch_dependency():
    import paper_1905_01341_b200 as bem
    out = subprocess.run(["cuobjdump", "-lelf", bem.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    ldd = subprocess.run(["ldd", bem.LIB_PATH], capture_output=True, text=True).stdout
    assert "torch" not in ldd and "c10" not in ldd


def test_no_cpu_fallback():
    """Without a device bem_create fails with BEM_ERR_CUDA; nothing is computed on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_1905_01341_b200 as bem
    import bem_inputs as bi
    V, F = bi.icosphere(1)
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(V, F)
    assert e.value.status == bem.BEM_ERR_CUDA


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1905_01341_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "bem_oracle" not in txt, f
    hdr = open(os.path.join(ROOT, "include", "bem.h")).read()
    assert "oracle" not in hdr.lower()
