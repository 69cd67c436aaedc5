"""Host-side checks that need no GPU: the C-ABI library loads, exports every symbol include/hair.h
declares, agrees with the ctypes struct layouts, and the product path refuses to run without CUDA."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2607_04230_b200 import build
    return build.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "hair.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hair_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(built):
    lib = ctypes.CDLL(built)
    names = declared_functions()
    assert len(names) >= 16
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/hair.h but not exported"


def test_binding_covers_the_header_and_layouts_match(built):
    from paper_2607_04230_b200 import binding
    binding.load()  # raises on a struct layout mismatch (hair_abi_sizes)
    assert sorted(binding.EXPORTS) == declared_functions()


def test_no_cpu_fallback():
    import torch
    from paper_2607_04230_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(binding.HairError):
        binding.Hair(0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_04230_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "hair_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "hair.h\"" not in txt and "hair_internal" not in txt and "binding" not in txt.replace("foreign-language binding", ""), f
