"""The C-ABI library builds, loads and exports every symbol include/*.h declares (no GPU, no compute)."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2310_09200_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        text = re.sub(r"/\*.*?\*/", "", open(h).read(), flags=re.S)
        names |= set(re.findall(r"\b(bb_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_every_declared_symbol_is_exported(lib):
    from paper_2310_09200_b200 import binding
    decl = declared_symbols()
    assert len(decl) >= 15
    for name in decl:
        assert hasattr(lib, name), "header declares %s but the library does not export it" % name
    assert sorted(binding.EXPORTS) == decl


def test_status_strings_and_version(lib):
    assert lib.bb_status_string(0) == b"ok"
    assert b"invalid" in lib.bb_status_string(1)
    assert b"sm_100a" in lib.bb_version()


def test_no_silent_cpu_fallback(lib):
    """Without a CUDA device the context cannot be created: the product path fails loudly."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2310_09200_b200 import binding
    with pytest.raises(binding.BluebildError) as e:
        binding.Context(0)
    assert e.value.code == 3  # BB_ECUDA


def test_product_never_imports_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_2310_09200_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "liboracle" not in text and not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
    for f in glob.glob(os.path.join(ROOT, "oracle", "*")):
        if f.endswith((".py", ".cpp")):
            text = open(f).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2310_09200_b200", text, flags=re.M), f
            assert not re.search(r"#include\s+\"[^\"]*(paper_2310_09200_b200|bluebild\.h|internal\.h)", text), f
            assert "libbluebild" not in text, f
