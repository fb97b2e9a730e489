"""The C-ABI library loads and exports every symbol include/*.h declares (mcdc.h: the product boundary; mcdc_test.h: the
unit-level and micro-benchmark entry points) -- no compute call, no GPU."""
import ctypes
import os
import re

from paper_2501_05440_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include")))
                  if f.endswith(".h"))
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mcdc_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    so = binding.build()
    L = ctypes.CDLL(so)
    syms = declared_symbols()
    assert len(syms) >= 17
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(binding.SYMBOLS) == syms


def test_product_header_has_no_test_entry_points():
    src = open(os.path.join(ROOT, "include", "mcdc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    assert not re.findall(r"\bmcdc_(test_[a-z_]+|microbench)\s*\(", src)


def test_binding_struct_sizes_match_header():
    """Field-by-field layouts are plain C; spot-check sizes the header implies (LP64)."""
    assert ctypes.sizeof(binding.Device) == 48
    assert ctypes.sizeof(binding.Dims) == 24
    assert binding.TRACE_DTYPE.itemsize == 88 and binding.SITE_DTYPE.itemsize == 56
    assert ctypes.sizeof(binding.Source) == 3 * 8 * 3 + 8 + 8 + 16


def test_no_cpu_fallback_without_gpu():
    import pytest
    import torch
    from paper_2501_05440_b200 import inputs
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.McdcError):
        binding.Problem(inputs.config1(n_particles=10))


def test_product_never_imports_oracle():
    for f in ("binding.py", "inputs.py", "__init__.py"):
        s = open(os.path.join(ROOT, "paper_2501_05440_b200", f)).read()
        assert "import oracle" not in s and "from oracle" not in s
