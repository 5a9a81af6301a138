"""The C-ABI library loads and exports every symbol include/fsei.h declares; argument errors are
reported loudly and there is no CPU fallback (-m "not gpu": no compute calls)."""
import os
import re

import numpy as np
import pytest

from paper_2103_15187_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "fsei.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fsei_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported():
    L = binding.lib()
    names = declared_functions()
    assert len(names) >= 8 and set(names) == set(binding.EXPORTS)
    for n in names:
        assert hasattr(L, n), n


def test_argument_errors_and_no_cpu_fallback():
    import torch
    zc = np.linspace(0.0, 1.0, 9)
    with pytest.raises(binding.FseiError) as e:
        binding.Plan(10, 8, 8, 1.0, 1.0, zc)
    assert e.value.code == binding.ERR_SIZE
    with pytest.raises(binding.FseiError) as e:
        binding.Plan(8, 8, 8, -1.0, 1.0, zc)
    assert e.value.code == binding.ERR_GRID
    with pytest.raises(binding.FseiError) as e:
        binding.Plan(8, 8, 8, 1.0, 1.0, zc, 3, 0)
    assert e.value.code == binding.ERR_ARG
    with pytest.raises(binding.FseiError) as e:
        binding.Plan(8, 8, 8, 1.0, 1.0, zc[:5])
    assert e.value.code == binding.ERR_ARG
    if not torch.cuda.is_available():
        with pytest.raises(binding.FseiError) as e:       # valid arguments, no device: fails loudly
            binding.Plan(8, 8, 8, 1.0, 1.0, zc)
        assert e.value.code == binding.ERR_CUDA and "no CPU fallback" in str(e.value)


def test_product_does_not_touch_oracle():
    pkg = os.path.join(ROOT, "paper_2103_15187_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h", ".c")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(from|import)\s+oracle", r"liboracle", r"fsei_oracle", r"oracle/", r"oracle_[a-z]+\("):
                    assert not re.search(pat, src, flags=re.M), (dirpath, f, pat)
