"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol include/nnp.h
declares; without a CUDA device the compute entry points fail loudly (no fallback)."""
import os
import re

import numpy as np
import pytest

import gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nnp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nnp_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported():
    from paper_2604_21441_b200 import build, binding
    build.build()
    L = binding.lib()
    syms = declared_symbols()
    assert len(syms) >= 15
    for s in syms:
        assert hasattr(L, s), f"{s} declared in nnp.h but not exported"
    assert set(binding.EXPORTS) == set(syms)


def test_strerror_and_no_device_failure():
    import torch
    import paper_2604_21441_b200 as nnp
    assert nnp.nnp_strerror(0) == "ok"
    assert "box" in nnp.nnp_strerror(-3)
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    cfg = gen.get_config(0)
    with pytest.raises(nnp.NNPError) as e:
        nnp.Model(cfg["aev"], cfg["nets"])
    assert e.value.code == -6  # NNP_ERR_CUDA: no CPU fallback


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2604_21441_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "nnp_oracle" not in txt, f
