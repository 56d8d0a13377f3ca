"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/reann.h declares; the product path fails loudly without a device (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

import gen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def R():
    import __graft_entry__ as ge
    ge.build()
    import paper_2505_06711_b200 as R
    return R


def test_header_symbols_are_exported(R):
    hdr = open(os.path.join(ROOT, "include", "reann.h")).read()
    declared = set(re.findall(r"\b(reann_[a-z_]+)\s*\(", hdr))
    assert declared == set(R.EXPORTS)
    L = R.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2505_06711_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "reann_oracle" not in txt, f


def test_no_device_is_a_loud_error(R):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    cfg = gen.make_config(0)
    with pytest.raises(R.ReannError) as ei:
        R.Reann.from_config(cfg)
    assert ei.value.code == R.REANN_ERR_CUDA


def test_argument_validation_without_device(R):
    with pytest.raises(R.ReannError) as ei:
        R.reann_create(b"", np.zeros(1, dtype=np.int32), -1.0, 1.0, 1, 1, 4)
    assert ei.value.code == R.REANN_ERR_ARG
