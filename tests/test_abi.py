"""The C-ABI library loads and exports every symbol include/rosa.h declares (CPU only; no compute)."""
import os
import re

import numpy as np
import pytest

from paper_2607_01088_b200 import binding as rosa
from paper_2607_01088_b200 import build as rosa_build
from paper_2607_01088_b200 import cases

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    rosa_build.build()
    return rosa.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rosa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rosa_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    syms = declared_symbols()
    assert set(syms) == set(rosa.EXPORTS), (syms, rosa.EXPORTS)
    for s in syms:
        assert hasattr(lib, s), s
    assert rosa.rosa_version() >= 1
    assert isinstance(rosa.rosa_last_error(), str)


def test_config_struct_layout_matches_header():
    text = open(os.path.join(ROOT, "include", "rosa.h")).read()
    body = text[text.index("typedef struct {", text.index("rosa_dtype_t;")):text.index("} rosa_expert_config_t;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = [n for decl in re.findall(r"(?:int32_t|float)\s+([^;]+);", body) for n in re.split(r"\s*,\s*", decl.strip())]
    assert names == [f[0] for f in rosa.rosa_expert_config_t._fields_]


def test_argument_validation_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("validation-without-device case is for the CPU box")
    c = cases.make_case(0)
    with pytest.raises(rosa.RosaError) as ei:
        rosa.rosa_expert_create(c.cfg.as_dict(), c.weights, max_robots=2, max_batch=2, max_prefix_len=64)
    assert ei.value.status == rosa.ROSA_ERR_CUDA          # no CPU fallback: fails loudly
    bad = dict(c.cfg.as_dict(), d_model=100)
    with pytest.raises(rosa.RosaError) as ei:
        rosa.rosa_expert_create(bad, c.weights, max_robots=2, max_batch=2, max_prefix_len=64)
    assert ei.value.status == rosa.ROSA_ERR_UNSUPPORTED
