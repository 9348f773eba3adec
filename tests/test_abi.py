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


def test_lane_plan_host_logic(lib):
    """Host logic of the opt-in two-lane split, through the C ABI without a device: the split
    point minimises 256-row tile blocks near batch / 2, the order is a permutation, and each lane is the stable
    descending sort of its robots by n_steps with the two lanes interleaved in proportion."""
    blocks = lambda b, H: (b * H + 255) // 256
    rng = np.random.default_rng(7)
    b0, order = rosa.rosa_debug_lane_plan(np.full(64, 10), 50)
    assert b0 == 30 and blocks(30, 50) + blocks(34, 50) == 13 == blocks(64, 50)   # BASELINE.json configs[2]: 6 + 7 row blocks
    assert sorted(order.tolist()) == list(range(64))
    for batch, H in [(2, 50), (3, 8), (12, 50), (64, 50), (256, 50), (37, 7), (512, 50)]:
        ns = rng.integers(1, 11, size=batch).astype(np.int32)
        b0, order = rosa.rosa_debug_lane_plan(ns, H)
        assert 1 <= b0 <= batch // 2 or (batch < 4 and b0 == batch // 2)
        cand = range(max(batch // 2 - batch // 4, 1), batch // 2 + 1)
        assert blocks(b0, H) + blocks(batch - b0, H) == min(blocks(c, H) + blocks(batch - c, H) for c in cand)
        assert sorted(order.tolist()) == list(range(batch))
        want = sorted(range(batch), key=lambda i: -int(ns[i]))                      # stable descending
        for lane in (order[:b0], order[b0:]):
            assert all(ns[a] >= ns[b] for a, b in zip(lane[:-1], lane[1:]))
            assert [i for i in want if i in set(lane.tolist())] == lane.tolist()    # a subsequence of the stable sort
        # dealt in proportion: after any prefix of the sorted robots the lanes hold their share to within one robot
        pos = {int(r): q for q, r in enumerate(want)}
        for q in range(1, batch + 1):
            in0 = sum(1 for r in order[:b0] if pos[int(r)] < q)
            assert abs(in0 - q * b0 / batch) < 1.0
    with pytest.raises(RuntimeError):
        rosa.rosa_debug_lane_plan(np.array([3], dtype=np.int32), 50)
