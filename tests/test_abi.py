"""The C-ABI library loads and exports every symbol include/*.h declares (CPU only; no compute), and the host
logic behind it that needs no device."""
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


def declared_symbols(header):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rosa_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["rosa.h", "rosa_debug.h"]
    for header, names in (("rosa.h", rosa.EXPORTS), ("rosa_debug.h", rosa.DEBUG_EXPORTS)):
        syms = declared_symbols(header)
        assert set(syms) == set(names), (header, syms, names)
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


def check_attn_plan(H, lens, n_cta):
    """Invariants of the stream-K split of the attention step (attn_tcgen05.cu): every key block of every item is
    covered exactly once; an item is whole or cut in two; the head segment (kb0 = 0) of a cut item is the LAST entry
    of its CTA's list and names the CTA of the continuation (the same tile's CTA of the next group: + tiles), where
    the continuation is the FIRST entry of the list (a CTA never waits for work queued behind something that
    waits); the tiles of a robot are cut at the same key block; nothing is shorter than 2 blocks unless the item is."""
    offs, segs = rosa.rosa_debug_attn_plan(H, lens, n_cta)
    tiles = (H + 15) // 16
    assert offs[0] == 0 and offs[-1] == len(segs) and np.all(np.diff(offs) >= 0)
    cta_of = np.repeat(np.arange(n_cta), np.diff(offs))
    cover = {}
    for i, (p, tt, kb0, kb1, n_part, part0) in enumerate(segs):
        nb = (lens[p] + 63) // 64 + 1
        assert 0 <= tt < tiles and 0 <= kb0 < kb1 <= nb
        cover.setdefault((p, tt), []).append((kb0, kb1, n_part, part0, cta_of[i], i))
    assert set(cover) == {(p, t) for p in range(len(lens)) for t in range(tiles)}
    loads = np.zeros(n_cta)
    for (p, tt), parts in cover.items():
        nb = (lens[p] + 63) // 64 + 1
        parts.sort()
        assert parts[0][0] == 0 and parts[-1][1] == nb
        for a, b in zip(parts, parts[1:]):
            assert a[1] == b[0]                                   # contiguous, no overlap
        head = parts[0]
        assert head[2] == len(parts) - 1 and len(parts) <= 2       # n_part of the head = number of continuations (at most one)
        if len(parts) > 1:
            assert head[5] == offs[head[4] + 1] - 1               # the head ends its CTA's list
            assert head[3] == head[4] + tiles                     # the continuation: same tile, next group of CTAs
            c = parts[1]
            assert c[2] == -1 and c[4] == head[3] and c[5] == offs[c[4]]              # first entry of that CTA
            assert parts[0][1] == cover[(p, 0)][0][1]             # every tile of the robot is cut at the same block
            assert all(b - a >= 2 for a, b, *_ in parts)
        for a, b, _, _, cta, _ in parts:
            loads[cta] += b - a + 6.0
    return loads


def test_attn_plan_host_logic(lib):
    """Host logic of the attention work split through the C ABI without a device (pins: brute-force invariants
    above; balance: the busiest CTA is within 25% of the equal share, whichever of the two plans - items cut into
    per-CTA shares, or whole items longest-first - the planner kept)."""
    rng = np.random.default_rng(3)
    # cfg2-like fleet on 148 CTAs: shares are balanced to within a few blocks
    lens = rng.integers(600, 1001, size=64)
    loads = check_attn_plan(50, lens, 148)
    assert np.count_nonzero(loads) == 148
    assert loads.max() <= 1.25 * loads.sum() / 148, (loads.max(), loads.sum() / 148)
    # one robot: the four items are cut so that several CTAs share each key stream
    loads = check_attn_plan(50, [816], 148)
    assert np.count_nonzero(loads) >= 6
    # degenerate and ragged cases, few CTAs, L = 0
    for lens, n_cta, H in (([0], 148, 50), ([0, 1, 63, 64, 65], 7, 50), ([5000], 3, 8), (list(rng.integers(0, 1300, size=256)), 148, 50),
                           ([816] * 512, 148, 50), ([100, 100], 1, 50), ([1200] * 3, 148, 64)):
        check_attn_plan(H, np.asarray(lens), n_cta)
    with pytest.raises(rosa.RosaError):
        rosa.rosa_debug_attn_plan(0, [1], 4)
