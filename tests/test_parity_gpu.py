"""GPU parity: rosa_denoise_batch* (through the C ABI) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star (3):
final actions max-abs <= 2e-2 and rel-L2 <= 1e-2; per-step velocity rel-L2 <= 5e-3."""
import numpy as np
import pytest
import torch

from oracle import rosa_oracle as O
from paper_2607_01088_b200 import binding as rosa
from paper_2607_01088_b200 import build as rosa_build
from paper_2607_01088_b200 import cases
from paper_2607_01088_b200.runner import LoadedCase, rel_l2

pytestmark = pytest.mark.gpu

TOL_ACT_ABS, TOL_ACT_REL, TOL_VEL_REL = 2e-2, 1e-2, 5e-3


@pytest.fixture(scope="module", autouse=True)
def _built():
    rosa_build.build()
    rosa.load()


def check_against_oracle(case, lc, robots, label):
    """Run the listed robots as ONE batch on the GPU; oracle on the same robots."""
    got_x, got_v = lc.run(robots=robots, want_velocity=True)
    want_x, want_v = O.denoise_case(case, robots=robots, return_velocity=True)
    assert np.all(np.isfinite(got_x)), label
    err_abs = float(np.abs(got_x - want_x).max())
    err_rel = rel_l2(got_x, want_x)
    vel_rel = [rel_l2(got_v[k], want_v[k]) for k in range(len(want_v))]
    print(f"[{label}] actions max-abs {err_abs:.3e} rel-L2 {err_rel:.3e}; velocity rel-L2 max {max(vel_rel):.3e}")
    assert err_abs <= TOL_ACT_ABS, (label, err_abs)
    assert err_rel <= TOL_ACT_REL, (label, err_rel)
    assert max(vel_rel) <= TOL_VEL_REL, (label, vel_rel)
    return got_x


def test_cfg0_tiny_fp32():
    case = cases.make_case(0)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, [0, 1], "cfg0")
    lc.close()


def test_cfg1_pi0_b8():
    case = cases.make_case(1)
    lc = LoadedCase(case)
    check_against_oracle(case, lc, list(range(8)), "cfg1")
    lc.close()
