"""Closed-loop fleet simulator pins on CPU, and the continuous
batcher against one-shot calls on the GPU (step composition, pin P6)."""
import numpy as np
import pytest

from paper_2607_01088_b200 import batcher as bt


def test_closed_loop_unsaturated_rate_is_eq4():
    # 4 robots, b = 1, service 10 ms, t_act 190 ms: each robot cycles in 200 ms + queueing (none when desynchronised)
    r = bt.closed_loop_fleet(4, 0.19, None, 60.0, 0.2, "discrete", 1, lambda b: 0.010)
    assert abs(r["actions_per_s"] - 4 / 0.2) / (4 / 0.2) < 0.03
    assert r["p50_ms"] >= 10.0 - 1e-6 and r["slo_meet_rate"] == 1.0


def test_closed_loop_saturated_is_service_bound():
    # 50 robots, b = 1, service 10 ms, t_act 50 ms: the worker saturates at 100 actions/s; latency = queue of ~45
    r = bt.closed_loop_fleet(50, 0.05, None, 60.0, 0.2, "discrete", 1, lambda b: 0.010)
    assert abs(r["actions_per_s"] - 100.0) < 2.0
    assert r["qualified_actions_per_s"] < 5.0            # ~450 ms latency: nothing meets a 200 ms SLO


def test_rate_cap_restores_slo():
    # same fleet capped at 1.5 Hz per robot: load 75/s < 100/s, latency drops under the SLO
    r = bt.closed_loop_fleet(50, 0.05, 1.5, 120.0, 0.2, "discrete", 1, lambda b: 0.010)
    assert abs(r["actions_per_s"] - 75.0) < 2.0 and r["slo_meet_rate"] > 0.99


def test_discrete_batching_raises_capacity():
    call = lambda b: 0.015 + 0.00025 * b                  # measured shape: almost flat in b
    r1 = bt.closed_loop_fleet(64, 0.2, None, 60.0, 0.2, "discrete", 1, call)
    r16 = bt.closed_loop_fleet(64, 0.2, None, 60.0, 0.2, "discrete", 16, call)
    assert r16["actions_per_s"] > 2.5 * r1["actions_per_s"]


def test_continuous_mode_conserves_work():
    # 8 robots, launches of 2 ms, 10 steps per chunk, t_act 30 ms: cycle = 20 ms + 30 ms
    r = bt.closed_loop_fleet(8, 0.03, None, 30.0, 0.2, "continuous", 8, None, step_time=lambda m: 0.002)
    assert abs(r["actions_per_s"] - 8 / 0.05) / 160.0 < 0.08


@pytest.mark.gpu
def test_continuous_batcher_matches_one_shot_calls():
    import torch
    from paper_2607_01088_b200 import binding as rosa, cases
    from paper_2607_01088_b200.runner import LoadedCase
    mini = cases.ExpertConfig(layers=2, d_model=256, n_q_heads=8, n_kv_heads=1, head_dim=256, ffn=512,
                              horizon=50, action_dim=32)
    case = cases.build_case("cb", 31, mini, bf16=True, prefix_lens=[70, 150, 33, 90, 64, 200], n_steps=10)
    lc = LoadedCase(case)
    want, _ = lc.run()                                     # one 10-step call for all six robots
    cb = bt.ContinuousBatcher(lc.expert, 50, 32, max_batch=4, n_steps=10)
    noise = torch.from_numpy(case.noise).cuda()
    pending, got, launches = list(range(6)), {}, 0
    while pending or len(cb):
        while pending and len(cb) < 4 and (launches % 3 == 0 or len(cb) == 0):   # staggered admissions
            r = pending.pop(0)
            cb.admit(r, noise[r])
        for r, x in cb.step():
            got[r] = x.cpu().numpy()
        launches += 1
    torch.cuda.synchronize()
    assert sorted(got) == list(range(6)) and launches > 10
    for r in range(6):
        assert np.abs(got[r] - want[r]).max() <= 2e-3, r   # step composition (P6): same chunk, rounding noise only
    lc.close()
