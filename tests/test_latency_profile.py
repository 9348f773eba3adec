"""Host logic of the latency-profile harness: the discrete-batch
worker simulation against closed forms, and the feasible-configuration rule.  CPU only."""
import numpy as np
import pytest

from paper_2607_01088_b200 import latency_profile as lp


def test_b1_underloaded_latency_is_service_time():
    arr = np.arange(50) * 0.010                      # one request every 10 ms, service 4 ms
    lat = lp.simulate_discrete_batching(arr, 1, lambda n: 0.004)
    assert np.allclose(lat, 0.004)


def test_b2_periodic_closed_form():
    T, S = 0.010, 0.003
    lat = lp.simulate_discrete_batching(np.arange(40) * T, 2, lambda n: S)
    assert np.allclose(lat[0::2], T + S) and np.allclose(lat[1::2], S)   # first waits for the second, then both run


def test_b1_overloaded_queue_grows_linearly():
    T, S = 0.002, 0.005                              # arrivals faster than service: D/D/1 backlog
    lat = lp.simulate_discrete_batching(np.arange(100) * T, 1, lambda n: S)
    assert np.allclose(lat, S + np.arange(100) * (S - T))


def test_partial_tail_and_flush():
    arr = np.array([0.0, 0.001, 0.002])
    lat = lp.simulate_discrete_batching(arr, 2, lambda n: 0.01)
    assert np.allclose(lat[:2], [0.011, 0.010]) and np.isnan(lat[2])       # third request never fills a batch
    lat = lp.simulate_discrete_batching(arr, 2, lambda n: 0.01 * n, flush_after=0.05)
    assert np.isclose(lat[2], 0.05 + 0.01)                                  # flushed alone after 50 ms


def test_utilisation_law_and_monotone_profile():
    pools = {1: [0.015], 8: [0.0165], 64: [0.031]}
    prof = lp.profile([1, 8, 64], pools, n_requests=4000, seed=3)
    for b, p in prof.items():
        assert np.isclose(p["max_throughput_per_s"], b / pools[b][0])
        p99 = [r["p99_ms"] for r in p["rates"]]
        if b == 1:
            assert p99[-1] > 3 * p99[2]              # the knee: queueing blows up towards 100% load
        else:
            assert p99[0] > p99[5]                   # strict full batches: at light load the fill time dominates
        assert min(r["p50_ms"] for r in p["rates"]) >= 1e3 * pools[b][0] - 1e-9   # never below one service time
    # batching trades latency at light load for throughput
    assert prof[64]["max_throughput_per_s"] > 25 * prof[1]["max_throughput_per_s"]
    assert prof[64]["rates"][0]["p50_ms"] > prof[1]["rates"][0]["p50_ms"]


def test_feasible_configs_rule():
    prof = {4: {"rates": [{"rate_per_s": 10.0 * j, "p99_ms": 20.0 + 20.0 * j} for j in range(1, 11)]}}
    conf = lp.feasible_configs(prof, freq_hz=5.0, slo_ms=120.0)
    ks = [c["robots"] for c in conf]
    assert ks == list(range(4, 11))                  # k f <= 50/s  <=>  p99 <= 120 ms ; k >= b
    assert [c for c in conf if c.get("best")][0]["robots"] == 10
    assert lp.feasible_configs(prof, freq_hz=5.0, slo_ms=30.0) == []


@pytest.mark.gpu
def test_profile_on_gpu_small():
    from paper_2607_01088_b200 import cases
    from paper_2607_01088_b200.runner import DeviceFleet
    mini = cases.ExpertConfig(layers=2, d_model=256, n_q_heads=8, n_kv_heads=1, head_dim=256, ffn=512,
                              horizon=50, action_dim=32)
    base = cases.build_case("lp", 4, mini, bf16=True, prefix_lens=[1], with_prefix=False)
    fl = DeviceFleet(base, [100] * 8, seed=1)
    pools = lp.measure_service_pool(fl, [1, 8], calls=5)
    fl.close()
    prof = lp.profile([1, 8], pools, n_requests=500)
    assert all(t > 0 for b in pools for t in pools[b])
    assert prof[8]["max_throughput_per_s"] > prof[1]["max_throughput_per_s"]


def test_bench_work_accounting_for_both_time_conditionings():
    """bench.py's algorithmic FLOPs / bytes: SURVEY 8(d) figures for the base path, and the variant's extra terms."""
    import importlib.util, os
    from dataclasses import replace
    from paper_2607_01088_b200 import cases
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(__file__), "..", "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    lens, ns = [816] * 64, [10] * 64
    fl = bench.class_flops(cases.PI0, lens, ns)
    tot = sum(v for k, v in fl.items() if k != "gemm_fused_o_gateup_down")
    assert abs(tot / 1e12 - 24.16) < 0.02       # 24.22 TFLOP per call, minus the hoisted per-token time half of W_1
    assert abs(bench.call_bytes(cases.PI0, lens, ns) / 1e9 - 15.92) < 0.05   # 10 x (629.36 MB + 64 x 15.04 MB)
    ada = replace(cases.PI0, time_conditioning=1)
    fa = bench.class_flops(ada, lens, ns)
    assert "gemm_embed" not in fa and fa["timevec"] == 2.0 * 640 * (2 * 1024 ** 2 + 37 * 3 * 1024 ** 2)
    assert fa["attention"] == fl["attention"] and fa["gemm_gateup_geglu"] == fl["gemm_gateup_geglu"]
    extra = bench.call_bytes(ada, lens, ns) - bench.call_bytes(cases.PI0, lens, ns)
    # parameters per step (2 B each): + 37 modulation matrices and biases, - the action half of W_1, - the 37 gain vectors
    assert abs(extra / 10 / 2 - (37 * (3 * 1024 ** 2 + 3 * 1024) - 1024 ** 2 - 37 * 1024)) < 1


def test_feasible_configs_does_not_extrapolate_flat_below_the_profiled_rates():
    """b = 16, 13.5 ms service, 16 robots at 1 Hz sits below the lowest profiled rate (10% of the maximum
    throughput); the discrete-batch worker's first request of a batch waits ~15 inter-arrival times there.  The
    feasible set must agree with the simulator on the same load: not feasible under a 200 ms deadline."""
    from paper_2607_01088_b200 import latency_profile as lp
    b, service = 16, 13.5e-3
    prof = lp.profile([b], {b: [service] * 8}, n_requests=1500, seed=1)
    lam = 16 * 1.0
    assert lam < prof[b]["rates"][0]["rate_per_s"]
    rng = np.random.default_rng(0)
    arr = lp.periodic_arrivals(16, 1.0, 1600, rng)
    lat = lp.simulate_discrete_batching(arr, b, lambda m: service)
    lat = lat[~np.isnan(lat)][200:]
    p99_sim = 1e3 * float(np.percentile(lat, 99))
    assert p99_sim > 200.0                                          # the simulator says: deadline missed
    conf = lp.feasible_configs(prof, 1.0, 200.0)
    assert not any(c["batch"] == b and c["robots"] == 16 for c in conf)
    # and where the bound applies it is within the simulator's percentile (a lower bound, not a guess)
    bound = prof[b]["service_ms_mean"] + 1e3 * (b - 1) / lam
    assert bound <= p99_sim * 1.05
