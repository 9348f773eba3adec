"""serving.py against the real library for a few seconds of real time: the measured open-loop latency agrees with the
virtual-time simulator fed with the measured service time, and closed-loop fleets are served by the discrete and the
continuous worker with consistent SLO accounting."""
import numpy as np
import pytest

from paper_2607_01088_b200 import build as rosa_build
from paper_2607_01088_b200 import binding as rosa
from paper_2607_01088_b200 import cases
from paper_2607_01088_b200 import serving as sv

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fleet():
    from paper_2607_01088_b200.runner import DeviceFleet
    rosa_build.build()
    rosa.load()
    base = cases.make_case(4, batch=1, with_prefix=False)
    fl = DeviceFleet(base, [816] * 16, seed=4)
    yield fl
    fl.close()


def test_measured_latency_profile_agrees_with_the_simulator(fleet):
    prof = sv.measure_latency_profile(fleet, [4], slo_s=0.2, seconds_per_point=1.2, fractions=(0.3, 0.7))
    p = prof[4]
    assert 5.0 <= p["service_ms_mean"] <= 40.0                       # one 10-step call of 4 robots on a B200
    for row in p["rates"]:
        assert row["unserved"] == 0 and row["requests"] >= 20
        assert row["p50_ms"] >= 0.9 * p["service_ms_mean"]           # nobody is served faster than one call
        # real time against virtual time on the same arrivals: same queueing, plus host jitter
        assert abs(row["mean_ms"] - row["sim_mean_ms"]) <= 0.25 * row["sim_mean_ms"] + 3.0, row
        assert row["p99_ms"] <= 2.0 * row["sim_p99_ms"] + 10.0, row
    lo, hi = p["rates"]
    assert hi["worker_busy_frac"] > lo["worker_busy_frac"]           # more load, busier worker (~0.3 and ~0.7)
    assert abs(hi["worker_busy_frac"] - 0.7) <= 0.2


def test_closed_loop_fleets_discrete_and_continuous(fleet):
    slo = 0.2
    w = sv.Worker(8, sv.gpu_batch_call(fleet), n_clients=16).start()
    disc = sv.closed_loop(w, 16, t_act=0.05, rate_cap_hz=None, duration_s=2.0, slo_s=slo)
    w.stop()
    w = sv.continuous_worker(fleet, 16).start()
    cont = sv.closed_loop(w, 16, t_act=0.05, rate_cap_hz=None, duration_s=2.0, slo_s=slo)
    w.stop()
    w = sv.continuous_worker(fleet, 16).start()
    capped = sv.closed_loop(w, 16, t_act=0.05, rate_cap_hz=2.0, duration_s=2.0, slo_s=slo)
    w.stop()
    for r in (disc, cont, capped):
        assert r["requests"] > 0 and np.isfinite(r["p99_ms"])
        assert r["qualified_actions_per_s"] <= r["actions_per_s"] + 1e-9
        assert abs(r["qualified_actions_per_s"] - r["slo_meet_rate"] * r["actions_per_s"]) <= 1e-6 * max(1.0, r["actions_per_s"])
    # closed-loop bound of Eq. 4: a robot cannot send faster than 1 / (t_act + latency)
    for r in (disc, cont):
        assert r["actions_per_s"] <= 16 / (0.05 + 1e-3 * r["p50_ms"]) * 1.25 + 1.0
    # request-rate control: 16 robots capped at 2 Hz send 32 requests/s, whatever the worker could do
    assert abs(capped["actions_per_s"] - 32.0) <= 6.0
    assert capped["p99_ms"] <= cont["p99_ms"] + 5.0                  # a lighter load is not served slower
