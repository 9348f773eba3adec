"""The real-time request queue / worker / client drivers (paper_2607_01088_b200/serving.py) on CPU: the batch call is
a sleep of known length, so the measured latencies and rates have closed forms (D/D/1 with batch forming, the
closed-loop cycle of PAPER.md Eq. 4, request-rate control) and must also agree with the virtual-time simulator of
latency_profile.py on the same arrivals.  Real time: tolerances allow for a few milliseconds of scheduling jitter."""
import time

import numpy as np

from paper_2607_01088_b200 import latency_profile as lp
from paper_2607_01088_b200 import serving as sv

JIT = 12.0   # ms: generous on purpose (a loaded test box); a logic error moves these numbers by 2x, not by milliseconds


def sleeper(service_s, log=None):
    def run(robots):
        assert len(set(robots)) == len(robots)          # a batch never carries a robot twice
        if log is not None:
            log.append(len(robots))
        time.sleep(service_s)
    return run


def test_open_loop_discrete_batches_match_closed_form_and_simulator():
    # service 20 ms per call, b = 2, one arrival every 20 ms (50% of mu = 100 req/s): a batch forms every 40 ms; its
    # first request waits 20 ms for the second, then both are served: latencies 40 ms and 20 ms, alternating
    s, b = 0.020, 2
    arr = 0.020 * np.arange(1, 61)
    sizes = []
    w = sv.Worker(b, sleeper(s, sizes)).start()
    res = sv.open_loop(w, arr, n_robots=4, slo_s=0.035)
    w.stop()
    assert res["unserved"] == 0 and set(sizes) == {2} and w.calls == 30
    sim = lp.simulate_discrete_batching(arr, b, lambda m: s)
    assert abs(res["mean_ms"] - 30.0) <= JIT and abs(res["mean_ms"] - 1e3 * sim[6:].mean()) <= JIT
    # (p99 of ~55 requests is their maximum: one scheduling hiccup of the test box lands there, so it only gets an upper bound)
    assert 40.0 - JIT <= res["p99_ms"] <= 40.0 + 30.0 and abs(res["p50_ms"] - 30.0) <= 10.0 + JIT
    assert 0.25 <= res["slo_meet_rate"] <= 0.75                 # the 20 ms half meets a 35 ms deadline, the 40 ms half does not
    assert abs(res["actions_per_s"] - 50.0) <= 8.0
    assert abs(res["qualified_actions_per_s"] - 25.0) <= 10.0


def test_open_loop_flush_serves_partial_batches():
    # b = 4 but only three requests, 5 ms apart: without a flush nothing is ever served; with flush_after = 30 ms the
    # partial batch starts 30 ms after the first arrival
    arr = np.array([0.005, 0.010, 0.015])
    sizes = []
    w = sv.Worker(4, sleeper(0.010, sizes), flush_after=0.030).start()
    res = sv.open_loop(w, arr, n_robots=4, slo_s=1.0, warm_frac=0.0, drain_s=1.0)
    w.stop()
    assert sizes == [3] and res["unserved"] == 0
    assert 40.0 - JIT <= res["p99_ms"] <= 40.0 + 30.0            # first request: 30 ms flush + 10 ms service


def test_closed_loop_cycle_and_rate_cap():
    # 4 robots, one worker with b = 4 that starts when all four wait: every cycle is service + t_act = 10 + 30 ms
    # (Eq. 4's closed-loop bound 1 / (t_act + l) per robot): 4 / 0.04 = 100 actions/s, latency = the service time
    w = sv.Worker(4, sleeper(0.010), n_clients=4).start()
    res = sv.closed_loop(w, 4, t_act=0.030, rate_cap_hz=None, duration_s=1.2, slo_s=0.015)
    w.stop()
    assert abs(res["actions_per_s"] - 100.0) <= 25.0
    assert res["p50_ms"] <= 10.0 + JIT and res["slo_meet_rate"] >= 0.5
    # request-rate control: capped at 10 Hz per robot the fleet sends 40 requests/s however fast the worker is
    w = sv.Worker(4, sleeper(0.010), n_clients=4).start()
    res = sv.closed_loop(w, 4, t_act=0.030, rate_cap_hz=10.0, duration_s=1.2, slo_s=0.015)
    w.stop()
    assert abs(res["actions_per_s"] - 40.0) <= 10.0


class FakeStepper:
    """Continuous batching without a device: every step advances all in-flight robots by one of n_steps."""
    def __init__(self, n_steps, step_s):
        self.n_steps, self.step_s, self.left, self.sizes = n_steps, step_s, {}, []

    def admit(self, robot, noise):
        assert robot not in self.left
        self.left[robot] = self.n_steps

    def step(self):
        self.sizes.append(len(self.left))
        time.sleep(self.step_s)
        for r in self.left:
            self.left[r] -= 1
        fin = [(r, None) for r, k in self.left.items() if k == 0]
        for r, _ in fin:
            del self.left[r]
        return fin

    def __len__(self):
        return len(self.left)


def test_continuous_worker_admits_at_step_boundaries():
    # 5 steps of 4 ms per chunk; a request that arrives mid-step joins at the next boundary: latency in [20, 24] ms + jitter,
    # and requests that overlap in time share launches (some steps carry more than one robot)
    st = FakeStepper(5, 0.004)
    w = sv.Worker(8, stepper=st, sync=lambda: None, noise_of=lambda r: None).start()
    arr = 0.007 * np.arange(1, 41)
    res = sv.open_loop(w, arr, n_robots=16, slo_s=0.040, warm_frac=0.0)
    w.stop()
    assert res["unserved"] == 0 and res["requests"] == 40
    assert 20.0 - 1.0 <= res["p50_ms"] <= 24.0 + JIT and res["p99_ms"] <= 24.0 + 30.0
    assert max(st.sizes) >= 3 and res["slo_meet_rate"] >= 0.7


def test_summarize_counts_only_the_window():
    done = [sv.Request(0.0, 0, 0.010), sv.Request(1.0, 1, 1.050), sv.Request(2.0, 2, 2.300)]
    r = sv.summarize(done, 0.5, 3.0, slo_s=0.1)
    assert r["requests"] == 2 and abs(r["actions_per_s"] - 0.8) < 1e-9 and abs(r["qualified_actions_per_s"] - 0.4) < 1e-9
    assert abs(r["slo_meet_rate"] - 0.5) < 1e-9 and sv.summarize([], 0, 1, 0.1)["requests"] == 0
