"""Pins for the homogeneous scheduler: Eq. 3 ILP against brute-force enumeration,
Eq. 4 closed form, and the whole binary search against a closed form on a flat latency profile.  CPU only."""
import itertools

import numpy as np

from paper_2607_01088_b200 import scheduler as sch


def flat_profile(latency_ms, mu):
    """Latency independent of load up to the capacity mu (requests/s) of one server."""
    rates = [{"rate_per_s": mu * j / 10, "p99_ms": latency_ms, "mean_ms": latency_ms} for j in range(1, 11)]
    return {1: {"rates": rates}}


def test_closed_loop_rate_eq4():
    assert np.isclose(sch.closed_loop_rate(0.2, 0.05), 4.0)
    assert np.isclose(sch.closed_loop_rate(0.2, 0.05, 0.5, 10), 1.0 / 0.3)


def test_ilp_matches_brute_force():
    rng = np.random.default_rng(0)
    for trial in range(20):
        configs = [{"batch": 1, "robots": int(k), "mean_ms": float(rng.uniform(10, 100))}
                   for k in rng.choice(np.arange(1, 9), size=4, replace=False)]
        R, S = int(rng.integers(3, 20)), int(rng.integers(1, 5))
        best = None
        for y in itertools.product(range(S + 1), repeat=len(configs)):
            if sum(y) <= S and sum(n * c["robots"] for n, c in zip(y, configs)) == R:
                cost = sum(y) + 1e-4 * sum(n * c["robots"] * c["mean_ms"] for n, c in zip(y, configs)) / R
                if best is None or cost < best[0] - 1e-12:
                    best = (cost, y)
        got = sch.pack_configurations_ilp(configs, R, S)
        if best is None:
            assert got is None
        else:
            assert got is not None and sum(got) <= S
            assert sum(n * c["robots"] for n, c in zip(got, configs)) == R
            cost = sum(got) + 1e-4 * sum(n * c["robots"] * c["mean_ms"] for n, c in zip(got, configs)) / R
            assert abs(cost - best[0]) <= 1e-9


def test_schedule_closed_form_on_flat_profile():
    # latency 50 ms whatever the load, capacity 40 req/s per server, t_act = 200 ms:
    # f* = min( 1/(0.2 + 0.05) = 4 Hz  (Eq. 4),  S mu / R  (capacity) )
    prof = flat_profile(50.0, 40.0)
    r = sch.schedule_homogeneous(prof, n_robots=16, n_servers=4, t_act=0.2, slo_ms=200.0)
    assert abs(r["f"] - 4.0) <= 0.02 and r["servers_used"] <= 4
    r = sch.schedule_homogeneous(prof, n_robots=64, n_servers=4, t_act=0.2, slo_ms=200.0)
    assert abs(r["f"] - 4 * 40.0 / 64) <= 0.05                      # capacity-bound: 2.5 Hz
    assert sum(a["robots"] * a["servers"] for a in r["assignment"]) == 64
    assert sch.schedule_homogeneous(prof, n_robots=16, n_servers=4, t_act=0.2, slo_ms=20.0) is None   # SLO never met


def test_more_servers_never_hurt():
    prof = flat_profile(30.0, 25.0)
    fs = [sch.schedule_homogeneous(prof, 48, s, 0.1, 200.0)["f"] for s in (2, 4, 8, 16)]
    assert all(b >= a - 0.02 for a, b in zip(fs, fs[1:]))
