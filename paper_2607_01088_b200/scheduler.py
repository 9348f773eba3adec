"""Homogeneous-fleet scheduler for the action-only pipeline.

The paper's algorithm for a fleet whose only goal-coupled model is System 1
(pipeline P1, Table 1): binary search on the shared action rate f; for each candidate f build the
feasible per-server configurations P(f) from the measured latency profile (step 2.1, PAPER.md:352;
`latency_profile.feasible_configs`), pack them onto the servers with the ILP of Eq. 3 (PAPER.md:356:
sum_p y_p <= |S|, sum_p y_p a_p = |R|, y_p non-negative integers; tie-break cost = servers used, then
measured latency), and accept f if the closed-loop bound of Eq. 4 holds (PAPER.md:362:
f <= 1 / (t_act + l_S1 + l_S2 / H)).  Obligation models (step 1) and System 2 are outside this
build (their models are not); with no System 2, l_S2 = 0.  CPU only: scipy's MILP solver stands in for
OR-Tools.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

import numpy as np
from scipy.optimize import Bounds, LinearConstraint, milp

from .latency_profile import feasible_configs


def closed_loop_rate(t_act: float, l_s1: float, l_s2: float = 0.0, horizon: int = 1) -> float:
    """Eq. 4, seconds in, Hz out."""
    return 1.0 / (t_act + l_s1 + l_s2 / horizon)


def pack_configurations_ilp(configs: Sequence[dict], n_robots: int, n_servers: int, latency_weight: float = 1e-4
                            ) -> Optional[List[int]]:
    """Eq. 3 for one goal-coupled model: y_p servers run configuration p, which serves
    a_p = configs[p]["robots"] robot streams.  Minimises (servers used) + latency_weight * (robot-weighted
    mean latency in ms); returns y or None if infeasible."""
    if not configs:
        return None
    a = np.array([c["robots"] for c in configs], dtype=float)
    cost = 1.0 + latency_weight * a * np.array([c.get("mean_ms", 0.0) for c in configs]) / max(1, n_robots)
    cons = [LinearConstraint(np.ones((1, len(a))), -np.inf, n_servers), LinearConstraint(a[None, :], n_robots, n_robots)]
    res = milp(cost, constraints=cons, integrality=np.ones(len(a)), bounds=Bounds(0, n_servers))
    if not res.success:
        return None
    return [int(round(v)) for v in res.x]


def schedule_homogeneous(profile: Dict[int, dict], n_robots: int, n_servers: int, t_act: float, slo_ms: float,
                         eps: float = 1e-2, percentile: str = "p99_ms") -> Optional[dict]:
    """PAPER.md:320-339 with G = {System 1}.  Returns {"f": Hz, "assignment": [{batch, robots, servers}], ...}
    for the largest feasible shared action rate (within eps Hz), or None if even f -> 0 is infeasible."""
    lo, hi, best = 0.0, 1.0 / t_act, None            # f_max assumes zero inference latency
    while hi - lo > eps:
        f = 0.5 * (lo + hi)
        configs = feasible_configs(profile, f, slo_ms, percentile)
        y = pack_configurations_ilp(configs, n_robots, n_servers)
        ok = False
        if y is not None:
            used = [(c, n) for c, n in zip(configs, y) if n > 0]
            l_s1 = sum(c["mean_ms"] * c["robots"] * n for c, n in used) / n_robots * 1e-3
            if f <= closed_loop_rate(t_act, l_s1):
                ok = True
                best = {"f": f, "servers_used": int(sum(y)), "mean_latency_ms": 1e3 * l_s1, "actions_per_s": f * n_robots,
                        "assignment": [{"batch": c["batch"], "robots": c["robots"], "servers": n} for c, n in used]}
        if ok:
            lo = f
        else:
            hi = f
    return best
