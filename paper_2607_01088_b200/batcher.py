"""Request batchers in front of the library and a closed-loop fleet driver.

* `ContinuousBatcher` — iteration-level continuous batching of the action expert (BASELINE.json
  configs[3]; the paper describes continuous batching only for its autoregressive models):
  every `step()` is ONE `rosa_denoise_batch_ex` launch that advances all in-flight robots by one Euler
  step at their own (t_i, dt_i); robots are admitted and retired at step boundaries.  By the
  step-composition property (pin P6) a robot's chunk equals the one-shot N-step call.
* `closed_loop_fleet` — the paper's client model: a robot sends a request, waits
  for its chunk, executes for t_act, and sends the next one, never faster than the scheduled rate f
  (request-rate control).  The worker is either the discrete-batch worker of `latency_profile` or the
  continuous batcher.  Runs in virtual time with service durations measured on the GPU; reports raw
  and SLO-qualified actions/s and latency percentiles.

Only argument marshalling and device-row bookkeeping (torch indexing) happen here; every step of the
method runs in the library's kernels.
"""
from __future__ import annotations

from typing import Callable, Dict, List, Optional, Sequence, Tuple

import numpy as np


class ContinuousBatcher:
    """In-flight set of robots advanced one Euler step per launch."""

    def __init__(self, expert, horizon: int, action_dim: int, max_batch: int, n_steps: int = 10, device="cuda:0",
                 stream=None):
        import torch
        self.torch, self.expert, self.n_steps, self.max_batch = torch, expert, n_steps, max_batch
        self.stream = stream
        self.x = torch.empty((max_batch, horizon, action_dim), dtype=torch.float32, device=device)
        self.out = torch.empty_like(self.x)
        self.robots: List[int] = []          # robot id of row i of self.x
        self.done_steps: List[int] = []      # Euler steps already taken

    def __len__(self):
        return len(self.robots)

    def admit(self, robot: int, noise) -> None:
        """Add a robot at t = 1 with its initial noise (device tensor [H, A]) at the next step boundary."""
        assert len(self.robots) < self.max_batch and robot not in self.robots
        self.x[len(self.robots)].copy_(noise)
        self.robots.append(robot)
        self.done_steps.append(0)

    def step(self) -> List[Tuple[int, "object"]]:
        """One launch: every in-flight robot takes one Euler step.  Returns [(robot, actions tensor)] of the
        robots that finished; their rows are compacted away."""
        from . import binding as rosa
        n = len(self.robots)
        if n == 0:
            return []
        N = self.n_steps
        ids = np.asarray(self.robots, dtype=np.int32)
        t0 = np.asarray([1.0 - k / N for k in self.done_steps], dtype=np.float32)
        dt = np.full(n, -1.0 / N, dtype=np.float32)
        ns = np.ones(n, dtype=np.int32)
        rosa.rosa_denoise_batch_ex(self.expert, ids, self.x[:n], t0, dt, ns, self.out[:n], None, self.stream)
        self.x, self.out = self.out, self.x
        self.done_steps = [k + 1 for k in self.done_steps]
        finished = [i for i, k in enumerate(self.done_steps) if k >= N]
        res = [(self.robots[i], self.x[i].clone()) for i in finished]
        if finished:
            keep = [i for i in range(n) if i not in set(finished)]
            if keep:
                idx = self.torch.as_tensor(keep, device=self.x.device)
                self.out[:len(keep)].copy_(self.x.index_select(0, idx))
                self.x, self.out = self.out, self.x
            self.robots = [self.robots[i] for i in keep]
            self.done_steps = [self.done_steps[i] for i in keep]
        return res


# ------------------------------------------------------------------ closed-loop fleet in virtual time
def closed_loop_fleet(n_robots: int, t_act: float, rate_cap_hz: Optional[float], horizon_s: float, slo_s: float,
                      mode: str, batch: int, call_time: Callable[[int], float], step_time: Optional[Callable[[int], float]] = None,
                      n_steps: int = 10, seed: int = 0) -> Dict[str, float]:
    """Simulate `n_robots` closed-loop clients against one GPU worker for `horizon_s` seconds.

    mode "discrete": the worker starts a batch when `batch` requests wait (or all robots are waiting) and it is
    idle; the call takes `call_time(b)`.  mode "continuous": waiting requests are admitted at every Euler-step
    boundary (up to `batch` in flight); a launch with m robots in flight takes `step_time(m)`; a chunk needs
    `n_steps` launches.  A robot's next request is sent at max(completion + t_act, last send + 1 / rate_cap).
    Returns raw and SLO-qualified actions/s and latency percentiles (requests completed after a 10% warm-up)."""
    rng = np.random.default_rng(seed)
    period = 0.0 if not rate_cap_hz else 1.0 / rate_cap_hz
    next_send = rng.uniform(0.0, max(t_act, period), size=n_robots)   # desynchronised start over one robot cycle
    last_send = np.full(n_robots, -1e9)
    waiting: List[Tuple[float, int]] = []                      # (send time, robot)
    lat: List[Tuple[float, float]] = []                        # (completion time, latency)
    inflight: List[List] = []                                  # continuous: [robot, send time, steps done]
    t = 0.0

    def collect(now):
        for r in np.nonzero(next_send <= now)[0]:
            waiting.append((float(next_send[r]), int(r)))
            last_send[r] = next_send[r]
            next_send[r] = np.inf
        waiting.sort()

    def complete(r, sent, now):
        lat.append((now, now - sent))
        next_send[r] = max(now + t_act, last_send[r] + period)

    while t < horizon_s:
        collect(t)
        if mode == "discrete":
            if waiting and (len(waiting) >= batch or len(waiting) == n_robots):   # a full batch, or everyone is waiting
                take = waiting[:batch]
                del waiting[:batch]
                t_done = t + call_time(len(take))
                for sent, r in take:
                    complete(r, sent, t_done)
                t = t_done
                continue
        else:
            while waiting and len(inflight) < batch:
                sent, r = waiting.pop(0)
                inflight.append([r, sent, 0])
            if inflight:
                t += step_time(len(inflight))
                for it in inflight:
                    it[2] += 1
                for it in [it for it in inflight if it[2] >= n_steps]:
                    complete(it[0], it[1], t)
                inflight = [it for it in inflight if it[2] < n_steps]
                continue
        nxt = next_send[np.isfinite(next_send)]
        if nxt.size == 0:
            break
        t = max(t, float(nxt.min()))
    done = [(c, l) for c, l in lat if c >= 0.1 * horizon_s and c <= horizon_s]
    if not done:
        return {"actions_per_s": 0.0, "qualified_actions_per_s": 0.0, "p50_ms": float("nan"), "p99_ms": float("nan")}
    ls = np.array([l for _, l in done])
    span = 0.9 * horizon_s
    return {"actions_per_s": len(ls) / span, "qualified_actions_per_s": float((ls <= slo_s).sum()) / span,
            "p50_ms": 1e3 * float(np.percentile(ls, 50)), "p99_ms": 1e3 * float(np.percentile(ls, 99)),
            "slo_meet_rate": float((ls <= slo_s).mean())}


# ------------------------------------------------------------------ measured on the GPU
def measure_step_times(fleet, sizes: Sequence[int], calls: int = 10) -> Dict[int, float]:
    """Mean duration (s) of ONE-Euler-step launches (`n_steps = 1`) with m robots in flight."""
    import torch
    from . import binding as rosa
    stream = torch.cuda.Stream(device=fleet.device)
    out: Dict[int, float] = {}
    with torch.cuda.stream(stream):
        for m in sizes:
            ids = np.arange(m, dtype=np.int32)
            x = fleet.noise[:m].contiguous()
            y = torch.empty_like(x)
            t0 = np.full(m, 0.5, dtype=np.float32)
            dt = np.full(m, -0.1, dtype=np.float32)
            ns = np.ones(m, dtype=np.int32)
            for _ in range(3):
                rosa.rosa_denoise_batch_ex(fleet.expert, ids, x, t0, dt, ns, y, None, stream)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(calls):
                rosa.rosa_denoise_batch_ex(fleet.expert, ids, x, t0, dt, ns, y, None, stream)
            e1.record(stream)
            stream.synchronize()
            out[int(m)] = e0.elapsed_time(e1) * 1e-3 / calls
    return out


def main():
    import argparse
    import json
    import os
    from . import build as rosa_build, cases
    from .latency_profile import measure_service_pool
    from .runner import DeviceFleet
    ap = argparse.ArgumentParser(description="closed-loop fleets against one B200: discrete vs continuous batching, rate caps")
    ap.add_argument("--t-act", type=float, default=0.2)
    ap.add_argument("--slo-ms", type=float, default=200.0)
    ap.add_argument("--out", default=os.path.join("gpurun_out", "closed_loop.json"))
    args = ap.parse_args()
    rosa_build.build()
    base = cases.make_case(4, batch=1, with_prefix=False)
    fleet = DeviceFleet(base, [816] * 64, seed=4)
    sizes = [1, 2, 4, 8, 16, 32, 64]
    pools = measure_service_pool(fleet, sizes, calls=10)
    call_ms = {b: float(np.mean(pools[b])) for b in sizes}
    step_s = measure_step_times(fleet, sizes)
    fleet.close()
    interp = lambda tab: (lambda m: float(np.interp(m, sorted(tab), [tab[k] for k in sorted(tab)])))
    call_time, step_time = interp(call_ms), interp(step_s)
    rows = []
    for robots in (16, 64, 256, 512):
        for mode, b in (("discrete", 1), ("discrete", 16), ("discrete", 64), ("continuous", 64)):
            for cap in (None, 3.9):
                r = closed_loop_fleet(robots, args.t_act, cap, 30.0, args.slo_ms * 1e-3, mode, b, call_time, step_time)
                rows.append({"robots": robots, "mode": mode, "batch": b, "rate_cap_hz": cap, **r})
                print(rows[-1])
    os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
    with open(args.out, "w") as f:
        json.dump({"call_ms": {k: 1e3 * v for k, v in call_ms.items()}, "step_ms": {k: 1e3 * v for k, v in step_s.items()},
                   "t_act": args.t_act, "slo_ms": args.slo_ms, "rows": rows}, f, indent=1)


if __name__ == "__main__":
    main()
