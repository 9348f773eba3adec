"""A real request queue and GPU worker in front of the library, driven in real time.

The paper's System-1 worker hosts one model and serves per-robot requests with a scheduler-chosen DISCRETE batch
size; clients are closed-loop - send, wait for the chunk, act for t_act, send again,
never faster than the scheduled rate (request-rate control) - and the metric is
SLO-qualified actions per second.  `latency_profile.py` / `batcher.closed_loop_fleet` model this in
virtual time; here nothing is simulated:

* `Worker` - a thread with a request queue.  Discrete mode: when `batch` requests wait (or the oldest has waited
  `flush_after`, or every client is waiting) it takes the oldest and runs ONE blocking batch call.  Continuous mode
  (BASELINE.json configs[3]): waiting requests are admitted at every Euler-step boundary into a
  `batcher.ContinuousBatcher`, one launch per step.  Completion times are host timestamps taken after the stream
  has been synchronised, so launch cost, graph capture on a new shape and queueing are all inside the latency.
* `open_loop` - a pacing thread that submits requests at given arrival times: L(b, lambda) as a measurement
  (PAPER.md:346-348).
* `closed_loop` - n virtual robots with t_act and an optional per-robot rate cap against a worker.

Host logic only: the batch call is a function the caller passes in (`gpu_batch_call` below wraps
`rosa_denoise_batch_ex`; the CPU tests pass a sleep), so everything here is testable without a device.
"""
from __future__ import annotations

import heapq
import threading
import time
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional, Sequence

import numpy as np


@dataclass(order=True)
class Request:
    t_arrival: float                      # host clock (time.perf_counter) at which the robot sent it
    robot: int = field(compare=False)
    t_done: float = field(default=float("nan"), compare=False)


def _sleep_until(t: float) -> None:
    """Coarse sleep, then a short spin: arrival times are honoured to ~50 us."""
    while True:
        d = t - time.perf_counter()
        if d <= 0:
            return
        if d > 3e-4:
            time.sleep(d - 2e-4)


class Worker:
    """One GPU worker: request queue + serving thread.

    run_batch(robots: List[int]) -> None   blocking call that serves these robots' requests together (discrete mode)
    stepper                                 a `batcher.ContinuousBatcher`-like object (admit / step / __len__) and a
                                            `sync()` callable (continuous mode); `noise_of(robot)` gives the admit input
    """

    def __init__(self, batch: int, run_batch: Optional[Callable[[List[int]], None]] = None, *, flush_after: Optional[float] = None,
                 n_clients: Optional[int] = None, stepper=None, sync: Optional[Callable[[], None]] = None,
                 noise_of: Optional[Callable[[int], object]] = None, on_done: Optional[Callable[[Request], None]] = None):
        assert (run_batch is None) != (stepper is None), "either a batch call (discrete) or a stepper (continuous)"
        self.batch, self.run_batch, self.flush_after, self.n_clients = batch, run_batch, flush_after, n_clients
        self.stepper, self.sync, self.noise_of, self.on_done = stepper, sync, noise_of, on_done
        self.q: List[Request] = []            # heap by arrival time
        self.done: List[Request] = []
        self.cv = threading.Condition()
        self.stop_flag = False
        self.error: Optional[BaseException] = None
        self.busy_s = 0.0
        self.calls = 0
        self.thread = threading.Thread(target=self._guard, daemon=True)

    # -- client side
    def submit(self, req: Request) -> None:
        with self.cv:
            heapq.heappush(self.q, req)
            self.cv.notify_all()

    def start(self) -> "Worker":
        self.thread.start()
        return self

    def stop(self) -> None:
        with self.cv:
            self.stop_flag = True
            self.cv.notify_all()
        self.thread.join(timeout=60)
        if self.error is not None:
            raise self.error

    # -- worker side
    def _guard(self):
        try:
            (self._loop_discrete if self.stepper is None else self._loop_continuous)()
        except BaseException as e:  # surfaced by stop()
            self.error = e

    def _finish(self, reqs: Sequence[Request]) -> None:
        now = time.perf_counter()
        for r in reqs:
            r.t_done = now
        with self.cv:
            self.done.extend(reqs)
        if self.on_done:
            for r in reqs:
                self.on_done(r)

    def _loop_discrete(self):
        while True:
            with self.cv:
                while True:
                    if self.stop_flag:
                        return
                    n = len(self.q)
                    if n >= self.batch or (self.n_clients is not None and n > 0 and n >= self.n_clients):
                        break
                    timeout = None
                    if self.flush_after is not None and n > 0:
                        wait = self.q[0].t_arrival + self.flush_after - time.perf_counter()
                        if wait <= 0:
                            break
                        timeout = wait
                    self.cv.wait(timeout)
                take = [heapq.heappop(self.q) for _ in range(min(self.batch, len(self.q)))]
            t0 = time.perf_counter()
            self.run_batch([r.robot for r in take])
            self.busy_s += time.perf_counter() - t0
            self.calls += 1
            self._finish(take)

    def _loop_continuous(self):
        inflight: Dict[int, Request] = {}
        while True:
            with self.cv:
                while not self.stop_flag and not self.q and not inflight:
                    self.cv.wait()
                if self.stop_flag:
                    return
                admit = []
                while self.q and len(inflight) + len(admit) < self.batch:
                    admit.append(heapq.heappop(self.q))
            for r in admit:                       # admission at the step boundary
                self.stepper.admit(r.robot, self.noise_of(r.robot))
                inflight[r.robot] = r
            t0 = time.perf_counter()
            finished = self.stepper.step()
            self.sync()
            self.busy_s += time.perf_counter() - t0
            self.calls += 1
            if finished:
                self._finish([inflight.pop(robot) for robot, _ in finished])


# ------------------------------------------------------------------ accounting
def summarize(done: Sequence[Request], t_begin: float, t_end: float, slo_s: float) -> Dict[str, float]:
    """Raw and SLO-qualified actions/s and latency percentiles of the requests that completed in [t_begin, t_end]."""
    lat = np.array([r.t_done - r.t_arrival for r in done if t_begin <= r.t_done <= t_end])
    span = max(t_end - t_begin, 1e-9)
    if lat.size == 0:
        return {"requests": 0, "actions_per_s": 0.0, "qualified_actions_per_s": 0.0, "slo_meet_rate": float("nan"),
                "p50_ms": float("nan"), "p99_ms": float("nan"), "mean_ms": float("nan")}
    return {"requests": int(lat.size), "actions_per_s": lat.size / span,
            "qualified_actions_per_s": float((lat <= slo_s).sum()) / span, "slo_meet_rate": float((lat <= slo_s).mean()),
            "p50_ms": 1e3 * float(np.percentile(lat, 50)), "p99_ms": 1e3 * float(np.percentile(lat, 99)),
            "mean_ms": 1e3 * float(lat.mean())}


# ------------------------------------------------------------------ open loop: L(b, lambda) as a measurement
def open_loop(worker: Worker, arrivals: Sequence[float], n_robots: int, slo_s: float, warm_frac: float = 0.1,
              drain_s: float = 5.0) -> Dict[str, float]:
    """Submit one request at each (relative) arrival time, robots round-robin over n_robots (>= the batch size, so a
    batch never carries a robot twice), wait for the queue to drain, and summarise the requests after the first
    `warm_frac` of the run.  A request's latency counts from its SCHEDULED arrival: pacing lag is not hidden."""
    arr = np.asarray(arrivals, dtype=np.float64)
    assert n_robots >= worker.batch
    t0 = time.perf_counter() + 0.01
    for i, ta in enumerate(arr):
        _sleep_until(t0 + ta)
        worker.submit(Request(t0 + float(ta), int(i % n_robots)))
    served = len(arr) - (len(arr) % worker.batch if worker.flush_after is None and worker.stepper is None else 0)
    t_lim = time.perf_counter() + drain_s
    while len(worker.done) < served and time.perf_counter() < t_lim and worker.error is None:
        time.sleep(1e-3)
    with worker.cv:
        t_end = max([r.t_done for r in worker.done], default=time.perf_counter())   # the window ends with the last completion
    res = summarize(worker.done, t0 + warm_frac * float(arr[-1]), t_end, slo_s)
    res["offered_per_s"] = len(arr) / float(arr[-1]) if arr[-1] > 0 else float("nan")
    res["unserved"] = len(arr) - len(worker.done)
    return res


# ------------------------------------------------------------------ closed loop: robots with t_act and a rate cap
def closed_loop(worker: Worker, n_robots: int, t_act: float, rate_cap_hz: Optional[float], duration_s: float, slo_s: float,
                seed: int = 0, warm_frac: float = 0.1) -> Dict[str, float]:
    """n_robots closed-loop clients for duration_s of real time.  A robot sends, waits for its chunk, executes for
    t_act and sends again - never sooner than 1 / rate_cap after its previous request (request-rate control,
    PAPER.md:486-488).  Installs itself as the worker's completion callback."""
    period = 0.0 if not rate_cap_hz else 1.0 / rate_cap_hz
    rng = np.random.default_rng(seed)
    cv = threading.Condition()
    t0 = time.perf_counter() + 0.01
    heap = [(t0 + float(rng.uniform(0.0, max(t_act, period, 1e-3))), r) for r in range(n_robots)]   # desynchronised start
    heapq.heapify(heap)
    last_send = [-1e18] * n_robots

    def on_done(req: Request):
        with cv:
            heapq.heappush(heap, (max(req.t_done + t_act, last_send[req.robot] + period), req.robot))
            cv.notify()

    worker.on_done = on_done
    t_stop = t0 + duration_s
    while True:
        with cv:
            while not heap and time.perf_counter() < t_stop:
                cv.wait(timeout=max(1e-4, min(0.01, t_stop - time.perf_counter())))
            if time.perf_counter() >= t_stop or worker.error is not None:
                break
            t_next, robot = heap[0]
            if t_next > time.perf_counter() + 3e-4:
                cv.wait(timeout=min(t_next - time.perf_counter() - 2e-4, t_stop - time.perf_counter()))
                continue
            heapq.heappop(heap)
        _sleep_until(t_next)
        last_send[robot] = t_next
        worker.submit(Request(t_next, robot))
    return summarize(worker.done, t0 + warm_frac * duration_s, t_stop, slo_s)


# ------------------------------------------------------------------ the real batch call
def gpu_batch_call(fleet, n_steps: int = 10):
    """run_batch for `Worker` on a `runner.DeviceFleet` / `LoadedCase`-like object (expert, noise, device): one
    `rosa_denoise_batch_ex` call for the given robots on a private stream, synchronised before it returns."""
    import torch
    from . import binding as rosa
    stream = torch.cuda.Stream(device=fleet.device)
    noise_all = fleet.noise
    out = torch.empty_like(noise_all)

    def run(robots: List[int]) -> None:
        b = len(robots)
        ids = np.asarray(robots, dtype=np.int32)
        idx = torch.as_tensor(ids.astype(np.int64), device=noise_all.device)
        with torch.cuda.stream(stream):
            x = noise_all.index_select(0, idx)          # each request carries its own noise
            t0 = np.ones(b, dtype=np.float32)
            rosa.rosa_denoise_batch_ex(fleet.expert, ids, x, t0, (-t0 / n_steps).astype(np.float32),
                                       np.full(b, n_steps, dtype=np.int32), out[:b], None, stream)
        stream.synchronize()

    return run


def continuous_worker(fleet, max_inflight: int, n_steps: int = 10, **kw) -> Worker:
    """A `Worker` in continuous mode on a DeviceFleet: admissions at Euler-step boundaries (BASELINE.json configs[3])."""
    import torch
    from .batcher import ContinuousBatcher
    cfg = fleet.case.cfg
    stream = torch.cuda.Stream(device=fleet.device)
    cb = ContinuousBatcher(fleet.expert, cfg.horizon, cfg.action_dim, max_inflight, n_steps=n_steps, device=fleet.device, stream=stream)

    class _Stepper:
        def admit(self, robot, noise):
            with torch.cuda.stream(stream):
                cb.admit(robot, noise)

        def step(self):
            with torch.cuda.stream(stream):
                return cb.step()

        def __len__(self):
            return len(cb)

    return Worker(max_inflight, stepper=_Stepper(), sync=stream.synchronize, noise_of=lambda r: fleet.noise[r], **kw)


# ------------------------------------------------------------------ measurements on the GPU
def measure_latency_profile(fleet, batch_sizes: Sequence[int], slo_s: float, seconds_per_point: float = 2.5,
                            fractions: Sequence[float] = tuple(j / 10 for j in range(1, 11)), seed: int = 0) -> Dict[int, dict]:
    """L(b, lambda) MEASURED: per batch size, Poisson arrivals paced in real time at ten rates from
    10% to 100% of the measured maximum throughput mu_b = b / (mean duration of a back-to-back call), against a
    discrete-batch `Worker` making real `rosa_denoise_batch_ex` calls.  Next to every measured row: the virtual-time
    simulator of latency_profile.py on the SAME arrivals with the measured mean service time (the cross-check)."""
    from . import latency_profile as lp
    run = gpu_batch_call(fleet)
    n_robots = int(fleet.noise.shape[0])
    out: Dict[int, dict] = {}
    for b in batch_sizes:
        robots = list(range(b))
        for _ in range(3):
            run(robots)                                           # warm-up: graph capture for this bucket
        t0 = time.perf_counter()
        reps = 8
        for _ in range(reps):
            run(robots)
        service = (time.perf_counter() - t0) / reps               # host-to-host, synchronised: what a request sees
        mu = b / service
        rows = []
        for frac in fractions:
            rng = np.random.default_rng([seed, b, int(round(frac * 1000))])
            lam = frac * mu
            n = max(int(lam * seconds_per_point), 4 * b)
            n -= n % b                                            # whole batches (no flush: the paper's worker)
            arr = lp.poisson_arrivals(lam, n, rng)
            w = Worker(b, run).start()
            res = open_loop(w, arr, n_robots=max(n_robots, b), slo_s=slo_s, drain_s=10.0)
            w.stop()
            sim = lp.simulate_discrete_batching(arr, b, lambda m: service)
            sim = sim[~np.isnan(sim)][len(arr) // 10:]
            rows.append({"fraction": frac, "rate_per_s": lam, **{k: res[k] for k in ("requests", "p50_ms", "p99_ms", "mean_ms",
                         "slo_meet_rate", "actions_per_s", "unserved")},
                         "sim_p50_ms": 1e3 * float(np.percentile(sim, 50)), "sim_p99_ms": 1e3 * float(np.percentile(sim, 99)),
                         "sim_mean_ms": 1e3 * float(sim.mean()), "worker_busy_frac": w.busy_s / max(arr[-1], 1e-9)})
        out[int(b)] = {"service_ms_mean": 1e3 * service, "max_throughput_per_s": mu, "rates": rows}
    return out


def main():
    import argparse
    import json
    import os
    from . import build as rosa_build, cases
    from . import latency_profile as lp
    from .runner import DeviceFleet
    ap = argparse.ArgumentParser(description="real-time latency profile L(b, lambda) and closed-loop fleets against one B200")
    ap.add_argument("--batches", type=int, nargs="+", default=[1, 4, 16, 64])
    ap.add_argument("--robots", type=int, nargs="+", default=[16, 64, 256])
    ap.add_argument("--t-act", type=float, default=0.2)
    ap.add_argument("--slo-ms", type=float, default=200.0, help="p99 deadline (Table 1 of the paper: 200 ms)")
    ap.add_argument("--freq", type=float, default=3.9, help="scheduled per-robot request rate f (Hz): the rate cap")
    ap.add_argument("--seconds", type=float, default=2.5, help="real time per (b, rate) point; closed loops run twice as long")
    ap.add_argument("--out", default=os.path.join("gpurun_out", "serving.json"))
    args = ap.parse_args()
    rosa_build.build()
    base = cases.make_case(4, batch=1, with_prefix=False)
    n_fleet = max(max(args.robots), max(args.batches))
    fleet = DeviceFleet(base, [816] * n_fleet, seed=4)
    slo = args.slo_ms * 1e-3
    prof = measure_latency_profile(fleet, args.batches, slo, args.seconds)
    for b, p in prof.items():
        print(f"b={b}: service {p['service_ms_mean']:.2f} ms, max {p['max_throughput_per_s']:.0f} req/s; measured p99 (ms) at 10%..100%: "
              + " ".join(f"{r['p99_ms']:.0f}" for r in p["rates"]) + " | simulated: " + " ".join(f"{r['sim_p99_ms']:.0f}" for r in p["rates"]), flush=True)
    feas = [c for c in lp.feasible_configs(prof, args.freq, args.slo_ms) if c.get("best")]
    print("feasible (best k per b) at f = %.1f Hz, p99 <= %.0f ms:" % (args.freq, args.slo_ms), feas, flush=True)
    rows = []
    for robots in args.robots:
        for mode, b in (("discrete", 1), ("discrete", 16), ("discrete", 64), ("continuous", 64)):
            if mode == "discrete" and b > robots:
                continue
            for cap in (None, args.freq):
                if mode == "discrete":
                    w = Worker(b, gpu_batch_call(fleet), n_clients=robots).start()
                else:
                    w = continuous_worker(fleet, min(b, robots)).start()
                r = closed_loop(w, robots, args.t_act, cap, 2 * args.seconds, slo)
                w.stop()
                rows.append({"robots": robots, "mode": mode, "batch": b, "rate_cap_hz": cap, "launches": w.calls, **r})
                print(rows[-1], flush=True)
    fleet.close()
    os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
    with open(args.out, "w") as f:
        json.dump({"workload": "pi0-scale expert, prefix 816, 10 Euler steps (BASELINE.json configs[4]); real-time pacing, host clocks",
                   "slo_ms": args.slo_ms, "t_act": args.t_act, "freq_hz": args.freq, "profile": prof, "feasible": feas,
                   "closed_loop": rows}, f, indent=1)


if __name__ == "__main__":
    main()
