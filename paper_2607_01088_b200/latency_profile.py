"""Latency profile L(b, lambda) of the batched denoise call and the feasible per-server
configurations P(f) built from it — the scheduler's input.

PAPER.md:346-348: "ROSA measures a latency distribution L_{m,h}(b, lambda) for each batching
configuration b and aggregate request rate lambda ... for each System 1 batch size, we profile latency at
ten request rates, ranging from 10% to 100% of the measured maximum throughput for that batch size."
PAPER.md:352: a System-1 server configuration is (model, batch size b, number of robot streams k) with
aggregate load k f; it is valid only if it meets the latency SLO under that load.

Worker model (System 1 uses a *discrete* batch size): one GPU worker; when it is
idle and at least b requests are queued it takes the b oldest and runs one `rosa_denoise_batch` call; all
b requests complete together.  `flush_after` (seconds, optional) starts a partial batch when the oldest
request has waited that long (the paper is silent on partial batches; default: never).

Service times come from the GPU: `measure_service_pool` times real `rosa_denoise_batch_ex` calls with
CUDA events; the event simulation below then runs in virtual time and draws each batch's duration from
that measured pool (seeded), so a 10 x 10 profile takes seconds instead of minutes of real-time pacing.
No arithmetic of the method happens here.
"""
from __future__ import annotations

import argparse
import json
import os
from typing import Callable, Dict, List, Optional, Sequence

import numpy as np


# ------------------------------------------------------------------ arrivals
def periodic_arrivals(k: int, freq_hz: float, n: int, rng: np.random.Generator) -> np.ndarray:
    """k robot streams, each sending every 1/freq seconds with a uniform random phase; first n arrivals."""
    per = 1.0 / freq_hz
    phases = rng.uniform(0.0, per, size=k)
    rounds = int(np.ceil(n / k)) + 1
    t = (phases[None, :] + per * np.arange(rounds)[:, None]).ravel()
    return np.sort(t)[:n]


def poisson_arrivals(rate: float, n: int, rng: np.random.Generator) -> np.ndarray:
    return np.cumsum(rng.exponential(1.0 / rate, size=n))


# ------------------------------------------------------------------ worker simulation
def simulate_discrete_batching(arrivals: Sequence[float], b: int, service_fn: Callable[[int], float],
                               flush_after: Optional[float] = None) -> np.ndarray:
    """Per-request latency (completion - arrival) of one worker with discrete batch size b.
    `service_fn(n)` returns the duration of a call carrying n requests.  Requests that never get
    served (fewer than b left and no flush) get latency NaN."""
    arr = np.asarray(arrivals, dtype=np.float64)
    n = arr.shape[0]
    lat = np.full(n, np.nan)
    head, t_free = 0, 0.0
    while head < n:
        if head + b <= n:
            t_ready = arr[head + b - 1]          # b-th queued request arrives
            take = b
            if flush_after is not None and arr[head] + flush_after < t_ready:
                t_flush = arr[head] + flush_after
                # whoever has arrived by the flush time (or by the time the worker is free) goes
                t_start = max(t_flush, t_free)
                take = int(np.searchsorted(arr, t_start, side="right") - head)
                take = max(1, min(b, take))
                t_ready = t_flush
        else:
            if flush_after is None:
                break
            take = n - head
            t_ready = arr[head] + flush_after
        t_start = max(t_ready, t_free)
        t_done = t_start + float(service_fn(take))
        lat[head:head + take] = t_done - arr[head:head + take]
        head += take
        t_free = t_done
    return lat


def profile(batch_sizes: Sequence[int], service_pool: Dict[int, Sequence[float]], n_requests: int = 2000,
            arrivals: str = "poisson", seed: int = 0, fractions: Sequence[float] = tuple(j / 10 for j in range(1, 11))
            ) -> Dict[int, dict]:
    """L(b, lambda): for each b, latency percentiles at `fractions` of the measured maximum throughput
    mu_b = b / mean service time."""
    out: Dict[int, dict] = {}
    for b in batch_sizes:
        pool = np.asarray(service_pool[b], dtype=np.float64)
        mu = b / float(pool.mean())
        rows = []
        for frac in fractions:
            rng = np.random.default_rng([seed, b, int(round(frac * 1000))])
            lam = frac * mu
            n = max(n_requests, 20 * b)
            k = max(2 * b, 16)                               # periodic mode: k robot streams of lam / k Hz each
            arr = poisson_arrivals(lam, n, rng) if arrivals == "poisson" else periodic_arrivals(k, lam / k, n, rng)
            lat = simulate_discrete_batching(arr, b, lambda m: float(rng.choice(pool)))
            lat = lat[~np.isnan(lat)]
            warm = lat[len(lat) // 10:]                      # drop the start-up transient
            rows.append({"fraction": frac, "rate_per_s": lam, "p50_ms": 1e3 * float(np.percentile(warm, 50)),
                         "p99_ms": 1e3 * float(np.percentile(warm, 99)), "mean_ms": 1e3 * float(warm.mean())})
        out[int(b)] = {"service_ms_mean": 1e3 * float(pool.mean()), "max_throughput_per_s": mu, "rates": rows}
    return out


def feasible_configs(prof: Dict[int, dict], freq_hz: float, slo_ms: float, percentile: str = "p99_ms") -> List[dict]:
    """P(f) for one model: (b, k) with aggregate load k f under the worker's maximum
    throughput and the SLO percentile of L(b, k f) (linear interpolation between profiled rates) below
    the deadline.  For each b the largest feasible k is marked `best`.

    Below the lowest profiled rate nothing is extrapolated flat: a discrete-batch worker waits for
    b requests, so at low load the batch-fill wait grows as 1 / lambda - the first request of a batch waits for
    b - 1 more arrivals, (b - 1) / lambda, before the service time even starts (mean: half of that).  That lower
    bound (and never less than the lowest profiled point) is what is compared with the deadline there
    ("valid only if it satisfies the SLO under the corresponding load")."""
    out = []
    for b, p in sorted(prof.items()):
        rates = np.array([r["rate_per_s"] for r in p["rates"]])
        lats = np.array([r[percentile] for r in p["rates"]])
        means = np.array([r.get("mean_ms", r[percentile]) for r in p["rates"]])
        best = None
        k = b
        # service time of a batch: recorded by profile(); a hand-built profile without it: b / the highest profiled rate
        service_ms = float(p.get("service_ms_mean", 1e3 * b / rates[-1]))
        while k * freq_hz <= rates[-1]:
            lam = k * freq_hz
            fill_ms = 1e3 * (b - 1) / lam
            l = float(np.interp(lam, rates, lats)) if lam >= rates[0] else max(float(lats[0]), service_ms + fill_ms)
            if l <= slo_ms:
                mean = float(np.interp(lam, rates, means)) if lam >= rates[0] else max(float(means[0]), service_ms + 0.5 * fill_ms)
                best = {"batch": int(b), "robots": int(k), "load_per_s": lam, percentile: l, "mean_ms": mean}
                out.append(dict(best))
            k += 1
        if best:
            for c in out:
                if c["batch"] == b and c["robots"] == best["robots"]:
                    c["best"] = True
    return out


# ------------------------------------------------------------------ GPU side
def measure_service_pool(loaded, batch_sizes: Sequence[int], calls: int = 20, warmup: int = 3) -> Dict[int, List[float]]:
    """Durations (seconds, CUDA events on the launch stream) of `calls` real rosa_denoise_batch_ex calls
    per batch size, on the first b robots of a `runner.LoadedCase` / `runner.DeviceFleet`."""
    import torch
    from . import binding as rosa
    case = getattr(loaded, "case")
    noise_all = loaded.noise if hasattr(loaded, "noise") else torch.from_numpy(case.noise).to(loaded.device)
    stream = torch.cuda.Stream(device=loaded.device)
    pools: Dict[int, List[float]] = {}
    with torch.cuda.stream(stream):
        for b in batch_sizes:
            ids = np.arange(b, dtype=np.int32)
            noise = noise_all[:b].contiguous()
            out = torch.empty_like(noise)
            t0 = np.ones(b, dtype=np.float32)
            ns = np.full(b, 10, dtype=np.int32)
            dt = (-t0 / 10).astype(np.float32)
            for _ in range(warmup):
                rosa.rosa_denoise_batch_ex(loaded.expert, ids, noise, t0, dt, ns, out, None, stream)
            stream.synchronize()
            ts = []
            for _ in range(calls):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                rosa.rosa_denoise_batch_ex(loaded.expert, ids, noise, t0, dt, ns, out, None, stream)
                e1.record(stream)
                stream.synchronize()
                ts.append(e0.elapsed_time(e1) * 1e-3)
            pools[int(b)] = ts
    return pools


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n")[0])
    ap.add_argument("--batches", type=int, nargs="+", default=[1, 4, 16, 64])
    ap.add_argument("--freq", type=float, default=5.0, help="per-robot action request frequency f (Hz)")
    ap.add_argument("--slo-ms", type=float, default=200.0, help="p99 deadline (Table 1 of the paper: 200 ms)")
    ap.add_argument("--out", default=os.path.join("gpurun_out", "latency_profile.json"))
    args = ap.parse_args()
    from . import build as rosa_build, cases
    from .runner import DeviceFleet
    rosa_build.build()
    base = cases.make_case(4, batch=1, with_prefix=False)
    fleet = DeviceFleet(base, [816] * max(args.batches), seed=4)
    pools = measure_service_pool(fleet, args.batches)
    prof = profile(args.batches, pools)
    conf = feasible_configs(prof, args.freq, args.slo_ms)
    fleet.close()
    res = {"workload": "pi0-scale expert, prefix 816, 10 Euler steps (BASELINE.json configs[4])", "profile": prof,
           "freq_hz": args.freq, "slo_ms": args.slo_ms, "feasible": [c for c in conf if c.get("best")]}
    os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
    with open(args.out, "w") as f:
        json.dump(res, f, indent=1)
    for b, p in prof.items():
        print(f"b={b}: service {p['service_ms_mean']:.2f} ms, max {p['max_throughput_per_s']:.0f} req/s; p99 at 10%..100%: "
              + " ".join(f"{r['p99_ms']:.0f}" for r in p["rates"]))
    print("feasible (best k per b):", res["feasible"])


if __name__ == "__main__":
    main()
