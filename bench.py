#!/usr/bin/env python
"""bench.py — action chunks/sec of rosa_denoise_batch on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W]            # our arm (CUDA library)
  python bench.py --impl reference ...                           # the CPU oracle, as it stands
  python bench.py --sweep                                        # cfg4 batch sweep, long form -> gpurun_out/sweep.json

A *step* is one `rosa_denoise_batch` call: the whole hot path (a1..a11) over one batch of
synthetic robots — 10 Euler steps of the pi0-scale action expert for B=64 robots with ragged
prefix lengths U[600,1000] (BASELINE.json configs[2], the configuration the metric "chunks/sec
at B=64" is quoted on; seeds and recipe in DESIGN.md section 3).  One chunk = one robot's
[H, A] actions.  N>1 = N replicas, robots sharded across ranks, no collective in the data path
(DESIGN.md section 7), weak scaling.

Printed JSON keys beyond the base contract: `roofline` (dominant kernel class, event-timed in a
separate un-graphed profiling pass via rosa_profile_batch), `whole_path` (all algorithmic FLOPs
of a call / call time against the three peaks), `classes` (per kernel class ms per call),
`latency_ms` (p50/p99 per call = per chunk), `cpu_baseline`, `sweep` (BASELINE.json configs[4]: chunks/s, p50 / p99
and roofline fraction at B = 1..512, a few timed calls each; N = 1 only), `e2e.with_rebind_of_every_robot`.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "action_chunks_per_sec_B64_10step"
UNIT = "chunks/s"


def ncu_traffic(kernel_class):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel_class` from the `ncu --set full` capture
    recorded in profiles/r2_ncu_traffic.txt, or (None, why): the record names the sha256 of the kernel source it was
    captured with, and a number taken from another build of the kernel is not reported."""
    import hashlib
    rec = os.path.join(ROOT, "profiles", "r2_ncu_traffic.txt")
    if not os.path.exists(rec):
        return None, "no capture recorded"
    with open(rec) as f:
        d = json.load(f)
    ent = d.get(kernel_class)
    if not ent:
        return None, "no capture of this kernel class"
    src = os.path.join(ROOT, "paper_2607_01088_b200", "csrc", ent["source"])
    with open(src, "rb") as f:
        sha = hashlib.sha256(f.read()).hexdigest()
    if sha != ent["source_sha256"]:
        return None, f"capture is of another build of {ent['source']} (profiles/r2_ncu_traffic.txt)"
    return int(ent["dram_bytes_per_launch"]), ent.get("capture", "")


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


# ------------------------------------------------------------------ algorithmic work
def class_flops(cfg, lens, n_euler):
    """Algorithmic FLOPs of one call per kernel class: robots with prefix lengths `lens`, every
    robot active for `n_euler[i]` Euler steps."""
    d, F, H, A = cfg.d_model, cfg.ffn, cfg.horizon, cfg.action_dim
    nq, nkv, hd, Lyr = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.layers
    lens = np.asarray(lens, dtype=np.float64)
    ne = np.asarray(n_euler, dtype=np.float64)
    tok = float((ne * H).sum())                      # token-steps
    out = {
        "inproj": 2.0 * tok * d * A,
        "gemm_embed": 2.0 * tok * (d * d + d * d),   # action half of W_1 + W_2 (time half hoisted)
        "gemm_qkv_rope": 2.0 * tok * d * (nq + 2 * nkv) * hd * Lyr,
        "attention": float((4.0 * nq * H * (lens + H) * hd * Lyr * ne).sum()),
        "gemm_o_resid": 2.0 * tok * nq * hd * d * Lyr,
        "gemm_gateup_geglu": 2.0 * tok * d * 2 * F * Lyr,
        "gemm_down_resid": 2.0 * tok * F * d * Lyr,
        "final_norm_outproj_euler": 2.0 * tok * d * A,
    }
    if getattr(cfg, "time_conditioning", 0) == 1:    # adaptive-norm variant (R25)
        rs = float(ne.sum())                         # robot-steps
        del out["gemm_embed"]                        # h0 = W_in x + b_in only
        out["timevec"] = 2.0 * rs * (2 * d * d + (2 * Lyr + 1) * 3 * d * d)   # time MLP + all modulation vectors
    return out


def call_bytes(cfg, lens, n_euler):
    """Algorithmic HBM bytes of one call: weights once per Euler iteration + prefix K/V once per
    robot-step."""
    d, F, A = cfg.d_model, cfg.ffn, cfg.action_dim
    nq, nkv, hd, Lyr = cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.layers
    params = d * A + d + 2 * d * d + d + d * d + d + A * d + A + d + \
        Lyr * ((nq + 2 * nkv) * hd * d + nq * hd * d + 3 * F * d + 2 * d)
    if getattr(cfg, "time_conditioning", 0) == 1:
        params = d * A + d + 2 * (d * d + d) + A * d + A + (2 * Lyr + 1) * (3 * d * d + 3 * d) + \
            Lyr * ((nq + 2 * nkv) * hd * d + nq * hd * d + 3 * F * d)
    iters = int(np.max(n_euler))
    kv = float((np.asarray(lens, dtype=np.float64) * np.asarray(n_euler, dtype=np.float64)).sum()) * \
        2 * nkv * hd * 2 * Lyr
    return params * 2.0 * iters + kv


# ------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        return {"sm_mhz": (statistics.median(self.samples) if self.samples else None),
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------ reference arm / cpu baseline
def oracle_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def time_oracle(case, robots, n_euler, repeats=1):
    """Wall time of the oracle, as it stands, on `robots` for the first `n_euler` Euler steps."""
    from oracle import rosa_oracle as O
    sub = case.subset(robots)
    sub.n_steps = np.minimum(sub.n_steps, n_euler).astype(np.int32)
    ts = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        O.denoise_case(sub)
        ts.append(time.perf_counter() - t0)
    return ts


def run_reference(args, rank, world):
    """`--impl reference`: the CPU oracle on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    from paper_2607_01088_b200 import cases
    B = args.batch
    n_rob = 1
    case = cases.make_case(2, batch=n_rob)        # same recipe; only the sampled robots are drawn
    full_euler = int(case.n_steps[0])
    # size the per-step sample from one Euler step so that (K + W) steps end within ~3 minutes
    t_one = time_oracle(case, [0], 1)[0]
    budget = 170.0 / max(1, args.steps + args.warmup)
    n_euler = int(max(1, min(full_euler, budget // max(t_one, 1e-6))))
    for _ in range(args.warmup):
        time_oracle(case, [0], n_euler)
    ts = [time_oracle(case, [0], n_euler)[0] for _ in range(args.steps)]
    total = sum(ts)
    chunks = n_rob * args.steps * (n_euler / full_euler)
    value = chunks / total
    cores = oracle_threads()
    sample = (f"{n_rob} robot of the cfg2 recipe (prefix len {int(case.prefix_lens[0])}), first {n_euler} of "
              f"{full_euler} Euler steps per step, counted as {n_euler}/{full_euler} chunk")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"cfg2 fleet batch B={B} (bounded sample)", "inputs": "seeded synthetic"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ our arm
def pct(xs, q):
    xs = sorted(xs)
    if not xs:
        return None
    i = min(len(xs) - 1, max(0, int(round(q * (len(xs) - 1)))))
    return xs[i]


def measure(torch, rosa, expert, ids, noise, t0, dt, ns, out, stream, steps, warmup, barrier=None):
    """W warm-up calls, then exactly K calls timed with CUDA events on `stream`."""
    for _ in range(warmup):
        rosa.rosa_denoise_batch_ex(expert, ids, noise, t0, dt, ns, out, None, stream)
    stream.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    if barrier:
        barrier()
    torch.cuda.synchronize()
    evs[0].record(stream)
    for k in range(steps):
        rosa.rosa_denoise_batch_ex(expert, ids, noise, t0, dt, ns, out, None, stream)
        evs[k + 1].record(stream)
    torch.cuda.synchronize()
    if barrier:
        barrier()
    per_call = [evs[k].elapsed_time(evs[k + 1]) for k in range(steps)]
    return evs[0].elapsed_time(evs[steps]), per_call


def run_ours(args, rank, world, local_rank):
    import torch
    from paper_2607_01088_b200 import binding as rosa
    from paper_2607_01088_b200 import build as rosa_build
    from paper_2607_01088_b200 import cases
    from paper_2607_01088_b200.runner import LoadedCase
    from paper_2607_01088_b200.sharding import assign_robots, max_over_ranks, whole_job_rate

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(dev))
    rosa_build.build()
    rosa.load()
    peaks = load_peaks()

    B = args.batch
    # same weights on every rank, different robots; --config 3 = the continuous-batching mix (extra line, not the contract metric)
    ada = args.time_conditioning == "adarms"
    if args.scaling == "strong" and world > 1:
        # ONE fleet of B robots, partitioned over the ranks by prefix length (KV bytes and attention work, LPT);
        # every rank draws the same fleet and takes its shard: no communication
        fleet = cases.make_case(args.config, batch=B, time_conditioning=1 if ada else 0)
        case = fleet.subset(assign_robots(fleet.prefix_lens, fleet.cfg.horizon, world)[rank])
        B = case.batch
    else:   # weak: B robots per rank; same weights on every rank, different robots
        case = cases.make_case(args.config, batch=B, robot_stream=rank, time_conditioning=1 if ada else 0)
    cfg = case.cfg
    lc = LoadedCase(case, device=dev)
    stream = torch.cuda.Stream(device=dev)
    ids = np.arange(B, dtype=np.int32)
    noise = torch.from_numpy(case.noise).to(dev)
    out = torch.empty_like(noise)
    barrier = (lambda: dist.barrier()) if dist else None

    sampler = ClockSampler(local_rank)
    with torch.cuda.stream(stream):
        # one untimed call outside the sampler builds the graph
        rosa.rosa_denoise_batch_ex(lc.expert, ids, noise, case.t_start, case.dt, case.n_steps, out, None, stream)
        stream.synchronize()
        sampler.start()
        total_ms, per_call = measure(torch, rosa, lc.expert, ids, noise, case.t_start, case.dt, case.n_steps,
                                     out, stream, args.steps, args.warmup, barrier)
        clocks = sampler.stop()
    launches_per_call = rosa.rosa_last_launch_count(lc.expert)
    family = rosa.rosa_kernel_family(lc.expert)
    total_ms = max_over_ranks(total_ms, dist, dev)          # device time of the slowest rank
    units = [B] * world
    if dist and args.scaling == "strong":
        got = [None] * world
        dist.all_gather_object(got, B)
        units = [int(u) for u in got]
    value = whole_job_rate(units, args.steps, total_ms)     # chunks of all ranks / that time

    # ---- end to end: host buffers, H2D + D2H inside the timed region, through the C ABI
    noise_h = torch.from_numpy(case.noise).pin_memory()
    out_h = torch.empty_like(noise_h).pin_memory()
    for _ in range(min(3, args.warmup)):
        rosa.rosa_denoise_batch_host(lc.expert, ids, noise_h, case.t_start, case.dt, case.n_steps, out_h, stream)
    if barrier:
        barrier()
    torch.cuda.synchronize()
    t_e = time.perf_counter()
    for _ in range(args.steps):
        rosa.rosa_denoise_batch_host(lc.expert, ids, noise_h, case.t_start, case.dt, case.n_steps, out_h, stream)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t_e
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e_value = whole_job_rate(units, args.steps, e2e_s * 1e3)
    io_bytes = int(noise_h.numel() * 4)

    if rank != 0:
        lc.close()
        if dist:
            dist.destroy_process_group()
        return

    # ---- the paper's per-request pattern (every request carries a new observation, so its prefix
    # K/V is new): rosa_prefix_kv_bind of every robot before every call.  Host time of a bind, and the end-to-end
    # rate with the 64 re-binds inside the timed region.
    t_b = time.perf_counter()
    for _ in range(5):
        lc.rebind_all()
    bind_us = (time.perf_counter() - t_b) / (5 * B) * 1e6
    torch.cuda.synchronize()
    n_rb = max(3, args.steps // 2)
    for _ in range(2):
        lc.rebind_all()
        rosa.rosa_denoise_batch_host(lc.expert, ids, noise_h, case.t_start, case.dt, case.n_steps, out_h, stream)
    t_e = time.perf_counter()
    for _ in range(n_rb):
        lc.rebind_all()
        rosa.rosa_denoise_batch_host(lc.expert, ids, noise_h, case.t_start, case.dt, case.n_steps, out_h, stream)
    torch.cuda.synchronize()
    e2e_rebind_value = B * n_rb / (time.perf_counter() - t_e)

    # ---- per kernel class (separate un-graphed pass with an event between launches)
    n_prof = 3
    cls_ms, cls_n = {}, {}
    for _ in range(n_prof):
        r = rosa.rosa_profile_batch(lc.expert, ids, noise, case.t_start, case.dt, case.n_steps, out, stream)
        for k, (ms, n) in r.items():
            cls_ms[k] = cls_ms.get(k, 0.0) + ms / n_prof
            cls_n[k] = n
    flops = class_flops(cfg, case.prefix_lens, case.n_steps)
    tot_flops = sum(flops.values())
    tot_bytes = call_bytes(cfg, case.prefix_lens, case.n_steps)
    # The event-timed pass runs the launches un-graphed (an event between launches defeats the overlap of a kernel's
    # prologue with its predecessor's tail), so its classes sum to more than the graphed call: `ms_per_call` is the
    # share of the graphed call (scaled so that the classes sum to ms_per_step), `ms_ungraphed` the raw event time.
    ungraphed_sum = sum(cls_ms.values())
    scale = (total_ms / args.steps) / ungraphed_sum if ungraphed_sum > 0 else 1.0
    classes = {}
    for k, ms in cls_ms.items():
        if cls_n[k] == 0:
            continue
        ent = {"ms_per_call": round(ms * scale, 4), "ms_ungraphed": round(ms, 4), "launches": cls_n[k]}
        if k in flops and ms > 0:
            ent["tflops"] = round(flops[k] / (ms * scale * 1e-3) / 1e12, 1)
        classes[k] = ent
    dom = max((k for k in cls_ms if k in flops), key=lambda k: cls_ms[k])
    dom_tf = flops[dom] / (cls_ms[dom] * 1e-3) / 1e12
    traffic, traffic_note = ncu_traffic(dom)
    # SURVEY 8(d) / BASELINE.md 3: the measured BURST peak is the primary denominator; the sustained one beside it
    roofline = {"bound": "tensor", "kernel": dom, "achieved": round(dom_tf, 1), "peak": peaks["bf16_tflops"], "unit": "TFLOP/s",
                "frac": round(dom_tf / peaks["bf16_tflops"], 4), "traffic": traffic, "traffic_note": traffic_note,
                "peak_source": f"{peaks['source']} bf16_tflops (burst)",
                "peak_sustained": peaks["bf16_tflops_sustained"], "frac_sustained": round(dom_tf / peaks["bf16_tflops_sustained"], 4),
                "launches_per_call": cls_n[dom], "avg_launch_us": round(1e3 * cls_ms[dom] / cls_n[dom], 2),
                "flops_per_launch": flops[dom] / cls_n[dom],
                "timing": "CUDA events between un-graphed launches (rosa_profile_batch), averaged over the call's launches of the class"}
    ms_call = total_ms / args.steps
    t_roof = {name: max(tot_flops / (pk * 1e12), tot_bytes / (peaks["hbm_gbs"] * 1e9)) * 1e3
              for name, pk in (("burst", peaks["bf16_tflops"]), ("sustained", peaks["bf16_tflops_sustained"]),
                               ("nominal", 2250.0))}
    whole = {"tflop_per_call": round(tot_flops / 1e12, 3), "gb_per_call": round(tot_bytes / 1e9, 3),
             "achieved_tflops": round(tot_flops / (ms_call * 1e-3) / 1e12, 1),
             "roofline_ms": {k: round(v, 3) for k, v in t_roof.items()},
             "frac_of_measured_burst": round(t_roof["burst"] / ms_call, 4),
             "frac_of_measured_sustained": round(t_roof["sustained"] / ms_call, 4),
             "frac_of_nominal": round(t_roof["nominal"] / ms_call, 4)}

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample of the same workload
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_rob = 2
        t_cpu = time_oracle(case, list(range(n_rob)), 10)[0]
        cpu = {"value": n_rob / t_cpu, "unit": UNIT, "cores": oracle_threads(), "kind": "oracle",
               "sample": f"robots 0..{n_rob - 1} of the same cfg2 batch, all 10 Euler steps, numpy fp64, "
                         f"{t_cpu:.1f} s wall"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_call, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak",
            "vs_baseline": None, "dtype": "fp16 operands / fp32 accumulate" if os.environ.get("ROSA_GEMM_DTYPE") != "bf16"
            else "bf16 operands / fp32 accumulate", "data": "synthetic",
            "config": {"workload": f"cfg{args.config} " + ("fleet batch" if args.config == 2 else "continuous-batching mix (t_i in {1.0..0.1}, n_i = 10 t_i)") + (", adaptive-RMSNorm time conditioning (pi0.5-style variant, DESIGN.md R25; not the contract workload)" if ada else "") + f": B={B} robots/GPU, pi0-scale expert (18L d1024 8q/1kv hd256 "
                                   f"ffn4096 H50 A32), ragged prefix lengths (sum L={int(case.prefix_lens.sum())}), "
                                   f"up to 10 Euler steps per call, seed {args.config}",
                       "robot_steps_per_call": int(case.n_steps.sum()),
                       "robot_steps_per_sec": float(world * case.n_steps.sum() * args.steps / (total_ms * 1e-3)),
                       "l2": "inputs exceed L2 (%d MB weights + %.2f GB prefix K/V streamed per Euler step)"
                             % (862 if ada else 629, lc.kv_bytes() / 1e9),
                       "kernel_family": "tcgen05" if family == 1 else "cuda-core", "cuda_graph": True,
                       "parallelism": f"replicas x{world}, robots sharded, no collective"},
            "latency_ms": {"p50": pct(per_call, 0.5), "p99": pct(per_call, 0.99), "min": min(per_call)},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": io_bytes, "d2h_bytes_per_step": io_bytes,
                    "with_rebind_of_every_robot": {"value": e2e_rebind_value, "unit": UNIT, "calls": n_rb,
                                                   "bind_us_per_robot": round(bind_us, 2),
                                                   "what": "rosa_prefix_kv_bind of all robots before every call (borrowed bf16 K/V, "
                                                           "asynchronous table update), host wall clock, this rank"}},
            "gpu_launches": int(launches_per_call * args.steps),
            "roofline": roofline, "whole_path": whole, "classes": classes,
            "classes_ungraphed_sum_ms": round(ungraphed_sum, 3)}
    if cpu:
        line["cpu_baseline"] = cpu
    lc.close()
    del lc
    torch.cuda.empty_cache()
    if world == 1 and not args.no_sweep:
        line["sweep"] = sweep_rows(torch, rosa, cases, peaks, stream, compact=True)
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


def sweep_rows(torch, rosa, cases, peaks, stream, compact, sweep_max=512):
    """BASELINE.json configs[4]: B in {1..512}, prefix length 816, 10 Euler steps, ONE expert (max_batch 512) with 512
    robots bound; batch size B = its first B robots.  Per B: chunks/s, p50 / p99 per call (= per chunk), roofline
    fraction against the measured burst peak.  compact = the few-second version that rides in the default line."""
    from paper_2607_01088_b200.runner import DeviceFleet
    base = cases.make_case(4, batch=1, with_prefix=False)
    cfg = base.cfg
    n_rob = min(512, sweep_max)
    fl = DeviceFleet(base, [816] * n_rob, seed=4)
    rows = []
    for B in cases.SWEEP_BATCHES:
        if B > n_rob:
            break
        ids = np.arange(B, dtype=np.int32)
        t0 = np.ones(B, dtype=np.float32)
        ns = np.full(B, 10, dtype=np.int32)
        dt = (-t0 / 10).astype(np.float32)
        noise = fl.noise[:B].contiguous()
        out = torch.empty_like(noise)
        if compact:
            steps = 20 if B <= 64 else (10 if B <= 128 else 6)
        else:
            steps = max(10, min(200, int(2000 / max(1.0, B * 0.4))))
        with torch.cuda.stream(stream):
            total_ms, per_call = measure(torch, rosa, fl.expert, ids, noise, t0, dt, ns, out, stream, steps, 3)
        ms = total_ms / steps
        fl_tot = sum(class_flops(cfg, [816] * B, ns).values())
        by = call_bytes(cfg, [816] * B, ns)
        t_c, t_m = fl_tot / (peaks["bf16_tflops"] * 1e12) * 1e3, by / (peaks["hbm_gbs"] * 1e9) * 1e3
        row = {"B": B, "chunks_per_s": round(B / (ms * 1e-3), 1), "ms_per_call": round(ms, 3), "p50_ms": round(pct(per_call, 0.5), 3),
               "p99_ms": round(pct(per_call, 0.99), 3), "bound": "tensor" if t_c > t_m else "hbm",
               "roofline_ms": round(max(t_c, t_m), 3), "roofline_frac": round(max(t_c, t_m) / ms, 4), "calls": steps}
        if not compact:  # also against the sustained measured peak and the nominal 2250 TFLOP/s / 8 TB/s
            row["roofline_frac_sustained"] = max(fl_tot / (peaks["bf16_tflops_sustained"] * 1e12) * 1e3, t_m) / ms
            row["roofline_frac_nominal"] = max(fl_tot / 2250e12, by / 8000e9) * 1e3 / ms
        rows.append(row)
    fl.close()
    return rows


def run_sweep(args):
    """cfg4 on its own: more timed calls per batch size; rows printed and written to gpurun_out/sweep.json."""
    import torch
    from paper_2607_01088_b200 import binding as rosa
    from paper_2607_01088_b200 import build as rosa_build
    from paper_2607_01088_b200 import cases
    rosa_build.build()
    rosa.load()
    peaks = load_peaks()
    rows = sweep_rows(torch, rosa, cases, peaks, torch.cuda.Stream(), compact=False, sweep_max=args.sweep_max)
    for row in rows:
        print(json.dumps(row), flush=True)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "sweep.json"), "w") as f:
        json.dump({"peaks": peaks, "rows": rows}, f, indent=1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=None, help="robots per GPU (default 64 for cfg2, 256 for cfg3)")
    ap.add_argument("--config", type=int, default=2, choices=[2, 3], help="2 = fleet batch (the metric), 3 = continuous-batching mix")
    ap.add_argument("--time-conditioning", default="concat", choices=["concat", "adarms"],
                    help="concat = the contract workload (pi0-style); adarms = the adaptive-RMSNorm variant (extra line)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = --batch robots per GPU (default); strong = one fleet of --batch robots sharded by prefix length")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="leave the compact cfg4 sweep out of the default line")
    ap.add_argument("--sweep-max", type=int, default=512)
    args = ap.parse_args()
    if args.batch is None:
        args.batch = 64 if args.config == 2 else 256
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                       # timing rule: W >= 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    elif args.sweep:
        run_sweep(args)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
