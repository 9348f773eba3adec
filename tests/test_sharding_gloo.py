"""N>1 host logic on CPU: world_size-2 gloo run of the replica sharding and the max-over-ranks
timing reduction that bench.py uses under torchrun."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_01088_b200 import cases
from paper_2607_01088_b200.sharding import assign_robots, max_over_ranks, whole_job_rate


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.Generator(np.random.PCG64(2))
    lens = rng.integers(600, 1000, size=64, endpoint=True)
    mine = assign_robots(lens, 50, world)[rank]
    # every rank must hold the same partition without talking: gather and compare
    got = [None] * world
    dist.all_gather_object(got, mine)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    worst = max_over_ranks(ms, dist)
    dist.barrier()
    q.put((rank, mine, got, worst))
    dist.destroy_process_group()


def test_assign_robots_balanced_and_disjoint():
    lens = np.random.Generator(np.random.PCG64(3)).integers(400, 1200, size=256, endpoint=True)
    for world in (1, 2, 4, 8):
        shards = assign_robots(lens, 50, world)
        flat = sorted(i for s in shards for i in s)
        assert flat == list(range(256))
        loads = [int(sum(lens[i] + 50 for i in s)) for s in shards]
        assert max(loads) - min(loads) <= 1250          # LPT bound: at most one robot's work apart
        assert max(len(s) for s in shards) - min(len(s) for s in shards) <= 2


def test_world2_gloo_sharding_and_max_reduce():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, mine0, got0, worst0), (r1, mine1, got1, worst1) = res
    assert got0 == got1 == [mine0, mine1]
    assert sorted(mine0 + mine1) == list(range(64)) and not set(mine0) & set(mine1)
    assert worst0 == worst1 == 15.0
    assert whole_job_rate([len(mine0), len(mine1)], 10, worst0) == 64 * 10 / 15e-3


def test_rank_robot_streams_share_weights_and_differ_in_robots():
    a = cases.build_case("r0", 9, cases.TINY, bf16=True, draw_lens=(5, 9), batch=3, robot_stream=0)
    b = cases.build_case("r1", 9, cases.TINY, bf16=True, draw_lens=(5, 9), batch=3, robot_stream=1)
    assert all(np.array_equal(a.weights[k], b.weights[k]) for k in cases.GLOBAL_WEIGHTS + cases.BIASES)
    assert all(np.array_equal(x, y) for k in cases.LAYER_WEIGHTS for x, y in zip(a.weights[k], b.weights[k]))
    assert not np.array_equal(a.noise, b.noise)
