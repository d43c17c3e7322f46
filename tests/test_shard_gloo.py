"""The N>1 path is replicas only: ranks own disjoint event ranges and
only timings are reduced.  world_size-2 gloo processes on CPU check exactly that host logic."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import stcf_inputs as si
from paper_2607_04067_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_per_rank, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = si.config(0)
        first, last = shard.event_range(rank, world, n_per_rank)
        xy, off, _ = si.generate(w, last - first, first_event=first)
        ms = 10.0 + 5.0 * rank                                 # the slower rank decides
        agg = shard.max_over_ranks([ms, float(len(xy))])
        q.put((rank, first, last, xy.tobytes(), off.tolist(), agg, shard.job_throughput(n_per_rank, world, agg[0])))
    finally:
        dist.destroy_process_group()


def test_two_ranks_own_disjoint_event_ranges_and_reduce_by_max():
    world, n_per_rank = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_per_rank, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # the two shards together are exactly the single-process stream of 2*n events
    w = si.config(0)
    xy_all, off_all, _ = si.generate(w, world * n_per_rank)
    got = b"".join(r[3] for r in res)
    assert got == xy_all.tobytes()
    assert [r[1:3] for r in res] == [(0, 5), (5, 10)]
    assert res[1][4][-1] + res[0][4][-1] == off_all[-1]
    # timings: max over ranks on every rank; throughput = all events / slowest time
    for r in res:
        assert r[5][0] == 15.0
        assert r[5][1] == float(max(len(res[0][3]), len(res[1][3])) // 8)
        assert abs(r[6] - 10 / 0.015) < 1e-6


def test_event_ranges_of_the_ranks_tile_the_event_stream():
    assert shard.event_range(3, 4, 250) == (750, 1000)
    ranges = [shard.event_range(r, 8, 125) for r in range(8)]
    assert ranges[0][0] == 0 and all(a[1] == b[0] for a, b in zip(ranges, ranges[1:])) and ranges[-1][1] == 1000
