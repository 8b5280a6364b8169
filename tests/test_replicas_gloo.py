"""World-size-2 gloo test (CPU) of the N > 1 launch logic: replicas only, barrier + MAX-over-ranks
time, whole-job throughput = all tracks / slowest rank."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2105_01796_b200 import replicas
from paper_2105_01796_b200 import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist = replicas.init("gloo")
    assert replicas.rank_world() == (rank, rank, world)
    dist.barrier()
    # every rank builds the same seeded replica of the batch (no data-path exchange)
    wl = W.make_config(0, n_tracks=64)
    checksum = float(np.asarray(wl.loc).sum())
    ms_local = 10.0 * (rank + 1)           # rank 1 is the slow one
    n_local = wl.n_tracks + rank           # uneven counts are summed
    value, ms, total = replicas.job_throughput(n_local, ms_local, dist)
    q.put((rank, value, ms, total, checksum))
    dist.barrier()
    dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, v0, ms0, t0, c0), (r1, v1, ms1, t1, c1) = got
    assert ms0 == ms1 == 20.0                      # MAX over ranks
    assert t0 == t1 == 64 + 65
    assert v0 == v1 == pytest.approx(129 / 20e-3)
    assert c0 == c1                                # identical seeded replicas


def test_single_process_needs_no_group():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    assert replicas.init("gloo") is None
    v, ms, total = replicas.job_throughput(1000, 5.0, None)
    assert (v, ms, total) == (1000 / 5e-3, 5.0, 1000)
