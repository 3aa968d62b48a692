"""The N>1 path is "replicas only": covered on CPU with world_size 2 over gloo."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from harness import replicas, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        replicas.barrier(world)
        ms, e2e = [10.0, 30.0][rank], [0.5, 0.25][rank]
        mx = replicas.max_over_ranks([ms, e2e], world)
        cfg = synth.Config("r", N=3, W=4, L=0, iters=1, T=5, p_lc=0.0, seed=replicas.rank_seed(0, rank))
        d = synth.generate(cfg)
        out.put((rank, mx, float(d["odom"].sum())))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] == [30.0, 0.5]          # max over ranks, seen by every rank
    assert res[0][2] != res[1][2]                          # replicas draw different trajectories
    assert replicas.whole_job_rate(1000, 2, 0.03) == 2 * 1000 / 0.03


def test_single_rank_is_identity():
    assert replicas.max_over_ranks([1.5, 2.5], 1) == [1.5, 2.5]
    assert replicas.rank_seed(0, 0) == 0
