"""The N > 1 path on CPU: two processes over gloo run the host-side replica logic bench.py uses under torchrun
(seed per rank, max-over-ranks of the timed region, whole-job rate).  No GPU, no kernels: the path has no
data-path collective ("replicas only")."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2302_14720_b200 import replicas as rp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = rp.replica_seed(rank)
        ms = 2.0 + 0.5 * rank                       # the slower rank sets the job's time
        dist.barrier()
        ms_max = rp.max_over_ranks(ms, dist)
        seeds = [None] * world
        dist.all_gather_object(seeds, seed)
        out.put((rank, seed, ms_max, seeds, rp.whole_job_rate(1 << 20, 10, world, ms_max)))
    finally:
        dist.destroy_process_group()


def test_two_replicas_over_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [6, 7]                      # distinct seeds: independent lattices
    assert all(g[3] == [6, 7] for g in got)
    assert all(g[2] == 2.5 for g in got)                      # max over ranks, identical on every rank
    assert all(g[4] == pytest.approx(2 * (1 << 20) * 10 / 2.5e-3) for g in got)


def test_single_rank_needs_no_process_group():
    assert rp.max_over_ranks(3.25) == 3.25
    assert rp.whole_job_rate(100, 2, 1, 1.0) == pytest.approx(2.0e5)
    with pytest.raises(ValueError):
        rp.replica_seed(-1)
    with pytest.raises(ValueError):
        rp.whole_job_rate(1, 1, 1, 0.0)
