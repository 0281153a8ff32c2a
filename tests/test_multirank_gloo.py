"""CPU-only, world_size 2 over gloo: the host logic of the N > 1 path (paper_2601_21005_b200/shard.py).

The path shards over vectors with no data-path collective: each rank generates and
filters its own global vector range.  Checked here with the oracle standing in for the per-rank work: the
union of the ranks' shards equals the single-process batch bit for bit, and the timing reduction is a MAX.
"""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2601_21005_b200 import shard, workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nvec, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import sgw_oracle as o
    g = W.Grid(8, 8, 8, 0.5, 0.5, 0.5)
    mine = o.random_vectors(g, W.SEED_VEC, shard.first_vector(rank, nvec), nvec)
    # per-rank work: a 3-term filter with V = 0 (vectors are independent, so no exchange is needed)
    mine = o.cheb_filter(g, np.zeros(g.shape), None, mine, np.array([0.5, 0.25, 0.125]), 0.0, 60.0)
    parts = [torch.zeros(mine.shape, dtype=torch.complex128) for _ in range(world)]
    dist.all_gather(parts, torch.from_numpy(mine))
    ms = shard.max_over_ranks(10.0 + rank)
    if rank == 0:
        out.put((torch.cat(parts).numpy(), ms))
    dist.barrier()
    dist.destroy_process_group()


def test_vector_shards_over_two_ranks_match_single_process():
    world, nvec = 2, 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nvec, q)) for r in range(world)]
    for p in procs:
        p.start()
    got, ms = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    from oracle import sgw_oracle as o
    g = W.Grid(8, 8, 8, 0.5, 0.5, 0.5)
    want = o.random_vectors(g, W.SEED_VEC, 0, world * nvec)
    want = o.cheb_filter(g, np.zeros(g.shape), None, want, np.array([0.5, 0.25, 0.125]), 0.0, 60.0)
    assert np.array_equal(got.view(np.uint64), want.view(np.uint64))
    assert ms == 11.0                                   # MAX over ranks, not rank 0's value
    assert shard.whole_job_rate(100.0, 2, 3, 1000.0) == 600.0
    assert shard.first_vector(3, 64) == 192
