"""N > 1 host logic on CPU: world_size-2 `gloo` process group (rendezvous on 127.0.0.1).

The data path has no collective (the solve shards by right-hand side); what runs under
torch.distributed is the sharding recipe and the barrier / max-over-ranks timing that bench.py uses.
"""
import os
import socket

import numpy as np
import pytest

from paper_2502_02490_b200 import sharding


def test_shard_rhs_partitions_every_index_once():
    for nrhs in (0, 1, 5, 12, 13):
        for world in (1, 2, 3, 8):
            got = [k for r in range(world) for k in sharding.shard_rhs(nrhs, world, r)]
            assert got == list(range(nrhs))
            sizes = [len(sharding.shard_rhs(nrhs, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_rhs(4, 2, 2)


def test_single_process_identity():
    assert sharding.max_over_ranks(1.5) == 1.5
    assert sharding.whole_job_rate(10.0, 2.0) == (5.0, 2.0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, nrhs, out):
    import torch.distributed as dist
    import synth
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = sharding.shard_rhs(nrhs, world, rank)
        # each rank generates only its own sources, from the GLOBAL right-hand-side index
        sums = {k: complex(synth.gaussian_spinor((2, 2, 2, 2), sharding.rhs_seed(k)).sum()) for k in mine}
        dist.barrier()
        local_seconds = 1.0 + rank          # rank 1 is the slow one
        rate, sec = sharding.whole_job_rate(len(mine), local_seconds, dist)
        mx = sharding.max_over_ranks(local_seconds, dist)
        dist.barrier()
        out.put((rank, mine, sums, rate, sec, mx))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_sharding_and_max_over_ranks_timing():
    import torch.multiprocessing as mp
    import synth
    world, nrhs = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nrhs, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, m0, s0, rate0, sec0, mx0), (r1, m1, s1, rate1, sec1, mx1) = res
    assert m0 == [0, 1, 2] and m1 == [3, 4]
    # whole-job rate = all units / slowest rank's time, identical on both ranks
    assert sec0 == sec1 == mx0 == mx1 == 2.0
    assert rate0 == rate1 == nrhs / 2.0
    # the union of the shards is the single-process workload (same seeds, same sources)
    both = {**s0, **s1}
    for k in range(nrhs):
        exp = complex(synth.gaussian_spinor((2, 2, 2, 2), sharding.rhs_seed(k)).sum())
        assert np.isclose(both[k], exp, rtol=0, atol=0)
