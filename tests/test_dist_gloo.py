"""N > 1 plumbing on CPU (gloo, world_size 2): replicas only -- DESIGN.md "Multi-GPU".

Checks what bench.py relies on under torchrun: ranks take disjoint ranges of the counter-based particle
stream, the timed region is bracketed by a barrier, the step time is the MAX over ranks and the work is
the SUM over ranks.  No GPU, no data-path collective.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1710_07350_b200 import dist as pdist
    from elg_inputs import make_workload
    assert pdist.env_rank() == (rank, rank, world)
    assert pdist.init_process_group("gloo") == world
    n = 1000
    w = make_workload("cfg0", n=n)
    mine = w.particles(n, start=pdist.shard_start(rank, n))
    pdist.barrier()
    t_max, units = pdist.aggregate(10.0 + 5.0 * rank, float(n * 3), "cpu")
    q.put((rank, t_max, units, mine[:, :4].copy(), mine[:, -1].copy()))
    pdist.barrier()
    torch.distributed.destroy_process_group()


def test_two_ranks_gloo_replicas():
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=120) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t_max, units, head, last in got:
        assert t_max == 15.0                       # max over ranks
        assert units == 2 * 1000 * 3               # sum over ranks
    # disjoint, contiguous ranges of one stream: rank 1 continues where rank 0 stopped
    from elg_inputs import make_workload
    w = make_workload("cfg0", n=2000)
    both = w.particles(2000)
    assert np.array_equal(got[0][3], both[:, :4])
    assert np.array_equal(got[1][3], both[:, 1000:1004])
    assert np.array_equal(got[1][4], both[:, 1999])
    assert not np.array_equal(got[0][3], got[1][3])


def test_shard_start_and_single_process_identity():
    from paper_1710_07350_b200 import dist as pdist
    assert pdist.shard_start(0, 10) == 0 and pdist.shard_start(3, 10) == 30
    with pytest.raises(ValueError):
        pdist.shard_start(-1, 10)
    assert pdist.aggregate(2.5, 7.0) == (2.5, 7.0)   # no process group: identity
    pdist.barrier()                                   # no-op
