"""The N>1 path of bench.py / batch drivers on CPU: world_size 2, gloo.

Each rank runs its own disorder realisation (seed + rank) -- here with the CPU oracle standing in for the device
library, which is what a test may do -- and the harness logic under test is the sharding module: per-rank seeds,
MAX-over-ranks timing, whole-job rate, gather of observables.  Rank results must equal the same realisations run
serially in one process.
"""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1508_06268_b200 import sharding
from paper_1508_06268_b200.workloads import BIMODAL, linear_ladder

L, R, SWEEPS, K, BASE_SEED = 4, 4, 20, 5, 77


def _run_realisation(seed):
    import oracle
    o = oracle.Oracle(L, R, 1.0, 1.0, BIMODAL, seed)
    o.set_temperatures(linear_ladder(1.0, 4.0, R))
    o.sweep(SWEEPS, K)
    eb, ef, ms = o.get_energy_terms()
    return np.stack([eb, ef, ms]).astype(np.int64), o.get_permutation().astype(np.int64)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seeds = sharding.rank_seeds([BASE_SEED], rank)
        terms, perm = _run_realisation(seeds[0])
        fake_ms = [10.0 + 5.0 * rank, 3.0 - rank]            # rank-dependent "timings"
        mx = sharding.max_over_ranks(fake_ms)
        g_terms = sharding.gather_by_rank(torch.from_numpy(terms))
        g_perm = sharding.gather_by_rank(torch.from_numpy(perm))
        dist.barrier()
        if rank == 0:
            q.put((mx, [t.numpy() for t in g_terms], [p.numpy() for p in g_perm]))
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_ranks_equal_serial_realisations():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    mx, terms, perms = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert mx == [15.0, 3.0]                                   # MAX over ranks, element-wise
    for r in range(world):
        t_ref, p_ref = _run_realisation(BASE_SEED + r)
        assert np.array_equal(terms[r], t_ref) and np.array_equal(perms[r], p_ref)
    assert not np.array_equal(terms[0], terms[1])              # different disorder per rank
    # whole-job rate: both ranks' units over the slowest rank's time
    assert sharding.whole_job_rate(1e6, world, mx[0]) == 2e6 / (15.0 * 1e6)


def test_single_process_identities():
    assert sharding.rank_seeds([4, 9], 3) == [7, 12]
    assert sharding.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    x = torch.arange(3)
    assert len(sharding.gather_by_rank(x)) == 1
