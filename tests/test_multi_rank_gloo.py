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


# ---- replica distribution: windows of slots per rank + the all-gather of energy terms -----------
SH_L, SH_R, SH_K = 4, 6, 3


def _shard_worker(rank, world, port, q):
    """Each rank owns a window of the R replica slots.  The oracle stands in for the device library: every rank runs the
    whole chain (cheap at this size) but only CONTRIBUTES the energy terms of its own window; after the all-gather every
    rank must hold the full array and must take the same exchange decisions as a serial run fed with it."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        slot0, m = sharding.replica_window(SH_R, world, rank)
        o = oracle.Oracle(SH_L, SH_R, 1.0, 1.0, BIMODAL, 99)
        o.set_temperatures(linear_ladder(1.0, 4.0, SH_R))
        rows_seen = []
        for step in range(4):
            o.sweep(SH_K, 0)                                             # sweeps need no communication
            eb, ef, ms = o.get_energy_terms()                            # by rank; bring to slot order
            perm = o.get_permutation()
            full = np.zeros((world * m, 3), dtype=np.int64)
            full[perm, 0], full[perm, 1], full[perm, 2] = eb, ef, ms
            mine = torch.zeros((world * m, 3), dtype=torch.int64)
            mine[slot0:slot0 + m] = torch.from_numpy(full[slot0:slot0 + m])   # only my window is valid before the gather
            sharding.all_gather_rows(mine, rank, world)
            assert np.array_equal(mine.numpy()[:SH_R], full[:SH_R]), (rank, step)
            rows_seen.append(mine.numpy().copy())
        dist.barrier()
        if rank == 0:
            q.put(rows_seen)
    finally:
        dist.destroy_process_group()


def test_replica_windows_and_terms_all_gather():
    assert sharding.replica_window(128, 8, 3) == (48, 16)
    assert sharding.replica_window(5, 3, 2) == (4, 2)                     # last window reaches past R (padding)
    try:
        sharding.replica_window(6, 4, 0)
        raise AssertionError("a rank without slots must be refused")
    except ValueError:
        pass
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    rows = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert len(rows) == 4 and all(r.shape == (6, 3) for r in rows)


# ---- round-robin deal ("replica i goes to GPU i mod k") + the lattice broadcast of an inserting adaptation ----
def _rr_worker(rank, world, port, q):
    """Each rank owns slots rank, rank + world, ...  It contributes its rows in the rank-major layout the library hands to the
    gather function for a round-robin shard; after the all-gather, row (r, j) is slot j * world + r.  Then one lattice
    travels from its owner to every rank the way rfim_pt_adapt_temperatures moves an inserted replica's spins."""
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        R = 7
        mine = sharding.replica_round_robin(R, world, rank)
        m = -(-R // world)
        terms_by_slot = np.arange(world * m * 3, dtype=np.int64).reshape(world * m, 3) * 7 + 1     # what each slot's terms are
        rank_major = torch.zeros((world * m, 3), dtype=torch.int64)
        for j, slot in enumerate(mine):
            rank_major[rank * m + j] = torch.from_numpy(terms_by_slot[slot])
        sharding.all_gather_rows(rank_major, rank, world)
        by_slot = np.zeros_like(terms_by_slot)
        for r in range(world):
            for j in range(m):
                by_slot[j * world + r] = rank_major[r * m + j].numpy()
        ok_gather = np.array_equal(by_slot[:R], terms_by_slot[:R])
        # the new replica of pool slot 5 copies slot 2: owner of 2 is rank 2 % world; every rank ends up with the lattice
        src_slot, root = 2, 2 % world
        lattice = torch.full((64,), 255 if rank == root else 0, dtype=torch.uint8)
        dist.broadcast(lattice, src=root)
        ok_bcast = bool((lattice == 255).all())
        dist.barrier()
        q.put((rank, mine, ok_gather, ok_bcast))
    finally:
        dist.destroy_process_group()


def test_round_robin_deal_gather_layout_and_lattice_broadcast():
    assert sharding.replica_round_robin(7, 2, 0) == [0, 2, 4, 6] and sharding.replica_round_robin(7, 2, 1) == [1, 3, 5]
    assert sharding.replica_round_robin(128, 8, 3)[:3] == [3, 11, 19]      # slot i lives on rank i mod 8
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rr_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    slots = sorted(s for _, mine, _, _ in got for s in mine)
    assert slots == list(range(7))                                          # every slot stored by exactly one rank
    assert all(ok_g and ok_b for _, _, ok_g, ok_b in got)
