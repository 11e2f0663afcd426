"""-m gpu: replica distribution (include/rfim_pt.h "replica distribution over several GPUs").

The R slots of one realisation are dealt to G shard handles; each sweeps only the slots it stores, and before every
exchange step the 24-byte energy terms per slot are all-gathered so that every shard takes the same exchange decisions.
Only one GPU is available to the tests, so the G "ranks" are G handles of one process, each driven by its own host
thread and its own CUDA stream (no kernel waits for another kernel: the host threads meet at a barrier inside the
gather function and copy one another's rows).  A sharded run must equal the oracle -- hence the single-handle run --
bit for bit: spins of every slot, permutation, energy terms, exchange counters, time series.
"""
import threading

import numpy as np
import pytest
import torch

from paper_1508_06268_b200.sharding import _DevicePtr, replica_window
from paper_1508_06268_b200.workloads import geometric_ladder

pytestmark = pytest.mark.gpu

BIMODAL, GAUSSIAN = 0, 1
_KEEP = []


class LoopbackGather:
    """All-gather among G handles of one process: every participant publishes its rows, waits for the others at a host
    barrier, then copies their rows into its own array (device-to-device, on its own stream)."""

    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world)
        self.rows = [None] * world

    def make(self, rank):
        def gather(terms_ptr, local_offset, local_bytes, total_bytes, stream_ptr):
            t = torch.as_tensor(_DevicePtr(terms_ptr, total_bytes), device="cuda").view(self.world, -1)
            torch.cuda.current_stream().synchronize()           # my rows are final
            self.rows[rank] = t[rank]
            self.barrier.wait()
            for r in range(self.world):
                if r != rank:
                    t[r].copy_(self.rows[r])
            torch.cuda.current_stream().synchronize()
            self.barrier.wait()                                  # nobody overwrites rows a peer still reads
        return gather


class LoopbackBroadcast:
    """Broadcast of one lattice buffer among G handles of one process: the root publishes its buffer, everybody meets at
    a host barrier, the others copy it (device-to-device on their own stream), a second barrier keeps the root from
    overwriting the buffer while a peer still reads it."""

    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world)
        self.src = None

    def make(self, rank):
        def bcast(buf_ptr, nbytes, root, stream_ptr):
            from paper_1508_06268_b200.sharding import _BytePtr
            t = torch.as_tensor(_BytePtr(buf_ptr, nbytes), device="cuda")
            if rank == root:
                torch.cuda.current_stream().synchronize()
                self.src = t
            self.barrier.wait()
            if rank != root:
                t.copy_(self.src)
                torch.cuda.current_stream().synchronize()
            self.barrier.wait()
        return bcast


def _run_sharded(L, R, n, kind, h, seed, T, world, program, packing=8, round_robin=False):
    """program(handle) runs on every shard in its own thread; returns the shard handles."""
    from paper_1508_06268_b200 import binding
    lg = LoopbackGather(world)
    lb = LoopbackBroadcast(world)
    shards, errors = [None] * world, []
    streams = [torch.cuda.Stream() for _ in range(world)]
    _KEEP.append(streams)                                        # the handles keep using these streams after the threads end

    def worker(rank):
        try:
            with torch.cuda.stream(streams[rank]):
                if round_robin:
                    g = binding.RfimPT(L, R, 1.0, h, kind, seed=seed, shard_rr=(rank, world))
                else:
                    g = binding.RfimPT(L, R, 1.0, h, kind, seed=seed, shard=replica_window(R, world, rank))
                g.set_gather(lg.make(rank))
                g.set_broadcast(lb.make(rank))
                if packing != 8:
                    g.set_packing(packing)
                g.set_temperatures(T)
                shards[rank] = g
                program(g)
                g.synchronize()
        except Exception as e:                                   # a dead thread would leave the others at the barrier
            errors.append(e)
            lg.barrier.abort()
            lb.barrier.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not errors, errors
    return shards


@pytest.mark.parametrize("L,R,n,world", [(32, 6, 6, 2), (32, 8, 7, 4), (64, 4, 4, 2), (32, 5, 5, 3), (32, 8, 4, 4),
                                         (16, 6, 6, 2), (8, 8, 7, 4)])     # small lattices: the one-CTA-per-replica kernel visits the slot window
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_sharded_run_equals_oracle(L, R, n, world, kind, h):
    import oracle
    T = geometric_ladder(0.9, 5.0, n)
    o = oracle.Oracle(L, R, 1.0, h, kind, 41)
    o.set_temperatures(T)
    calls = [(3, 0), (8, 2), (5, 5), (7, 3)]
    for a, k in calls:
        o.sweep(a, k)

    def program(g):
        for a, k in calls:
            g.sweep(a, k)

    shards = _run_sharded(L, R, n, kind, h, 41, T, world, program)
    perm = o.get_permutation()
    terms = o.get_energy_terms()
    series = o.get_timeseries()
    for rank, g in enumerate(shards):
        slot0, m = replica_window(R, world, rank)
        for slot in range(slot0, min(slot0 + m, n)):
            assert np.array_equal(g.get_spins_slot(slot), o.get_spins_slot(slot)), (rank, slot)
        assert np.array_equal(g.get_permutation(), perm), rank
        assert g.get_counters() == o.get_counters()
        for x, y in zip(g.get_exchange_counts(), o.get_exchange_counts()):
            assert np.array_equal(x, y)
        for x, y in zip(g.get_timeseries(), series):
            assert np.array_equal(x, y)
        assert g.diagnostics()["ulp_ambiguous"] == 0
    # the energy getter gathers too: every rank must be inside it at the same time
    got = [None] * world
    lg = LoopbackGather(world)

    def getter(rank):
        shards[rank].set_gather(lg.make(rank))
        got[rank] = shards[rank].get_energy_terms()

    ts = [threading.Thread(target=getter, args=(r,)) for r in range(world)]
    [t.start() for t in ts]
    [t.join(timeout=120) for t in ts]
    for rank in range(world):
        for x, y in zip(got[rank], terms):
            assert np.array_equal(x, y), rank
    for g in shards:
        g.close()


def test_sharded_bit_packed_and_fixed_count_adaptation():
    """shards with bit-packed storage; the fixed-count (rank-preserving) adaptation moves no lattice and works sharded."""
    import oracle
    L, R, world = 32, 6, 2
    T = geometric_ladder(0.9, 5.0, R)
    o = oracle.Oracle(L, R, 1.0, 1.5, GAUSSIAN, 77)
    o.set_temperatures(T)
    o.set_adapt_params(4, 2)
    o.adapt_temperatures(40)
    o.sweep(12, 4)

    def program(g):
        g.set_adapt_params(4, 2)
        g.adapt_temperatures(40)
        g.sweep(12, 4)

    shards = _run_sharded(L, R, R, GAUSSIAN, 1.5, 77, T, world, program, packing=1)
    for rank, g in enumerate(shards):
        slot0, m = replica_window(R, world, rank)
        assert np.array_equal(g.get_temperatures(), o.get_temperatures())
        for slot in range(slot0, min(slot0 + m, R)):
            assert np.array_equal(g.get_spins_slot(slot), o.get_spins_slot(slot)), (rank, slot)
        assert np.array_equal(g.get_permutation(), o.get_permutation())
        g.close()


@pytest.mark.parametrize("L,R,n0,world,round_robin", [(32, 12, 5, 2, False), (32, 12, 5, 3, True), (16, 10, 4, 2, True), (32, 9, 6, 4, True),
                                                       (64, 6, 3, 2, True)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_sharded_growing_adaptation_equals_oracle(L, R, n0, world, round_robin, kind, h):
    """the adaptation inserts replicas (pool slots n, n+1, ...; with the round-robin deal the new replica i
    lives on rank i mod G) whose spins are copied from the colder neighbour -- across ranks through the lattice broadcast.
    Three growing trials then a run: every stored slot, the ladder, the permutation and the series equal the oracle's."""
    import oracle
    T = geometric_ladder(0.9, 5.0, n0)
    o = oracle.Oracle(L, R, 1.0, h, kind, 53)
    o.set_temperatures(T)
    o.set_adapt_params(3, 2)
    for _ in range(3):
        o.adapt_temperatures(30)
    o.sweep(9, 3)

    def program(g):
        g.set_adapt_params(3, 2)
        for _ in range(3):
            g.adapt_temperatures(30)
        g.sweep(9, 3)

    shards = _run_sharded(L, R, n0, kind, h, 53, T, world, program, round_robin=round_robin)
    n = o.n
    assert n == min(R, n0 + 6)
    seen = set()
    for rank, g in enumerate(shards):
        assert g.n == n and np.array_equal(g.get_temperatures(), o.get_temperatures())
        for slot in g.stored_slot_ids():
            if slot < n:
                assert np.array_equal(g.get_spins_slot(slot), o.get_spins_slot(slot)), (rank, slot)
                seen.add(slot)
        assert np.array_equal(g.get_permutation(), o.get_permutation()), rank
        assert g.get_counters() == o.get_counters()
        for x, y in zip(g.get_timeseries(), o.get_timeseries()):
            assert np.array_equal(x, y)
        if round_robin:
            assert g.stored_slot_ids() == list(range(rank, R, world))       # slot i lives on rank i mod G
    assert seen == set(range(n))                                              # every active lattice is stored by exactly one rank
    for g in shards:
        g.close()


def test_handles_on_several_host_threads_share_the_kernels():
    """Handles of different sizes (different shared-memory plans of the same kernels) swept concurrently from several host threads,
    many short calls each: every launch must succeed (the kernels' launch attributes are shared, process-wide state) and each
    handle must reproduce what it computes alone."""
    from paper_1508_06268_b200 import binding
    specs = [(32, 3, GAUSSIAN, 1.5, 11), (64, 2, GAUSSIAN, 1.5, 12), (32, 7, BIMODAL, 2.0, 13), (16, 5, GAUSSIAN, 1.0, 14), (8, 6, BIMODAL, 1.0, 15)]
    calls = 25

    def run(spec, stream, out, errors):
        L, R, kind, h, seed = spec
        try:
            with torch.cuda.stream(stream):
                g = binding.RfimPT(L, R, 1.0, h, kind, seed=seed)
                g.set_temperatures(geometric_ladder(0.9, 5.0, R))
                for _ in range(calls):
                    g.sweep(4, 2)
                out.append((g.get_spins_all(), g.get_permutation()))
                g.close()
        except Exception as e:
            errors.append(e)

    alone = []
    for spec in specs:
        out, errors = [], []
        run(spec, torch.cuda.Stream(), out, errors)
        assert not errors, errors
        alone.append(out[0])
    streams = [torch.cuda.Stream() for _ in specs]
    outs, errors = [[] for _ in specs], []
    threads = [threading.Thread(target=run, args=(spec, streams[i], outs[i], errors)) for i, spec in enumerate(specs)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not errors, errors
    for (s0, p0), out in zip(alone, outs):
        assert np.array_equal(out[0][0], s0) and np.array_equal(out[0][1], p0)


def test_trial_rates_getter_matches_oracle_trial():
    """rfim_pt_get_trial_rates returns the rates the last adaptation's update was decided on (Figure 9's per-trial numbers)."""
    import oracle
    from paper_1508_06268_b200 import binding
    T = geometric_ladder(0.9, 5.0, 6)
    g = binding.RfimPT(16, 10, 1.0, 1.0, BIMODAL, seed=3); g.set_temperatures(T); g.set_adapt_params(2, 2)
    o = oracle.Oracle(16, 10, 1.0, 1.0, BIMODAL, 3); o.set_temperatures(T)
    with pytest.raises(binding.RfimPtError):
        g.get_trial_rates()
    o.sweep(40, 2)                                # the trial adapt_temperatures(40) runs: statistics start from zero
    att, acc = o.get_exchange_counts()
    g.adapt_temperatures(40)
    assert np.array_equal(g.get_trial_rates(), acc / att)
    g.close(); o.close()


def test_shard_errors():
    from paper_1508_06268_b200 import binding
    with pytest.raises(binding.RfimPtError):
        binding.RfimPT(32, 6, 1.0, 1.0, BIMODAL, seed=1, shard=(1, 3))     # window not aligned
    with pytest.raises(binding.RfimPtError):
        binding.RfimPT(32, 6, 1.0, 1.0, BIMODAL, seed=1, shard=(6, 3))     # window past R
    g = binding.RfimPT(32, 6, 1.0, 1.0, BIMODAL, seed=1, shard=(3, 3))
    g.set_temperatures(geometric_ladder(1.0, 4.0, 6))
    with pytest.raises(binding.RfimPtError):
        g.get_spins_slot(0)                                                # not stored here
    with pytest.raises(binding.RfimPtError) as e:
        g.sweep(2, 2)                                                      # exchange step without a gather function
    assert e.value.code == binding.ESTATE
    g.close()
    g = binding.RfimPT(32, 6, 1.0, 1.0, BIMODAL, seed=1)
    with pytest.raises(binding.RfimPtError):
        g.set_gather(lambda *a: None)                                      # not a shard
    g.close()
