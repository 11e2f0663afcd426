"""Helpers for the -m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle."""
import os

import numpy as np


def oracle_threads():
    return max(1, min(16, (os.cpu_count() or 1)))


def make_pair(L, R, J, h, kind, seed, T=None, threads=None, **gpu_kw):
    import oracle
    from paper_1508_06268_b200 import binding
    g = binding.RfimPT(L, R, J, h, kind, seed=seed, **gpu_kw)
    o = oracle.Oracle(L, R, J, h, kind, seed, threads=threads or oracle_threads())
    if T is not None:
        g.set_temperatures(T)
        o.set_temperatures(T)
    return g, o


def assert_same_state(g, o, d=0, what="", slots=None):
    """Bit-exact: every slot's spins, the permutation, integer energy terms, counters, exchange counts."""
    assert g.n == o.n, what
    for r in (range(o.R) if slots is None else slots):
        a, b = g.get_spins_slot(r, d=d), o.get_spins_slot(r)
        assert np.array_equal(a, b), f"{what}: spins of slot {r} differ at {np.flatnonzero(a != b)[:8]} ({(a != b).sum()} sites)"
    assert np.array_equal(g.get_permutation(d=d), o.get_permutation()), f"{what}: permutation"
    for x, y, name in zip(g.get_energy_terms(d=d), o.get_energy_terms(), ("Eb", "Ef", "Msum")):
        assert np.array_equal(x, y), f"{what}: {name}"
    assert g.get_counters() == o.get_counters(), f"{what}: counters"
    for x, y, name in zip(g.get_exchange_counts(d=d), o.get_exchange_counts(), ("attempted", "accepted")):
        assert np.array_equal(x, y), f"{what}: {name}"


def assert_same_series(g, o, d=0, what=""):
    for x, y, name in zip(g.get_timeseries(d=d), o.get_timeseries(), ("Eb", "Ef", "Msum")):
        assert x.shape == y.shape and np.array_equal(x, y), f"{what}: series {name}"
