"""Energy / magnetisation reduction against a numpy recomputation of Eq. 1, and call composition."""
import numpy as np
import pytest


def numpy_terms(spins, field, L):
    s = spins.astype(np.int64).reshape(L, L, L)          # [z, y, x]
    eb = (s * (np.roll(s, -1, 2) + np.roll(s, -1, 1) + np.roll(s, -1, 0))).sum()
    ef = (s.reshape(-1) * field.astype(np.int64)).sum()
    return int(eb), int(ef), int(s.sum())


@pytest.mark.parametrize("kind,L", [(0, 4), (1, 6), (0, 2), (1, 8)])
def test_energy_terms_equal_recomputed_hamiltonian_after_every_sweep(oracle_mod, kind, L):
    R, J, h = 3, 1.0, 1.7
    o = oracle_mod.Oracle(L, R, J, h, kind, 99)
    T = np.array([1.0, 2.5, 5.0])
    o.set_temperatures(T)
    f = o.get_field()
    hs = h if kind == 0 else h / 2 ** 20
    for sweep in range(8):
        o.sweep(1, 2)
        Eb, Ef, Ms = o.get_energy_terms()
        E, M, _ = o.observables()
        for t in range(R):
            eb, ef, ms = numpy_terms(o.get_spins(t), f, L)
            assert (Eb[t], Ef[t], Ms[t]) == (eb, ef, ms)
            assert E[t] == (-J * eb) - (hs * ef)
            assert M[t] == ms / L ** 3
    # the series recorded at exchange steps holds the same numbers, by rank at that time
    sEb, sEf, sMs = o.get_timeseries()
    assert sEb.shape == (4, R)


def test_uniform_configurations(oracle_mod):
    # all up: Eb = 3N, Msum = N, Ef = sum h_i ; checkerboard: Eb = -3N
    L = 4
    o = oracle_mod.Oracle(L, 2, 1.0, 1.0, 0, 3)
    o.set_temperatures([1.0, 2.0])
    N = L ** 3
    o.set_spins_slot(0, np.ones(N, dtype=np.int8))
    x, y, z = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    cb = np.zeros(N, dtype=np.int8)
    cb[(x + L * (y + L * z)).reshape(-1)] = (1 - 2 * ((x + y + z) & 1)).reshape(-1)
    o.set_spins_slot(1, cb)
    Eb, Ef, Ms = o.get_energy_terms()
    assert Eb[0] == 3 * N and Ms[0] == N and Ef[0] == o.get_field().sum()
    assert Eb[1] == -3 * N and Ms[1] == 0


def test_sweep_calls_compose(oracle_mod):
    # sweep(20,10) == sweep(10,10); sweep(10,10) == sweep(7,10); sweep(13,10): the exchange fires on the
    # global sweep counter, and every random number is a function of (seed, slot, sweep, site) only
    def run(chunks):
        o = oracle_mod.Oracle(6, 5, 1.0, 1.0, 1, 42)
        o.set_temperatures(np.linspace(1.0, 4.0, 5))
        for n in chunks:
            o.sweep(n, 10)
        return o
    a, b, c = run([20]), run([10, 10]), run([7, 13])
    for o in (b, c):
        assert np.array_equal(a.get_permutation(), o.get_permutation())
        assert a.get_counters() == o.get_counters() == (20, 2)
        for r in range(5):
            assert np.array_equal(a.get_spins_slot(r), o.get_spins_slot(r))


def test_restart_from_snapshot(oracle_mod):
    # state = spins + permutation + counters: a second oracle seeded from a snapshot continues identically
    T = np.linspace(1.0, 4.0, 4)
    a = oracle_mod.Oracle(6, 4, 1.0, 2.0, 0, 8); a.set_temperatures(T); a.sweep(15, 5)
    b = oracle_mod.Oracle(6, 4, 1.0, 2.0, 0, 8); b.set_temperatures(T)
    for r in range(4):
        b.set_spins_slot(r, a.get_spins_slot(r))
    b.set_permutation(a.get_permutation()); b.set_counters(*a.get_counters())
    a.sweep(10, 5); b.sweep(10, 5)
    assert np.array_equal(a.get_permutation(), b.get_permutation())
    for r in range(4):
        assert np.array_equal(a.get_spins_slot(r), b.get_spins_slot(r))


def test_omp_threads_bit_identical(oracle_mod):
    T = np.linspace(1.0, 4.0, 6)
    a = oracle_mod.Oracle(6, 6, 1.0, 1.0, 1, 5); a.set_temperatures(T); a.sweep(12, 4)
    b = oracle_mod.Oracle(6, 6, 1.0, 1.0, 1, 5, threads=3); b.set_temperatures(T); b.sweep(12, 4)
    assert np.array_equal(a.get_permutation(), b.get_permutation())
    for r in range(6):
        assert np.array_equal(a.get_spins_slot(r), b.get_spins_slot(r))
