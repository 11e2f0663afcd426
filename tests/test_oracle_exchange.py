"""Pins for the exchange step (Eq. 2 with reading G1: W = min(1, e^Delta))."""
import numpy as np


def test_exchange_detailed_balance_two_frozen_replicas(oracle_mod):
    # Two replicas with frozen configurations A, B (no sweeps in between).  Only even steps hold a pair.
    # The arrangement process is a 2-state chain whose stationary law must be the joint Boltzmann weight
    #   P(A at T0, B at T1) / P(B at T0, A at T1) = exp(-(b0 E_A + b1 E_B) + (b0 E_B + b1 E_A)).
    L = 4
    T = np.array([2.0, 2.6])
    o = oracle_mod.Oracle(L, 2, 1.0, 1.0, 0, 11)
    o.set_temperatures(T)
    N = L ** 3
    A = np.ones(N, dtype=np.int8)
    B = np.ones(N, dtype=np.int8); B[:1] = -1           # one flipped spin: E_B - E_A = 12 J +- 2 h
    o.set_spins_slot(0, A); o.set_spins_slot(1, B)
    E, _, _ = o.observables()
    b = 1.0 / T
    EA, EB = E[0], E[1]
    w_id = np.exp(-(b[0] * EA + b[1] * EB))
    w_sw = np.exp(-(b[0] * EB + b[1] * EA))
    p_id_exact = w_id / (w_id + w_sw)
    assert 0.02 < p_id_exact < 0.98
    n = 40000
    count_id = 0
    for _ in range(n):
        o.exchange_step()        # even step: pair (0,1)
        o.exchange_step()        # odd step: no pair when n = 2
        count_id += int(o.get_permutation()[0] == 0)
    att, acc = o.get_exchange_counts()
    assert att[0] == n
    p = count_id / n
    # binomial error inflated by the chain's autocorrelation (2-state chain, bounded by 1/gap)
    assert abs(p - p_id_exact) < 5 * np.sqrt(p_id_exact * (1 - p_id_exact) / n) * 3, (p, p_id_exact)
    # the downhill direction is always accepted: Delta >= 0  <=>  colder replica gets the lower energy
    o2 = oracle_mod.Oracle(L, 2, 1.0, 1.0, 0, 11)
    o2.set_temperatures(T)
    o2.set_spins_slot(0, B); o2.set_spins_slot(1, A)     # hot energy at cold T
    o2.exchange_step()
    assert np.array_equal(o2.get_permutation(), [1, 0])


def test_odd_even_alternation_and_bookkeeping(oracle_mod):
    # reading G3: step x (0-based) uses pairs starting at x mod 2; pairs in a step are disjoint
    R = 6
    o = oracle_mod.Oracle(4, R, 1.0, 1.0, 0, 5)
    o.set_temperatures(np.linspace(1.0, 5.0, R))
    o.exchange_step()
    att, acc = o.get_exchange_counts()
    assert list(att) == [1, 0, 1, 0, 1]
    o.exchange_step()
    att, acc = o.get_exchange_counts()
    assert list(att) == [1, 1, 1, 1, 1]
    assert np.all(acc <= att)
    perm = o.get_permutation()
    assert sorted(perm) == list(range(R))
    # get_spins(rank) follows the permutation: temperatures moved, lattices did not
    for t in range(R):
        assert np.array_equal(o.get_spins(t), o.get_spins_slot(perm[t]))


def test_temperature_swap_equals_configuration_swap(oracle_mod):
    # PAPER.md:131 "swap temperatures, which is totally equivalent": after an accepted swap of ranks t,t+1
    # the configuration found at rank t is the one that was at rank t+1, and sweeping it uses T_t.
    T = np.array([1.0, 1.05])
    o = oracle_mod.Oracle(4, 2, 1.0, 1.0, 0, 21)
    o.set_temperatures(T)
    N = 64
    A = np.ones(N, dtype=np.int8); B = np.ones(N, dtype=np.int8); B[:8] = -1
    o.set_spins_slot(0, B); o.set_spins_slot(1, A)      # cold rank holds the higher energy: swap is certain
    o.exchange_step()
    assert np.array_equal(o.get_permutation(), [1, 0])
    assert np.array_equal(o.get_spins(0), A) and np.array_equal(o.get_spins(1), B)
    # the threshold used for slot 1 (now rank 0) is computed with T[0]
    thr_cold = o.site_threshold(1, 0, 0, 0)
    o.set_permutation([0, 1])
    thr_hot = o.site_threshold(1, 0, 0, 0)
    assert thr_cold < thr_hot        # flipping a spin of the all-up state costs energy; colder = smaller
