"""Adaptive temperatures.  The insertion half is the paper's rule and is pinned
here against a recomputation from the trial's exchange rates; the fixed-R prune half is DESIGN.md
reading S8 ("parity unpinned" by the paper) and is checked for the invariants it promises."""
import numpy as np


def _trial_rates(oracle_mod, L, R, n, J, h, kind, seed, T, trial, k):
    o = oracle_mod.Oracle(L, R, J, h, kind, seed)
    o.set_temperatures(T)
    o.set_adapt_params(k, 4)
    o.sweep(trial, k)
    att, acc = o.get_exchange_counts()
    return acc / att, o


def test_insertion_rule_matches_paper(oracle_mod):
    # M replicas equally spaced; after a trial the a lowest-rate intervals get their midpoint
    L, cap, n0, a, k, trial = 6, 12, 6, 2, 2, 400
    T0 = np.linspace(0.8, 5.0, n0)
    rates, ref = _trial_rates(oracle_mod, L, cap, n0, 1.0, 1.5, 0, 17, T0, trial, k)
    o = oracle_mod.Oracle(L, cap, 1.0, 1.5, 0, 17)
    o.set_temperatures(T0)
    o.set_adapt_params(k, a)
    o.adapt_temperatures(trial)
    T1 = o.get_temperatures()
    assert len(T1) == n0 + a
    lowest = sorted(np.argsort(rates, kind="stable")[:a])
    want = sorted(list(T0) + [(T0[t] + T0[t + 1]) / 2.0 for t in lowest])
    assert np.array_equal(T1, want)
    assert T1[0] == T0[0] and T1[-1] == T0[-1] and np.all(np.diff(T1) > 0)
    # statistics were reset; the run continued on the same global counters
    att, acc = o.get_exchange_counts()
    assert att.sum() == 0 and o.get_counters()[0] == trial
    # new replicas start from the colder neighbour's configuration (reading G6), survivors keep their slots
    perm1 = o.get_permutation()
    perm_trial = ref.get_permutation()
    new_ranks = [i for i, t in enumerate(T1) if t not in T0]
    for q, j in enumerate(new_ranks):
        assert perm1[j] == n0 + q
        assert np.array_equal(o.get_spins(j), ref.get_spins_slot(perm_trial[lowest[q]]))
        assert np.array_equal(o.get_spins(j), o.get_spins(j - 1))
    old_ranks = [i for i, t in enumerate(T1) if t in T0]
    assert np.array_equal(perm1[old_ranks], perm_trial)


def test_insertion_lifts_the_minimum_rate(oracle_mod):
    # as replicas are added the minimum exchange rate rises
    L, cap, k, trial = 6, 20, 2, 600
    o = oracle_mod.Oracle(L, cap, 1.0, 1.0, 0, 5)
    o.set_temperatures(np.linspace(1.0, 5.0, 6))
    o.set_adapt_params(k, 3)
    o.sweep(trial, k)
    r0 = o.observables()[2].min()
    for _ in range(4):
        o.adapt_temperatures(trial)
    assert o.n == 6 + 12
    o.sweep(trial, k)
    r1 = o.observables()[2].min()
    assert r1 > r0 + 0.1, (r0, r1)
    # capacity reached: further calls keep n fixed
    o.adapt_temperatures(trial); o.adapt_temperatures(trial)
    assert o.n == cap


def test_fixed_count_insert_and_prune_invariants(oracle_mod):
    L, R, k, trial, a = 6, 16, 2, 500, 3
    T0 = np.linspace(0.8, 6.0, R)
    rates, ref = _trial_rates(oracle_mod, L, R, R, 1.0, 2.0, 0, 3, T0, trial, k)
    o = oracle_mod.Oracle(L, R, 1.0, 2.0, 0, 3)
    o.set_temperatures(T0)
    o.set_adapt_params(k, a)
    o.adapt_temperatures(trial)
    T1 = o.get_temperatures()
    assert len(T1) == R and T1[0] == T0[0] and T1[-1] == T0[-1] and np.all(np.diff(T1) > 0)
    S = list(np.argsort(rates, kind="stable")[:a])
    rho = rates[S[-1]]
    inserted = [t for t in T1 if t not in T0]
    removed = [i for i, t in enumerate(T0) if t not in T1]
    assert 1 <= len(inserted) == len(removed) <= a
    mids = [(T0[t] + T0[t + 1]) / 2.0 for t in S[:len(inserted)]]
    assert sorted(inserted) == sorted(mids)
    for u in removed:
        assert 1 <= u <= R - 2 and (u - 1) not in S and u not in S      # never next to a split interval
        assert (u - 1) not in removed and (u + 1) not in removed        # never two adjacent
        assert rates[u - 1] * rates[u] * min(rates[u - 1], rates[u]) > rho   # predicted merged rate stays above rho
    # rank preserving: no lattice moved
    assert np.array_equal(o.get_permutation(), ref.get_permutation())
    for r in range(R):
        assert np.array_equal(o.get_spins_slot(r), ref.get_spins_slot(r))
    # moving temperatures toward the slow region raises the worst rate over a few rounds
    for _ in range(3):
        o.adapt_temperatures(trial)
    o.sweep(trial, k)
    assert o.observables()[2].min() > rates.min()
