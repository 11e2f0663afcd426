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


# ---- the planning step alone, pinned by hand-derived ladders (S8) and by brute force -------------------------
# Every expected ladder below was worked out by hand from the text of DESIGN.md S8, not by running any code:
#   S   = the a lowest-rate intervals (ties: lower rank first), rho = the largest rate in S;
#   a rank u in [1, n-2] may be given up iff neither interval next to it is in S and (r[u-1] r[u]) min(r[u-1], r[u]) > rho;
#   ranks are given up in descending order of that product (ties: larger u first), never two adjacent, at most a;
#   the |removed| lowest-rate intervals of S get their midpoint temperature.
PLAN_CASES = [
    # name, T, rates, R, a, expected ladder
    # S = {0 (0.1), 5 (0.2)}, rho = 0.2.  u=1, 5, 6 touch S.  u=2: .5*.9*.5 = .225, u=3: .729, u=4: .9*.8*.8 = .576: all > rho.
    # Order 3, 4, 2: take 3; 4 and 2 are adjacent to 3.  One removal -> only interval 0 (the lowest of S) is split.
    ("candidates run out", [1, 2, 3, 4, 5, 6, 7, 8], [0.1, 0.5, 0.9, 0.9, 0.8, 0.2, 0.7], 8, 2, [1, 1.5, 2, 3, 5, 6, 7, 8]),
    # three intervals tie at 0.3: S takes the two of lower rank, {0, 1}, rho = 0.3.  u=1, 2 touch S; u=6: .9*.3*.3 = .081 < rho.
    # u=3, 4, 5 tie at .729: larger u first -> 5, then 4 (adjacent to 5: skipped), then 3.  Both intervals of S are split.
    ("ties on rate and on score", [1, 2, 3, 4, 5, 6, 7, 8], [0.3, 0.3, 0.9, 0.9, 0.9, 0.9, 0.3], 8, 2, [1, 1.5, 2, 2.5, 3, 5, 7, 8]),
    # a = min(5, n-1) = 3: every interval is in S, every interior rank touches S: nothing can be given up, nothing is inserted
    ("a larger than n-1", [1, 2, 3, 4], [0.2, 0.6, 0.4], 4, 5, [1, 2, 3, 4]),
    # S = {0}, rho = 0.125.  u=3: .5*.5*.5 = .125 is not > rho.  u=2 and u=4 tie at (.9*.5)*.5: larger u first -> rank 4 goes.
    ("strict inequality against rho", [1, 2, 3, 4, 5, 6], [0.125, 0.9, 0.5, 0.5, 0.9], 6, 1, [1, 1.5, 2, 3, 4, 6]),
    # the two best candidates (u=2: .9*.9*.9, u=3: .9*1*.9 = .81) are adjacent: 3 first (higher score), 2 skipped, then u=5
    # (.8*.8*.8 = .512).  S = {0, 6} (0.05, 0.1), both split.
    ("two adjacent candidates", [1, 2, 3, 4, 5, 6, 7, 8], [0.05, 0.9, 0.9, 1.0, 0.8, 0.8, 0.1], 8, 2, [1, 1.5, 2, 3, 5, 7, 7.5, 8]),
    # growing mode: n = 4 < R = 8, a = min(4, R-n, n-1) = 3: every interval gets its midpoint
    ("paper rule, a capped by n-1", [1, 2, 3, 4], [0.5, 0.1, 0.3], 8, 4, [1, 1.5, 2, 2.5, 3, 3.5, 4]),
    # growing mode, a capped by the pool: R - n = 1 -> only the lowest-rate interval (1) is split
    ("paper rule, a capped by the pool", [1, 2, 3, 4], [0.5, 0.1, 0.3], 5, 4, [1, 2, 2.5, 3, 4]),
    # growing mode, tie: intervals 0 and 2 both 0.2, a = 1 -> the lower rank
    ("paper rule, tie", [1, 2, 4, 8], [0.2, 0.9, 0.2], 6, 1, [1, 1.5, 2, 4, 8]),
]


def test_plan_matches_hand_derived_ladders(oracle_mod):
    for name, T, rate, R, a, want in PLAN_CASES:
        got = oracle_mod.plan_adaptation(T, rate, R, a)
        assert np.array_equal(got, np.array(want, dtype=np.float64)), (name, got)


def test_library_plan_matches_hand_derived_ladders():
    # the CUDA library's host-side planner (rfim_pt_plan_adaptation: no GPU involved) against the same literals
    from paper_1508_06268_b200 import binding
    for name, T, rate, R, a, want in PLAN_CASES:
        got = binding.plan_adaptation(T, rate, R, a)
        assert np.array_equal(got, np.array(want, dtype=np.float64)), (name, got)


def test_fixed_count_plan_is_the_best_admissible_set_by_brute_force(oracle_mod):
    """n == R: over ALL subsets of interior ranks, the ranks given up are the lexicographically first admissible set in S8's
    priority order (descending predicted merged rate, ties larger rank), found here by enumeration; and the ladder inserts
    midpoints into exactly as many of the lowest-rate intervals as ranks were given up."""
    import itertools
    rng = np.random.default_rng(12345)
    from paper_1508_06268_b200 import binding
    for trial in range(300):
        n = int(rng.integers(4, 10))
        a = int(rng.integers(1, 5))
        T = np.cumsum(rng.integers(1, 4, size=n)).astype(np.float64)       # distinct midpoints: T is an integer ladder
        rate = np.round(rng.uniform(0.02, 1.0, size=n - 1), 1 if trial % 3 == 0 else 3)   # coarse rounding -> many ties
        rate = np.maximum(rate, 0.1 if trial % 3 == 0 else 0.001)
        got = oracle_mod.plan_adaptation(T, rate, n, a)
        assert np.array_equal(got, binding.plan_adaptation(T, rate, n, a))
        assert len(got) == n and got[0] == T[0] and got[-1] == T[-1] and np.all(np.diff(got) > 0)
        removed = [u for u in range(n) if T[u] not in got]
        inserted = sorted(t for t in got if t not in T)
        # S, rho and the priority order, as DESIGN.md S8 states them
        a_eff = min(a, n - 1)
        S = list(np.argsort(rate, kind="stable")[:a_eff])
        rho = rate[S[-1]]
        merged = {u: (rate[u - 1] * rate[u]) * min(rate[u - 1], rate[u]) for u in range(1, n - 1)}
        eligible = [u for u in range(1, n - 1) if (u - 1) not in S and u not in S and merged[u] > rho]
        priority = sorted(eligible, key=lambda u: (-merged[u], -u))
        best = None
        for m in range(min(a_eff, len(priority)), -1, -1):
            for sub in itertools.combinations(range(len(priority)), m):       # index tuples come in lexicographic order
                ranks = [priority[i] for i in sub]
                if all(abs(p - q) != 1 for p, q in itertools.combinations(ranks, 2)):
                    key = tuple(1 if i in sub else 0 for i in range(len(priority)))
                    if best is None or key > best[0]:
                        best = (key, sorted(ranks))
        assert sorted(removed) == best[1], (T, rate, a, removed, best)
        mids = sorted((T[t] + T[t + 1]) / 2.0 for t in S[:len(removed)])
        assert inserted == mids, (T, rate, a, inserted, mids)
