"""Closed forms and special cases that pin the Metropolis rule, thresholds and update mechanics."""
import numpy as np
import pytest

from stats import binned_mean_se


@pytest.mark.parametrize("kind", [0, 1])
def test_j0_independent_spins_tanh(oracle_mod, kind):
    # J = 0: sites decouple, <s_i> = tanh(beta h h_i), <E> = -h sum_i h_i tanh(beta h h_i)  (Eq. 1 with J=0)
    L, h, T = 4, 0.8, np.array([0.9, 2.0])
    o = oracle_mod.Oracle(L, 2, 0.0, h, kind, 31 + kind)
    o.set_temperatures(T)
    f = o.get_field().astype(np.float64) * (1.0 if kind == 0 else 2.0 ** -20)
    o.sweep(200, 0)
    n = 6000
    E = np.zeros((n, 2)); S = np.zeros((2, L ** 3))
    for i in range(n):
        o.sweep(1, 0)
        for t in range(2):
            s = o.get_spins(t).astype(np.float64)
            S[t] += s
            E[i, t] = -h * (f * s).sum()
    for t in range(2):
        e_exact = -h * (f * np.tanh(h * f / T[t])).sum()
        e_mean, e_se = binned_mean_se(E[:, t])
        assert abs(e_mean - e_exact) < 4 * e_se, (e_mean, e_exact, e_se)
        # per-site magnetisation follows tanh (each site: n samples, sd <= 1/sqrt(n) modulo autocorrelation)
        assert np.abs(S[t] / n - np.tanh(h * f / T[t])).max() < 0.08


@pytest.mark.parametrize("kind", [0, 1])
def test_zero_couplings_every_attempt_accepted(oracle_mod, kind):
    # J = 0, h = 0: dE = 0 for every attempt, min(1, e^0) = 1, so one sweep maps s -> -s exactly, at any T
    o = oracle_mod.Oracle(6, 3, 0.0, 0.0, kind, 9)
    o.set_temperatures([0.5, 1.0, 1e30])
    before = [o.get_spins_slot(r).copy() for r in range(3)]
    o.sweep(1, 0)
    for r in range(3):
        assert np.array_equal(o.get_spins_slot(r), -before[r])
    o.sweep(1, 0)
    for r in range(3):
        assert np.array_equal(o.get_spins_slot(r), before[r])


@pytest.mark.parametrize("kind", [0, 1])
def test_zero_temperature_never_raises_energy(oracle_mod, kind):
    # T -> 0+: thresholds for dE > 0 are 0, dE <= 0 always accepted: each half-sweep is a descent step
    o = oracle_mod.Oracle(6, 1, 1.0, 1.3, kind, 4)
    o.set_temperatures([1e-30])
    E_prev = o.observables()[0][0]
    for sweep in range(6):
        for colour in (0, 1):
            o.half_sweep(0, colour, sweep)
            E = o.observables()[0][0]
            assert E <= E_prev + 1e-9
            E_prev = E
    assert E_prev < -1.5 * 6 ** 3      # and it really descended from a random start (E ~ 0)


def test_threshold_function_values(oracle_mod):
    # floor(min(1, e^-x) 2^32): closed-form spot values
    thr = oracle_mod.threshold_from_x
    assert thr(0.0) == 2 ** 32 and thr(-3.0) == 2 ** 32
    assert thr(np.log(2.0)) in (2 ** 31 - 1, 2 ** 31)        # e^-ln2 = 1/2 up to one rounding of exp
    assert thr(32 * np.log(2.0) + 1e-3) == 0 and thr(1e30) == 0
    assert thr(10 * np.log(2.0)) in (2 ** 22 - 1, 2 ** 22)
    xs = np.linspace(0.0, 25.0, 400)
    t = np.array([thr(x) for x in xs], dtype=np.float64)
    assert np.all(np.diff(t) <= 0)
    assert np.abs(t / 2 ** 32 - np.exp(-xs)).max() < 2.0 ** -31


def test_bimodal_table_is_the_metropolis_ratio(oracle_mod):
    # thr[t][k][b] / 2^32 = min(1, exp(-dE/T)), dE = 2 (J (2k-6) + h (2b-1)); k = (s n + 6)/2, b = (s h_i + 1)/2
    J, h, T = 1.0, 2.0, np.array([0.8, 2.0, 6.0])
    o = oracle_mod.Oracle(4, 3, J, h, 0, 1)
    o.set_temperatures(T)
    for t in range(3):
        for k in range(7):
            for b in range(2):
                dE = 2 * (J * (2 * k - 6) + h * (2 * b - 1))
                want = min(1.0, np.exp(-dE / T[t]))
                got = o.bimodal_threshold(t, k, b) / 2 ** 32
                assert abs(got - want) < 2.0 ** -31
                if dE <= 0:
                    assert o.bimodal_threshold(t, k, b) == 2 ** 32


@pytest.mark.parametrize("kind", [0, 1])
def test_mirror_symmetry(oracle_mod, kind):
    # h_i -> -h_i, s -> -s with the same seed: the mirrored run stays the exact negative forever
    L, R = 6, 4
    T = np.linspace(3.0, 4.2, R)
    a = oracle_mod.Oracle(L, R, 1.0, 1.5, kind, 2718)
    b = oracle_mod.Oracle(L, R, 1.0, 1.5, kind, 2718)
    b.set_field(-a.get_field())
    for r in range(R):
        b.set_spins_slot(r, -a.get_spins_slot(r))
    a.set_temperatures(T); b.set_temperatures(T)
    for _ in range(5):
        a.sweep(6, 3); b.sweep(6, 3)
        assert np.array_equal(a.get_permutation(), b.get_permutation())
        for r in range(R):
            assert np.array_equal(a.get_spins_slot(r), -b.get_spins_slot(r))
        Ea, Ma, _ = a.observables(); Eb_, Mb, _ = b.observables()
        assert np.array_equal(Ea, Eb_) and np.array_equal(Ma, -Mb)
    assert a.get_exchange_counts()[1].sum() > 0                      # exchanges did happen
