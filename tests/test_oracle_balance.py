"""Exact pins on the 2^3 lattice: global balance of one checkerboard sweep built from the oracle's
integer thresholds (zero statistical noise), and long-run averages against brute-force enumeration
(north_star: "brute-force exact enumeration of Boltzmann averages on a 2^3 lattice (bimodal and
Gaussian field)").  PAPER.md:47 -- checkerboard updates keep global balance.
"""
import numpy as np
import pytest

from exact_l2 import all_states, boltzmann, exact_averages
from stats import binned_mean_se

TWO32 = 4294967296.0


def _field_values(o):
    f = o.get_field().astype(np.float64)
    return (f, o.h) if o.kind == 0 else (f, o.h / 2 ** 20)


def _half_sweep_matrix(o, states, colour):
    """P[a, b] = probability that one half-sweep of `colour` takes state a to state b (slot 0)."""
    P = np.zeros((256, 256))
    sites = [(x, y, z) for z in range(2) for y in range(2) for x in range(2) if (x + y + z) % 2 == colour]
    for a in range(256):
        o.set_spins_slot(0, states[a].astype(np.int8))
        p = [o.site_threshold(0, x, y, z) / TWO32 for (x, y, z) in sites]
        for mask in range(16):
            prob, b = 1.0, a
            for q, (x, y, z) in enumerate(sites):
                if mask >> q & 1:
                    prob *= p[q]
                    b ^= 1 << (x + 2 * (y + 2 * z))
                else:
                    prob *= 1.0 - p[q]
            P[a, b] += prob
    return P


@pytest.mark.parametrize("kind,h,T", [(0, 1.0, 1.7), (0, 2.0, 0.9), (1, 1.0, 2.3), (1, 2.0, 1.1), (0, 0.7, 4.0)])
def test_checkerboard_sweep_keeps_boltzmann_stationary(oracle_mod, kind, h, T):
    o = oracle_mod.Oracle(2, 1, 1.0, h, kind, 77 + kind)
    o.set_temperatures([T])
    states = all_states()
    f, hs = _field_values(o)
    H, pi = boltzmann(states, 1.0, hs, f, T)
    P0 = _half_sweep_matrix(o, states, 0)
    P1 = _half_sweep_matrix(o, states, 1)
    assert np.allclose(P0.sum(axis=1), 1.0) and np.allclose(P1.sum(axis=1), 1.0)
    # each half-sweep alone and the full sweep (colour 0 then colour 1) leave pi invariant,
    # up to the 2^-32 quantisation of the thresholds
    for P in (P0, P1, P0 @ P1):
        assert np.abs(pi @ P - pi).max() < 1e-8
    # and a wrong rule would not: dropping the field term breaks it by orders of magnitude more
    assert np.abs(pi[::-1] @ (P0 @ P1) - pi[::-1]).max() > 1e-4 or np.allclose(pi, pi[::-1])


@pytest.mark.parametrize("kind,h", [(0, 1.0), (1, 1.0), (0, 2.0)])
def test_long_run_averages_match_enumeration_with_exchange(oracle_mod, kind, h):
    # PT on L=2 with exchange every sweep: per-temperature averages must still be canonical
    # (pins the Metropolis path and the sign/form of the exchange rule, reading G1)
    T = np.array([1.0, 1.6, 2.4, 3.5])
    o = oracle_mod.Oracle(2, len(T), 1.0, h, kind, 2024 + kind)
    o.set_temperatures(T)
    o.sweep(2000, 1)
    o.set_temperatures(T)            # resets statistics; keeps spins
    n = 120000
    o.sweep(n, 1)
    Eb, Ef, Ms = o.get_timeseries()
    f, hs = _field_values(o)
    att, acc = o.get_exchange_counts()
    assert att.sum() == (n // 2) * 2 + (n - n // 2) * 1 and acc.sum() > 0
    for t in range(len(T)):
        E = -1.0 * Eb[:, t] - hs * Ef[:, t]
        am = np.abs(Ms[:, t]) / 8.0
        e_exact, m_exact = exact_averages(1.0, hs, f, T[t])
        e_mean, e_se = binned_mean_se(E)
        m_mean, m_se = binned_mean_se(am)
        assert abs(e_mean - e_exact) < 4 * e_se + 1e-9, (t, e_mean, e_exact, e_se)
        assert abs(m_mean - m_exact) < 4 * m_se + 1e-9, (t, m_mean, m_exact, m_se)
        assert e_se < 0.05          # the check has teeth


def test_long_run_averages_without_exchange(oracle_mod):
    T = [2.5, 4.0]      # high enough that single-temperature Metropolis mixes on its own
    o = oracle_mod.Oracle(2, 2, 1.0, 1.0, 1, 5)
    o.set_temperatures(T)
    f, hs = _field_values(o)
    n = 30000
    E = np.zeros((n, 2)); M = np.zeros((n, 2))
    for i in range(n):
        o.sweep(1, 0)
        Eb, Ef, Ms = o.get_energy_terms()
        E[i] = -Eb - hs * Ef
        M[i] = np.abs(Ms) / 8.0
    assert np.array_equal(o.get_permutation(), [0, 1])
    for t in range(2):
        e_exact, m_exact = exact_averages(1.0, hs, f, T[t])
        e_mean, e_se = binned_mean_se(E[:, t], drop=0.05)
        m_mean, m_se = binned_mean_se(M[:, t], drop=0.05)
        assert abs(e_mean - e_exact) < 4 * e_se
        assert abs(m_mean - m_exact) < 4 * m_se
