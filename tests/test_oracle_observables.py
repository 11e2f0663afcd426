"""Pins of the oracle's thermal moments and of the observables of PAPER.md:249-260 (Eq. 11-13): exact enumeration of
the 2x2x2 lattice under parallel tempering, the J = 0 closed forms (independent spins), and the limits of the Binder
factor.  None of these recomputes the oracle's own sums: the expected values come from enumeration or closed forms."""
import numpy as np
import pytest

from exact_l2 import exact_moments
from stats import binned_mean_se


def _series_quantities(o, hs, skip):
    """per-step e, e^2, |m|, m^2, m^4 by rank from the integer time series (only to estimate standard errors)."""
    eb, ef, ms = o.get_timeseries()
    e = (-o.J * eb[skip:] - hs * ef[skip:]) / o.N
    m = ms[skip:] / o.N
    return [e, e * e, np.abs(m), m * m, m ** 4]


@pytest.mark.parametrize("kind", [0, 1])
def test_l2_parallel_tempering_moments_match_enumeration(oracle_mod, kind):
    h, T = 1.2, np.array([1.5, 2.5, 4.0])
    o = oracle_mod.Oracle(2, 3, 1.0, h, kind, 17 + kind)
    o.set_temperatures(T)
    hs = h if kind == 0 else h * 2.0 ** -20
    f = o.get_field().astype(np.float64)
    o.sweep(40000, 2)
    skip = 2000
    mom = o.thermal_moments(skip)
    q = _series_quantities(o, hs, skip)
    for t in range(3):
        exact = exact_moments(1.0, hs, f, T[t])
        for j in range(5):
            mean, se = binned_mean_se(q[j][:, t], nbins=32)
            assert abs(mom[t, j] - q[j][:, t].mean()) < 1e-11 * max(1.0, abs(mean))               # same average ...
            assert abs(mom[t, j] - exact[j]) < 4.5 * se + 1e-12, (t, j, mom[t, j], exact[j], se)   # ... equal to the exact one


def test_j0_closed_forms_specific_heat_and_magnetisation_moments(oracle_mod):
    # J = 0, bimodal field: spins are independent, s_i = h_i * sigma_i with <sigma> = t = tanh(beta h).
    #   <e> = -h t;  Var(E_total) = N h^2 (1 - t^2)  =>  C = N/T^2 (<e^2> - <e>^2) = (beta h)^2 (1 - t^2)   (Eq. 12)
    #   m = mu + X, mu = t (N+ - N-)/N, X centred: E X^2 = v/N, E X^3 = -2 t v (N+ - N-)/N^3, E X^4 = (v (1 + 3 t^2) + 3 (N-1) v^2)/N^3, v = 1 - t^2
    L, h, T = 4, 0.9, np.array([1.1, 2.3])
    N = L ** 3
    o = oracle_mod.Oracle(L, 2, 0.0, h, 0, 5)
    o.set_temperatures(T)
    f = o.get_field().astype(np.float64)
    dn = (f > 0).sum() - (f < 0).sum()
    o.sweep(60000, 0 + 3)                       # exchanges are harmless at J = 0 only if ... they are: PT keeps each marginal
    skip = 1000
    mom = o.thermal_moments(skip)
    q = _series_quantities(o, h, skip)
    absM, C, g = oracle_mod.thermal_observables(mom, T, N)
    for t in range(2):
        b = 1.0 / T[t]
        th = np.tanh(b * h); v = 1.0 - th * th
        mu = th * dn / N
        ex2, ex3, ex4 = v / N, -2.0 * th * v * dn / N ** 3, (v * (1 + 3 * th * th) + 3 * (N - 1) * v * v) / N ** 3
        m2 = mu * mu + ex2
        m4 = mu ** 4 + 6 * mu * mu * ex2 + 4 * mu * ex3 + ex4
        for j, exact in ((0, -h * th), (3, m2), (4, m4)):
            _, se = binned_mean_se(q[j][:, t], nbins=32)
            assert abs(mom[t, j] - exact) < 4.5 * se, (t, j, mom[t, j], exact, se)
        # specific heat: error from the binned variance estimates of e and e^2 (dominated by e^2 - <e>^2 fluctuations)
        c_exact = (b * h) ** 2 * v
        e = q[0][:, t]
        cs = np.array([N / T[t] ** 2 * chunk.var() for chunk in np.array_split(e, 32)])
        assert abs(C[t] - c_exact) < 4.5 * cs.std(ddof=1) / np.sqrt(32) + 0.01 * c_exact, (C[t], c_exact)


def test_binder_and_disorder_average_limits(oracle_mod):
    # Eq. 13: fully ordered (m = +-1 always) -> g = 1; Gaussian m (<m^4> = 3 <m^2>^2) -> g = 0;
    # the ratio is taken of the disorder AVERAGES: two realisations with <m^2> = 0.2 / 0.6 and <m^4> = 0.1 / 0.5
    # give g = (3 - 0.3 / 0.16) / 2, not the mean of the two per-realisation factors.
    T = np.array([2.0])
    ordered = np.array([[[-3.0, 9.0, 1.0, 1.0, 1.0]]])
    absM, C, g = oracle_mod.thermal_observables(ordered, T, 64)
    assert g[0] == 1.0 and absM[0] == 1.0 and C[0] == 0.0
    gauss = np.array([[[-1.0, 1.5, 0.3, 0.25, 3 * 0.25 ** 2]]])
    absM, C, g = oracle_mod.thermal_observables(gauss, T, 64)
    assert abs(g[0]) < 1e-15 and abs(C[0] - 64 / 4.0 * 0.5) < 1e-12
    two = np.array([[[0.0, 0.0, 0.4, 0.2, 0.1]], [[0.0, 0.0, 0.7, 0.6, 0.5]]])
    absM, C, g = oracle_mod.thermal_observables(two, T, 64)
    assert abs(g[0] - 0.5 * (3 - 0.3 / 0.16)) < 1e-15 and abs(absM[0] - 0.55) < 1e-15
