"""Gaussian sampler moments, bimodal balance, and the h = 0 pure-Ising susceptibility peak."""
import numpy as np
from scipy import stats as sps

from stats import binned_mean_se


def test_gaussian_field_is_standard_normal(oracle_mod):
    o = oracle_mod.Oracle(24, 1, 1.0, 1.0, 1, 2)
    g = o.get_field().astype(np.float64) * 2.0 ** -20
    n = g.size
    assert abs(g.mean()) < 4 / np.sqrt(n)
    assert abs(g.var() - 1.0) < 4 * np.sqrt(2.0 / n)
    assert abs(sps.kurtosis(g, fisher=False) - 3.0) < 4 * np.sqrt(24.0 / n)
    assert abs(sps.skew(g)) < 4 * np.sqrt(6.0 / n)
    assert sps.kstest(g, "norm").pvalue > 1e-3
    assert np.abs(o.get_field()).max() <= 8 * 2 ** 20
    # sites are independent: lag-1 correlation along x is noise
    assert abs(np.corrcoef(g[:-1], g[1:])[0, 1]) < 4 / np.sqrt(n)


def test_bimodal_field_is_fair_pm1(oracle_mod):
    o = oracle_mod.Oracle(24, 1, 1.0, 1.0, 0, 3)
    f = o.get_field()
    assert set(np.unique(f)) == {-1, 1}
    assert abs(f.mean()) < 4 / np.sqrt(f.size)          # p = 1/2 ("h_i = rand(+-1)")
    o2 = oracle_mod.Oracle(24, 1, 1.0, 1.0, 0, 4)
    assert abs(np.mean(f * o2.get_field())) < 4 / np.sqrt(f.size)   # different seeds: independent fields


def test_pure_ising_susceptibility_peak_near_tc(oracle_mod):
    # north_star: "the h=0 limit reproducing the pure 3D Ising susceptibility peak near T ~ 4.51".
    # chi = N (<m^2> - <|m|>^2) / T on L = 8; the finite-size peak sits slightly above T_c = 4.5115.
    L = 8
    T = np.array([3.3, 3.7, 4.1, 4.4, 4.7, 5.0, 5.4, 5.9, 6.5])
    o = oracle_mod.Oracle(L, len(T), 1.0, 0.0, 0, 7, threads=2)
    o.set_temperatures(T)
    o.sweep(2000, 5)
    o.set_temperatures(T)
    o.sweep(30000, 5)
    _, _, Ms = o.get_timeseries()
    m = Ms.astype(np.float64) / L ** 3
    chi = L ** 3 * ((m ** 2).mean(axis=0) - np.abs(m).mean(axis=0) ** 2) / T
    peak = T[int(np.argmax(chi))]
    assert 4.3 <= peak <= 5.1, (peak, chi)
    assert chi.max() > 3 * chi[0] and chi.max() > 3 * chi[-1]
    # ordered below, disordered above
    assert np.abs(m).mean(axis=0)[0] > 0.85 and np.abs(m).mean(axis=0)[-1] < 0.25
    # energy per site at T = 3.3, 6.5 against high/low-T sanity: monotone increasing with T
    Eb, _, _ = o.get_timeseries()
    e = (-Eb.astype(np.float64) / L ** 3).mean(axis=0)
    assert np.all(np.diff(e) > 0)
