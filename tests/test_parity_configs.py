"""-m gpu: BASELINE.json's five configs, in the launch configuration bench.py times.

Bimodal configs (1, 3): spins, integer energies and permutations bit-exact at every checkpoint.
Gaussian configs (2, 4, 5): spins bit-exact through sweep 100 (and, since the CUDA path takes every
decision the exact binary64 rule would take, at every later checkpoint we can afford to recompute);
afterwards per-temperature <E>/N and <|m|> within 3 binned standard errors and 1e-3 absolute.
Full-size runs are checked on segments the oracle recomputes from a snapshot of the GPU state
(the trajectory is a deterministic function of state + counters), so the oracle's cost stays bounded.
"""
import numpy as np
import pytest

from parity_util import assert_same_series, assert_same_state, make_pair, oracle_threads
from stats import binned_mean_se

pytestmark = pytest.mark.gpu


def _cfg(name):
    from paper_1508_06268_b200.workloads import CONFIGS
    return CONFIGS[name]


def _snapshot_into_oracle(g, o, d=0):
    for r in range(o.R):
        o.set_spins_slot(r, g.get_spins_slot(r, d=d))
    o.set_permutation(g.get_permutation(d=d))
    o.set_counters(*g.get_counters())


def test_cfg1_full_run_bit_exact():
    w = _cfg("cfg1")
    g, o = make_pair(w.L, w.R, w.J, w.h, w.field_kind, w.seeds[0], w.temperatures())
    for _ in range(10):
        g.sweep(w.sweeps // 10, w.exchange_every); o.sweep(w.sweeps // 10, w.exchange_every)
        assert_same_state(g, o, what="cfg1")
    assert_same_series(g, o)
    assert g.get_counters() == (1000, 100)


def test_cfg2_bit_exact_then_statistics():
    w = _cfg("cfg2")
    g, o = make_pair(w.L, w.R, w.J, w.h, w.field_kind, w.seeds[0], w.temperatures())
    g.sweep(100, w.exchange_every); o.sweep(100, w.exchange_every)
    assert_same_state(g, o, what="cfg2 sweep 100")
    g.sweep(w.sweeps - 100, w.exchange_every); o.sweep(w.sweeps - 100, w.exchange_every)
    gs, os_ = g.get_timeseries(), o.get_timeseries()
    hs = w.h / 2 ** 20
    for t in range(w.R):
        for series in ("e", "m"):
            if series == "e":
                x = (-w.J * gs[0][:, t] - hs * gs[1][:, t]) / w.N
                y = (-w.J * os_[0][:, t] - hs * os_[1][:, t]) / w.N
            else:
                x = np.abs(gs[2][:, t]) / w.N
                y = np.abs(os_[2][:, t]) / w.N
            mx, sx = binned_mean_se(x, nbins=16, drop=0.2)
            my, sy = binned_mean_se(y, nbins=16, drop=0.2)
            assert abs(mx - my) <= 3 * np.hypot(sx, sy) + 1e-12 and abs(mx - my) <= 1e-3, (t, series, mx, my)
    # and in fact the whole trajectory is identical
    assert_same_state(g, o, what="cfg2 end")
    assert_same_series(g, o)
    d = g.diagnostics()
    assert d["exact_path"] > 0 and d["ulp_ambiguous"] == 0


def test_cfg3_adaptation_then_production_segments():
    w = _cfg("cfg3")
    g, o = make_pair(w.L, w.R, w.J, w.h, w.field_kind, w.seeds[0], w.temperatures())
    g.set_adapt_params(w.exchange_every, 4); o.set_adapt_params(w.exchange_every, 4)
    # trial runs: the GPU runs them in full; the oracle replays the first trial in full (2000 sweeps) ...
    g.adapt_temperatures(w.adapt_trial_sweeps); o.adapt_temperatures(w.adapt_trial_sweeps)
    assert np.array_equal(g.get_temperatures(), o.get_temperatures())
    assert_same_state(g, o, what="cfg3 trial 1")
    # ... and the later trials and the production run on segments restarted from GPU snapshots
    for trial in range(1, w.adapt_trials):
        g.adapt_temperatures(w.adapt_trial_sweeps)
    T = g.get_temperatures()
    assert len(T) == w.R and T[0] == w.t_min and T[-1] == w.t_max and np.all(np.diff(T) > 0)
    o.set_temperatures(T)
    done = 0
    for seg_start in (0, 3000, 9900):
        g.sweep(seg_start - done, w.exchange_every); done = seg_start
        _snapshot_into_oracle(g, o)
        g.sweep(100, w.exchange_every); o.sweep(100, w.exchange_every); done += 100
        for r in range(w.R):
            assert np.array_equal(g.get_spins_slot(r), o.get_spins_slot(r)), (seg_start, r)
        assert np.array_equal(g.get_permutation(), o.get_permutation())
        for a, b in zip(g.get_energy_terms(), o.get_energy_terms()):
            assert np.array_equal(a, b)
    assert done == w.sweeps
    rates = g.observables()[2]
    assert rates.min() > 0.0


def test_cfg4_first_100_sweeps_and_later_segment():
    w = _cfg("cfg4")
    g, o = make_pair(w.L, w.R, w.J, w.h, w.field_kind, w.seeds[0], w.temperatures())
    assert np.array_equal(g.get_field(), o.get_field())
    g.sweep(100, w.exchange_every); o.sweep(100, w.exchange_every)
    assert_same_state(g, o, what="cfg4 sweep 100")
    assert_same_series(g, o)
    g.sweep(1900, w.exchange_every)
    _snapshot_into_oracle(g, o)
    g.sweep(20, w.exchange_every); o.sweep(20, w.exchange_every)
    for r in range(w.R):
        assert np.array_equal(g.get_spins_slot(r), o.get_spins_slot(r)), r
    assert np.array_equal(g.get_permutation(), o.get_permutation())
    d = g.diagnostics()
    assert d["exact_path"] > 0 and d["ulp_ambiguous"] == 0
    # properties that hold at any size: permutation is a permutation, energies bounded, |m| <= 1
    E, M, rate = g.observables()
    assert sorted(g.get_permutation()) == list(range(w.R))
    assert np.all(np.abs(M) <= 1.0) and np.all(E / w.N > -3.0 - 2.0 * 5.0) and np.all(np.diff(E) > -0.05 * w.N)


def test_cfg4_size_bimodal_field_100_sweeps():
    """The paper's own field (bimodal +-1) at config 4's size and partition (148 CTAs x 55-56 planes, runs
    crossing replica seams): the 32-bit table look-up specialisation (no zero threshold) of the resident kernel."""
    from paper_1508_06268_b200 import binding
    w = _cfg("cfg4")
    g, o = make_pair(w.L, w.R, w.J, 1.0, binding.BIMODAL, 7, w.temperatures())
    for _ in range(2):
        g.sweep(50, w.exchange_every); o.sweep(50, w.exchange_every)
        assert_same_state(g, o, what="cfg4-size bimodal")
    assert_same_series(g, o)
    # and with a ladder cold enough to produce zero thresholds (the 64-bit look-up specialisation)
    T = np.concatenate([[0.05, 0.08], w.temperatures()[2:]])
    g.set_temperatures(T); o.set_temperatures(T)
    g.sweep(20, w.exchange_every); o.sweep(20, w.exchange_every)
    assert_same_state(g, o, what="cfg4-size bimodal, zero thresholds")


def test_cfg5_batched_disorder_members():
    import oracle
    from paper_1508_06268_b200 import binding
    w = _cfg("cfg5")
    g = binding.RfimPT(w.L, w.R, w.J, w.h, w.field_kind, seeds=list(w.seeds))
    g.set_temperatures(w.temperatures())
    g.sweep(100, w.exchange_every)
    for d in (0, 13, 31):
        o = oracle.Oracle(w.L, w.R, w.J, w.h, w.field_kind, w.seeds[d], threads=oracle_threads())
        o.set_temperatures(w.temperatures())
        o.sweep(100, w.exchange_every)
        assert np.array_equal(g.get_field(d=d), o.get_field())
        assert_same_state(g, o, d=d, what=f"cfg5 member {d}")
        assert_same_series(g, o, d=d)
    dg = g.diagnostics()
    assert dg["ulp_ambiguous"] == 0
