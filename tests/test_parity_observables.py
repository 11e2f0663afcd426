"""-m gpu: thermal moments and the observables of PAPER.md:249-260 (Eq. 11-13) from the device time series against the
oracle.  The two series are identical integers (the trajectories are bit-exact), the energies per site are the same
binary64 values, so only the order of the sums differs: a mean of `cnt` terms bounded by X differs from the sequential
sum by at most ~cnt * 2^-53 * X; the tolerance below is 1e-11 * X for cnt <= 10^4.  C subtracts <e>^2 from <e^2>, so its
tolerance is N/T^2 * 2e-11 * max(e^2)."""
import numpy as np
import pytest

from parity_util import make_pair
from paper_1508_06268_b200.workloads import geometric_ladder

pytestmark = pytest.mark.gpu

BIMODAL, GAUSSIAN = 0, 1


@pytest.mark.parametrize("L,R,kind,h", [(16, 8, GAUSSIAN, 1.0), (8, 6, BIMODAL, 1.0), (32, 4, BIMODAL, 2.0)])
def test_thermal_moments_match_oracle(L, R, kind, h):
    T = geometric_ladder(1.0, 5.0, R)
    g, o = make_pair(L, R, 1.0, h, kind, 3, T)
    g.sweep(1500, 5); o.sweep(1500, 5)
    for skip in (0, 60, 299):
        a, b = g.thermal_moments(skip), o.thermal_moments(skip)
        scale = np.array([3.0 + 8 * h, (3.0 + 8 * h) ** 2, 1.0, 1.0, 1.0])
        assert np.all(np.abs(a - b) <= 1e-11 * scale), (skip, np.abs(a - b).max(axis=0))
    import oracle
    absM, C, bg = g.thermal_observables(60)
    oM, oC, og = oracle.thermal_observables(o.thermal_moments(60), T, L ** 3)
    assert np.all(np.abs(absM - oM) <= 1e-11)
    assert np.all(np.abs(C - oC) <= (L ** 3 / T ** 2) * 2e-11 * (3.0 + 8 * h) ** 2)
    assert np.all(np.abs(bg - og) <= 1e-9)
    g.close()


def test_disorder_averaged_observables_match_oracle():
    import oracle
    from paper_1508_06268_b200 import binding
    L, R, seeds = 8, 5, [21, 22, 23, 24]
    T = geometric_ladder(1.5, 5.0, R)
    g = binding.RfimPT(L, R, 1.0, 1.0, GAUSSIAN, seeds=seeds)
    g.set_temperatures(T)
    g.sweep(1000, 4)
    moms = []
    for d, seed in enumerate(seeds):
        o = oracle.Oracle(L, R, 1.0, 1.0, GAUSSIAN, seed)
        o.set_temperatures(T)
        o.sweep(1000, 4)
        moms.append(o.thermal_moments(50))
        assert np.all(np.abs(g.thermal_moments(50, d=d) - moms[-1]) <= 1e-10)
    absM, C, bg = g.thermal_observables(50)
    oM, oC, og = oracle.thermal_observables(moms, T, L ** 3)
    assert np.all(np.abs(absM - oM) <= 1e-11) and np.all(np.abs(bg - og) <= 1e-9)
    assert np.all(np.abs(C - oC) <= (L ** 3 / T ** 2) * 1e-9)
    # the specific heat is positive and the Binder factor lies in [0, 1] up to noise; |M| decreases with T
    assert np.all(C > 0) and np.all(bg < 1.0 + 1e-12) and absM[0] > absM[-1]
    g.close()


def test_thermal_moments_errors():
    from paper_1508_06268_b200 import binding
    g = binding.RfimPT(8, 3, 1.0, 1.0, BIMODAL, seed=1)
    g.set_temperatures([1.0, 2.0, 3.0])
    with pytest.raises(binding.RfimPtError) as e:
        g.thermal_moments(0)                       # nothing recorded yet
    assert e.value.code == binding.ESTATE
    g.sweep(10, 5)
    assert g.thermal_moments(1).shape == (3, 5)
    with pytest.raises(binding.RfimPtError):
        g.thermal_moments(2)                       # skip == steps
    g.close()
