"""-m gpu: bit-packed storage (rfim_pt_set_packing(1), SURVEY.md 8(b)/(c) "int8 == bit-packed").

One bit per spin in device memory; the resident kernel expands a run into shared memory at load and packs it at
store (boundary rows are published packed too).  Every result -- spins, integer energies, permutation, time series --
must equal the oracle's, hence the byte layout's, bit for bit.
"""
import numpy as np
import pytest

from parity_util import assert_same_series, assert_same_state, make_pair
from paper_1508_06268_b200.workloads import geometric_ladder, linear_ladder

pytestmark = pytest.mark.gpu

BIMODAL, GAUSSIAN = 0, 1


@pytest.mark.parametrize("L,R,grid,partition", [(32, 5, 0, 1), (32, 5, 7, 1), (64, 3, 0, 1), (64, 3, 5, 1), (32, 5, 0, 2), (32, 5, 3, 0)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_packed_storage_bit_exact(L, R, grid, partition, kind, h):
    """pack at the start, sweep with exchanges in several launch shapes, compare everything with the oracle."""
    T = geometric_ladder(0.9, 5.5, R)
    g, o = make_pair(L, R, 1.0, h, kind, 23, T)
    g.set_packing(1)
    if grid:
        g.set_tuning(1, grid)
    g.set_tuning(2, partition)               # 1: equal runs of planes (seams, halos through L2); 2 / 0: whole replicas per CTA
    for r in range(R):                       # the conversion kept the initial state
        assert np.array_equal(g.get_spins_slot(r), o.get_spins_slot(r))
    for n, k in ((3, 0), (10, 5), (7, 2)):
        g.sweep(n, k); o.sweep(n, k)
        assert_same_state(g, o, what=f"packed L={L} grid={grid} after sweep({n},{k})")
    assert_same_series(g, o)
    assert g.diagnostics()["ulp_ambiguous"] == 0
    g.close()


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_packing_roundtrip_set_get_and_mixed_modes(kind):
    """8 -> 1 -> 8 keeps every spin; set/get work in packed mode; sweeping packed then unpacked follows the oracle."""
    L, R = 32, 4
    T = linear_ladder(1.0, 5.0, R)
    g, o = make_pair(L, R, 1.0, 1.5, kind, 5, T)
    rng = np.random.default_rng(7)
    lat = (rng.integers(0, 2, size=(R, L ** 3)) * 2 - 1).astype(np.int8)
    g.set_packing(1)
    for r in range(R):
        g.set_spins_slot(r, lat[r]); o.set_spins_slot(r, lat[r])
        assert np.array_equal(g.get_spins_slot(r), lat[r])
    g.sweep(6, 3); o.sweep(6, 3)
    assert_same_state(g, o, what="packed segment")
    g.set_packing(8)
    assert_same_state(g, o, what="after unpacking")
    g.sweep(5, 5); o.sweep(5, 5)
    assert_same_state(g, o, what="byte segment")
    g.set_packing(1)
    allspins = g.get_spins_all()
    for r in range(R):
        assert np.array_equal(allspins[0, r], o.get_spins_slot(r))
    g.set_spins_all(allspins)
    g.sweep(4, 2); o.sweep(4, 2)
    assert_same_state(g, o, what="packed again")
    g.close()


def test_packed_batch_and_adaptation():
    """batch members and the growing adaptation (copy of a lattice into a pool slot) in packed mode."""
    import oracle
    from paper_1508_06268_b200 import binding
    L, R, n = 32, 8, 5
    seeds = [101, 102, 103]
    T = geometric_ladder(1.0, 5.0, n)
    g = binding.RfimPT(L, R, 1.0, 1.5, GAUSSIAN, seeds=seeds)
    g.set_packing(1)
    g.set_temperatures(T)
    g.set_adapt_params(5, 2)
    g.adapt_temperatures(20)
    g.sweep(10, 5)
    for d, seed in enumerate(seeds):
        o = oracle.Oracle(L, R, 1.0, 1.5, GAUSSIAN, seed)
        o.set_temperatures(T)
        o.set_adapt_params(5, 2)
        o.adapt_temperatures(20)
        o.sweep(10, 5)
        assert np.array_equal(g.get_temperatures(d=d), o.get_temperatures())
        assert_same_state(g, o, d=d, what=f"packed batch member {d}")
    g.close()


def test_packing_errors():
    from paper_1508_06268_b200 import binding
    g = binding.RfimPT(16, 4, 1.0, 1.0, BIMODAL, seed=1)
    with pytest.raises(binding.RfimPtError) as e:
        g.set_packing(1)                     # L = 16: no resident kernel
    assert e.value.code == binding.EINVAL
    with pytest.raises(binding.RfimPtError):
        g.set_packing(4)
    g.close()
    g = binding.RfimPT(32, 4, 1.0, 1.0, BIMODAL, seed=1)
    g.set_kernel_variant(3)
    with pytest.raises(binding.RfimPtError):
        g.set_packing(1)                     # the flow kernel reads bytes
    g.set_kernel_variant(0)
    g.set_packing(1)
    with pytest.raises(binding.RfimPtError):
        g.set_kernel_variant(2)
    g.close()


def test_bit_packed_host_interface_roundtrip():
    """rfim_pt_get/set_spins_all_bits: natural-order bits on the host, both device storage modes, against the int8 getters."""
    from paper_1508_06268_b200 import binding
    for L, packing in ((8, 8), (12, 8), (16, 8), (32, 8), (32, 1), (64, 8), (64, 1)):
        g = binding.RfimPT(L, 3, 1.0, 1.0, BIMODAL, seeds=[5, 6])
        if packing == 1:
            g.set_packing(1)
        ref = g.get_spins_all()                                   # [D][R][N] of +-1
        bits = g.get_spins_all_bits()
        assert bits.shape == (2, 3, L ** 3 // 8)
        assert np.array_equal(np.unpackbits(bits, axis=-1, bitorder="little"), (ref > 0).astype(np.uint8))
        rng = np.random.default_rng(L + packing)
        new = rng.integers(0, 2, size=ref.shape, dtype=np.uint8)
        g.set_spins_all_bits(np.ascontiguousarray(np.packbits(new, axis=-1, bitorder="little")))
        assert np.array_equal(g.get_spins_all(), (2 * new.astype(np.int8) - 1))
        assert np.array_equal(g.get_spins_all_bits(), np.packbits(new, axis=-1, bitorder="little"))
        g.close()


def test_observables_reuse_the_in_kernel_measurement():
    """after a call that ends on an exchange step the getters return the terms measured inside the sweep kernel; after
    anything that touches the lattices they reduce again: both must equal the oracle's recomputed Hamiltonian."""
    T = geometric_ladder(1.0, 4.0, 4)
    g, o = make_pair(32, 4, 1.0, 1.5, GAUSSIAN, 8, T)
    g.sweep(10, 5); o.sweep(10, 5)                                 # ends on a step: cached terms
    for a, b in zip(g.get_energy_terms(), o.get_energy_terms()):
        assert np.array_equal(a, b)
    E, M, _ = g.observables(); Eo, Mo, _ = o.observables()
    assert np.array_equal(E, Eo) and np.array_equal(M, Mo)
    g.sweep(3, 5); o.sweep(3, 5)                                   # does not end on a step: fresh reduction
    for a, b in zip(g.get_energy_terms(), o.get_energy_terms()):
        assert np.array_equal(a, b)
    g.sweep(2, 5); o.sweep(2, 5)                                   # on a step again, then overwrite one lattice
    s = -g.get_spins_slot(1)
    g.set_spins_slot(1, s); o.set_spins_slot(1, s)
    for a, b in zip(g.get_energy_terms(), o.get_energy_terms()):
        assert np.array_equal(a, b)
    g.close()
