"""-m gpu: the CUDA path against the oracle, element by element, at sizes that span several tiles
and ragged tails, plus the method's edge cases.  Bit-exact everywhere (integer work)."""
import numpy as np
import pytest

from parity_util import assert_same_series, assert_same_state, make_pair

pytestmark = pytest.mark.gpu

BIMODAL, GAUSSIAN = 0, 1


@pytest.mark.parametrize("L", [2, 4, 6, 8, 10, 16, 24])
@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_initial_state_field_and_tables(L, kind):
    R = 5
    T = np.linspace(0.9, 4.1, R)
    g, o = make_pair(L, R, 1.0, 1.5, kind, 1000 + L, T)
    assert np.array_equal(g.get_field(), o.get_field())
    assert_same_state(g, o, what="initial")
    if kind == BIMODAL:
        for t in range(R):
            for k in range(7):
                for b in range(2):
                    assert g.bimodal_threshold(t, k, b) == o.bimodal_threshold(t, k, b)
    Eg, Mg, _ = g.observables(); Eo, Mo, _ = o.observables()
    assert np.array_equal(Eg, Eo) and np.array_equal(Mg, Mo)


@pytest.mark.parametrize("L,R,variant", [(2, 3, 1), (4, 4, 1), (6, 5, 1), (8, 6, 1), (8, 6, 2), (10, 3, 1), (12, 4, 1),
                                         (16, 9, 2), (16, 9, 1), (24, 5, 2), (32, 3, 2), (40, 2, 2),
                                         # variant 5: one CTA per replica, whole lattice in shared memory, one launch per exchange period
                                         (8, 6, 5), (16, 9, 5), (24, 5, 5), (32, 3, 5), (40, 2, 5)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 1.0), (BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_sweeps_with_exchange_bit_exact(L, R, variant, kind, h):
    T = np.geomspace(0.8, 5.0, R)
    g, o = make_pair(L, R, 1.0, h, kind, 7 * L + R, T)
    g.set_kernel_variant(variant)
    for chunk, k in [(1, 0), (6, 3), (5, 2), (8, 4)]:
        g.sweep(chunk, k); o.sweep(chunk, k)
        assert_same_state(g, o, what=f"L={L} after chunk {chunk},{k}")
    assert_same_series(g, o)
    d = g.diagnostics()
    assert d["ulp_ambiguous"] == 0 and d["launches"] > 0


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_site_and_word_kernels_agree(kind):
    T = np.linspace(1.0, 4.0, 4)
    a, o = make_pair(16, 4, 1.0, 1.0, kind, 99, T)
    b, _ = make_pair(16, 4, 1.0, 1.0, kind, 99, T)
    a.set_kernel_variant(1); b.set_kernel_variant(2)
    a.sweep(12, 4); b.sweep(12, 4)
    for r in range(4):
        assert np.array_equal(a.get_spins_slot(r), b.get_spins_slot(r))
    assert np.array_equal(a.get_permutation(), b.get_permutation())


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_extreme_temperatures(kind):
    # T -> 0 (thresholds 0: the "never" entries), T huge (thresholds 2^32 - tiny), and both in one ladder
    T = np.array([1e-30, 1e-3, 0.05, 1.0, 1e3, 1e30])
    g, o = make_pair(8, 6, 1.0, 1.3, kind, 5, T)
    for _ in range(3):
        g.sweep(4, 2); o.sweep(4, 2)
        assert_same_state(g, o, what="extreme T")
    E, _, _ = g.observables()


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_zero_couplings_flip_everything(kind):
    g, o = make_pair(8, 3, 0.0, 0.0, kind, 9, [0.5, 1.0, 1e30])
    before = [g.get_spins_slot(r).copy() for r in range(3)]
    g.sweep(1, 0); o.sweep(1, 0)
    for r in range(3):
        assert np.array_equal(g.get_spins_slot(r), -before[r])
    assert_same_state(g, o)


def test_degenerate_shapes():
    # one temperature (no pair), one slot, R > n, zero sweeps, exchange_every larger than the run
    g, o = make_pair(8, 1, 1.0, 1.0, BIMODAL, 3, [2.0])
    g.sweep(5, 1); o.sweep(5, 1)
    assert_same_state(g, o, what="R=1")
    assert_same_series(g, o)
    g, o = make_pair(8, 6, 1.0, 1.0, GAUSSIAN, 4, [1.5, 2.5])          # n = 2 < R = 6
    g.sweep(0, 5); o.sweep(0, 5)
    g.sweep(7, 100); o.sweep(7, 100)
    g.sweep(6, 1); o.sweep(6, 1)
    assert_same_state(g, o, what="n<R")
    assert_same_series(g, o)


def test_error_codes():
    from paper_1508_06268_b200 import binding
    with pytest.raises(binding.RfimPtError):
        binding.RfimPT(7, 2, 1.0, 1.0, 0, seed=1)                     # odd L
    with pytest.raises(binding.RfimPtError):
        binding.RfimPT(8, 0, 1.0, 1.0, 0, seed=1)                     # R < 1
    with pytest.raises(binding.RfimPtError):
        binding.RfimPT(8, 2, 1.0, 1.0, 5, seed=1)                     # field kind
    g = binding.RfimPT(8, 2, 1.0, 1.0, 0, seed=1)
    with pytest.raises(binding.RfimPtError) as e:
        g.sweep(1, 1)
    assert e.value.code == binding.ESTATE
    for bad in ([2.0, 1.0], [1.0, 1.0], [-1.0, 2.0], [1.0, 2.0, 3.0], []):
        with pytest.raises(binding.RfimPtError) as e:
            g.set_temperatures(bad)
        assert e.value.code == binding.EINVAL
    g.set_temperatures([1.0, 2.0])
    with pytest.raises(binding.RfimPtError):
        g.sweep(-1, 1)
    with pytest.raises(binding.RfimPtError):
        g.get_spins(2)
    with pytest.raises(binding.RfimPtError):
        g.set_spins_slot(0, np.zeros(512, dtype=np.int8))             # not +-1


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_set_get_roundtrip_and_mirror_symmetry(kind):
    from paper_1508_06268_b200.workloads import random_spins
    L, R = 8, 4
    T = np.linspace(3.0, 4.2, R)
    a, o = make_pair(L, R, 1.0, 1.5, kind, 2718, T)
    b, _ = make_pair(L, R, 1.0, 1.5, kind, 2718, None)
    s = random_spins(L, 11)
    a.set_spins_slot(2, s); o.set_spins_slot(2, s)
    assert np.array_equal(a.get_spins_slot(2), s)
    allspins = a.get_spins_all()
    assert np.array_equal(allspins[0, 2], s)
    b.set_field(-a.get_field())
    b.set_spins_all(np.ascontiguousarray(-allspins))
    b.set_temperatures(T)
    for _ in range(4):
        a.sweep(6, 3); b.sweep(6, 3); o.sweep(6, 3)
        assert_same_state(a, o, what="mirror/a")
        assert np.array_equal(a.get_permutation(), b.get_permutation())
        assert np.array_equal(a.get_spins_all(), -b.get_spins_all())
        Ea, Ma, _ = a.observables(); Eb, Mb, _ = b.observables()
        assert np.array_equal(Ea, Eb) and np.array_equal(Ma, -Mb)


def test_calls_compose_and_snapshot_restart():
    T = np.linspace(1.0, 4.0, 5)
    a, _ = make_pair(8, 5, 1.0, 1.0, GAUSSIAN, 42, T)
    b, _ = make_pair(8, 5, 1.0, 1.0, GAUSSIAN, 42, T)
    a.sweep(20, 10)
    b.sweep(7, 10); b.sweep(13, 10)
    assert np.array_equal(a.get_spins_all(), b.get_spins_all())
    assert np.array_equal(a.get_permutation(), b.get_permutation()) and a.get_counters() == b.get_counters() == (20, 2)
    # restart a third handle from a's snapshot
    c, o = make_pair(8, 5, 1.0, 1.0, GAUSSIAN, 42, T)
    c.set_spins_all(a.get_spins_all()); c.set_permutation(a.get_permutation()); c.set_counters(*a.get_counters())
    for r in range(5):
        o.set_spins_slot(r, a.get_spins_slot(r))
    o.set_permutation(a.get_permutation()); o.set_counters(*a.get_counters())
    a.sweep(10, 5); c.sweep(10, 5); o.sweep(10, 5)
    assert np.array_equal(a.get_spins_all(), c.get_spins_all())
    assert np.array_equal(a.get_permutation(), c.get_permutation())
    assert np.array_equal(a.get_permutation(), o.get_permutation())
    for r in range(5):
        assert np.array_equal(a.get_spins_slot(r), o.get_spins_slot(r))


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_batch_member_equals_single_handle(kind):
    from paper_1508_06268_b200 import binding
    import oracle
    seeds = [1000, 1001, 1002]
    T = np.geomspace(1.0, 6.0, 4)
    batch = binding.RfimPT(8, 4, 1.0, 1.5, kind, seeds=seeds)
    batch.set_temperatures(T)
    batch.sweep(12, 3)
    for d, sd in enumerate(seeds):
        o = oracle.Oracle(8, 4, 1.0, 1.5, kind, sd)
        o.set_temperatures(T); o.sweep(12, 3)
        assert np.array_equal(batch.get_field(d=d), o.get_field())
        assert_same_state(batch, o, d=d, what=f"member {d}")
        assert_same_series(batch, o, d=d)
    E, M, rate = batch.observables()
    assert E.shape == (3, 4) and rate.shape == (3, 3)


@pytest.mark.parametrize("grow", [True, False])
def test_adaptation_matches_oracle(grow):
    L, k, a, trial = 8, 2, 3, 200
    R = 14 if grow else 8
    T0 = np.linspace(0.8, 6.0, 8)
    g, o = make_pair(L, R, 1.0, 2.0, BIMODAL, 3, T0)
    g.set_adapt_params(k, a); o.set_adapt_params(k, a)
    for rnd in range(3):
        g.adapt_temperatures(trial); o.adapt_temperatures(trial)
        assert np.array_equal(g.get_temperatures(), o.get_temperatures()), rnd
        assert_same_state(g, o, what=f"adapt round {rnd}")
    assert g.n == (14 if grow else 8)
    g.sweep(20, k); o.sweep(20, k)
    assert_same_state(g, o, what="after adapt")
    assert_same_series(g, o)


# ---- the tuned persistent "flow" kernel (variant 3; L = 32 or 64) ---------------------------------------
@pytest.mark.parametrize("L,R", [(32, 5), (64, 3)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_flow_kernel_bit_exact(L, R, kind, h):
    T = np.geomspace(0.8, 5.0, R)                    # R is not a multiple of the replica group size
    g, o = make_pair(L, R, 1.0, h, kind, 31 * L + R, T)
    g.set_kernel_variant(3)
    for chunk, k in [(1, 0), (4, 2), (3, 3), (7, 5)]:
        g.sweep(chunk, k); o.sweep(chunk, k)
        assert_same_state(g, o, what=f"flow L={L} after chunk {chunk},{k}")
    assert_same_series(g, o)
    d = g.diagnostics()
    assert d["ulp_ambiguous"] == 0


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_flow_kernel_extreme_temperatures_and_long_launch(kind):
    # thresholds 0 (the "never" table entries) and ~2^32; 130 sweeps without exchange = two launches (127 + 3)
    T = np.array([1e-30, 0.05, 1.0, 1e3, 1e30])
    g, o = make_pair(32, 5, 1.0, 1.3, kind, 5, T)
    g.set_kernel_variant(3)
    g.sweep(6, 2); o.sweep(6, 2)
    assert_same_state(g, o, what="flow extreme T")
    g.sweep(130, 0); o.sweep(130, 0)
    assert_same_state(g, o, what="flow 130 sweeps")


def test_flow_kernel_batch_and_reference_kernels_agree():
    from paper_1508_06268_b200 import binding
    seeds = [11, 12, 13]
    T = np.geomspace(1.0, 6.0, 6)
    a = binding.RfimPT(32, 6, 1.0, 1.5, GAUSSIAN, seeds=seeds); a.set_kernel_variant(3)
    b = binding.RfimPT(32, 6, 1.0, 1.5, GAUSSIAN, seeds=seeds); b.set_kernel_variant(2)
    a.set_temperatures(T); b.set_temperatures(T)
    a.sweep(12, 4); b.sweep(12, 4)
    assert np.array_equal(a.get_spins_all(), b.get_spins_all())
    for d in range(3):
        assert np.array_equal(a.get_permutation(d=d), b.get_permutation(d=d))
        for x, y in zip(a.get_timeseries(d=d), b.get_timeseries(d=d)):
            assert np.array_equal(x, y)


# ---- the shared-memory-resident kernel (variant 4; L = 32 or 64) ------------------------------------------
@pytest.mark.parametrize("L,R,grid,partition", [(32, 5, 0, 1), (32, 5, 7, 1), (32, 3, 148, 1), (64, 3, 0, 1), (64, 3, 5, 1), (64, 2, 4, 1),
                                                # whole replicas per CTA (the automatic choice for small problems): one, two, ragged last CTA
                                                (32, 5, 0, 2), (32, 5, 3, 2), (32, 7, 2, 2), (32, 5, 0, 0)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_resident_kernel_bit_exact(L, R, grid, partition, kind, h):
    # equal runs (partition 1): grid limits force runs of many planes per CTA, runs that cross replica seams, odd plane
    # counts (ragged last 32-row block at L = 32) and the one-plane-per-CTA extreme.  Partition 2: whole replicas per CTA.
    T = np.geomspace(0.8, 5.0, R)
    g, o = make_pair(L, R, 1.0, h, kind, 31 * L + R, T)
    g.set_kernel_variant(4)
    g.set_tuning(1, grid)
    g.set_tuning(2, partition)
    for chunk, k in [(1, 0), (4, 2), (3, 3), (7, 5)]:
        g.sweep(chunk, k); o.sweep(chunk, k)
        assert_same_state(g, o, what=f"resident L={L} grid={grid} after chunk {chunk},{k}")
    assert_same_series(g, o)
    d = g.diagnostics()
    assert d["ulp_ambiguous"] == 0


@pytest.mark.parametrize("L,R,grid,partition", [(32, 5, 7, 1), (32, 3, 148, 1), (64, 3, 5, 1), (64, 2, 0, 1), (32, 5, 3, 2), (32, 7, 0, 0)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 2.0), (GAUSSIAN, 1.5)])
def test_resident_kernel_several_moves_per_launch(L, R, grid, partition, kind, h):
    """One launch of the resident kernel holds every exchange period that fits in 127 sweeps (the run stays in shared memory,
    the exchange steps run inside the kernel behind a grid-wide rendezvous): calls that start off a period boundary, end on
    one or past one, and a call long enough to need two launches -- against the oracle and against one launch per move."""
    T = np.geomspace(0.8, 5.0, R)
    g, o = make_pair(L, R, 1.0, h, kind, 17 * L + R, T)
    g1, _ = make_pair(L, R, 1.0, h, kind, 17 * L + R, T)
    for x in (g, g1):
        x.set_kernel_variant(4)
        x.set_tuning(1, grid)
        x.set_tuning(2, partition)
    g1.set_tuning(3, 0)                                            # one launch per move
    for chunk, k in [(2, 3), (13, 3), (20, 5), (9, 4), (133, 7)]:
        l0 = g.diagnostics()["launches"]
        g.sweep(chunk, k)
        if (chunk, k) == (20, 5):
            assert g.diagnostics()["launches"] - l0 == 1           # four exchange steps, one launch
        g1.sweep(chunk, k); o.sweep(chunk, k)
        assert_same_state(g, o, what=f"several moves per launch, L={L} grid={grid} after chunk {chunk},{k}")
        assert_same_state(g1, o, what=f"one move per launch, L={L} grid={grid} after chunk {chunk},{k}")
    assert_same_series(g, o)
    assert_same_series(g1, o)
    assert g.diagnostics()["ulp_ambiguous"] == 0
    g.close(); g1.close(); o.close()


@pytest.mark.parametrize("L,R", [(8, 6), (16, 9), (24, 5)])
@pytest.mark.parametrize("kind,h", [(BIMODAL, 1.0), (GAUSSIAN, 1.5)])
def test_small_lattice_kernel_several_moves_per_launch(L, R, kind, h):
    """The one-CTA-per-replica kernel also keeps the lattices in shared memory across exchange periods (a cooperative launch, the
    exchange steps inside it): against the oracle and against one launch per move, with calls that start off a period boundary."""
    T = np.geomspace(0.8, 5.0, R)
    g, o = make_pair(L, R, 1.0, h, kind, 13 * L + R, T)
    g1, _ = make_pair(L, R, 1.0, h, kind, 13 * L + R, T)
    g.set_kernel_variant(5); g1.set_kernel_variant(5)
    g1.set_tuning(3, 0)                                            # one launch per move
    for chunk, k in [(2, 3), (13, 3), (20, 5), (9, 4), (133, 7)]:
        l0 = g.diagnostics()["launches"]
        g.sweep(chunk, k)
        if (chunk, k) == (20, 5):
            assert g.diagnostics()["launches"] - l0 == 1           # four exchange steps, one launch
        g1.sweep(chunk, k); o.sweep(chunk, k)
        assert_same_state(g, o, what=f"small kernel, several moves per launch, L={L} after chunk {chunk},{k}")
        assert_same_state(g1, o, what=f"small kernel, one move per launch, L={L} after chunk {chunk},{k}")
    assert_same_series(g, o)
    assert_same_series(g1, o)
    g.close(); g1.close(); o.close()


@pytest.mark.parametrize("kind", [BIMODAL, GAUSSIAN])
def test_resident_kernel_extreme_temperatures_and_long_launch(kind):
    T = np.array([1e-30, 0.05, 1.0, 1e3, 1e30])
    g, o = make_pair(32, 5, 1.0, 1.3, kind, 5, T)
    g.set_kernel_variant(4)
    g.set_tuning(1, 11)
    g.set_tuning(2, 1)
    g.sweep(6, 2); o.sweep(6, 2)
    assert_same_state(g, o, what="resident extreme T")
    g.sweep(130, 0); o.sweep(130, 0)
    assert_same_state(g, o, what="resident 130 sweeps")


def test_resident_kernel_batch_n_less_than_R_and_flow_kernel_agree():
    from paper_1508_06268_b200 import binding
    seeds = [11, 12, 13]
    T = np.geomspace(1.0, 6.0, 5)                                      # n = 5 < R = 6
    a = binding.RfimPT(32, 6, 1.0, 1.5, GAUSSIAN, seeds=seeds); a.set_kernel_variant(4); a.set_tuning(1, 9); a.set_tuning(2, 1)
    b = binding.RfimPT(32, 6, 1.0, 1.5, GAUSSIAN, seeds=seeds); b.set_kernel_variant(3)
    a.set_temperatures(T); b.set_temperatures(T)
    a.sweep(12, 4); b.sweep(12, 4)
    assert np.array_equal(a.get_spins_all(), b.get_spins_all())
    for d in range(3):
        assert np.array_equal(a.get_permutation(d=d), b.get_permutation(d=d))
        for x, y in zip(a.get_timeseries(d=d), b.get_timeseries(d=d)):
            assert np.array_equal(x, y)
