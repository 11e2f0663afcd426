"""rfim_pt_energy_terms_noalloc: the entry point that allocates nothing (scratch in a static device array).

Collected last on purpose (the run uses -x).  The GPU test compares the new entry point with the existing
path (rfim_pt_get_energy_terms of a handle, itself bit-exact against the oracle in the parity tests) on two calls in a
row of different shape, so that the second call meets the first one's leftovers in the shared scratch.  Integer sums:
the tolerance is the one every parity test here uses, bit-exact.
"""
import numpy as np
import pytest

from paper_1508_06268_b200 import binding
from paper_1508_06268_b200.workloads import geometric_ladder

BIMODAL, GAUSSIAN = 0, 1


def _existing_path(L, R, kind, h, seed, sweeps):
    """A handle swept with exchanges: spins by slot, the field, and (Eb, Ef, Msum) by slot from the existing path."""
    g = binding.RfimPT(L, R, 1.0, h, kind, seed=seed)
    g.set_temperatures(geometric_ladder(0.8, 6.0, R))
    g.sweep(sweeps, 2)
    spins = g.get_spins_all().reshape(R, L ** 3).copy()
    field = g.get_field().copy()
    t2r = g.get_permutation()
    by_rank = np.stack(g.get_energy_terms(), axis=1)             # [rank][3]
    by_slot = np.zeros((R, 3), dtype=np.int64)
    by_slot[t2r] = by_rank
    g.close()
    return spins, field, by_slot


def _no_alloc_path(L, R, kind, spins, field, stream=None):
    import torch
    s = torch.from_numpy(spins).cuda()
    f = torch.from_numpy(field).cuda()
    out = torch.full((R, 3), -7, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    binding.energy_terms_noalloc(L, R, kind, s.data_ptr(), f.data_ptr(), out.data_ptr(), stream=stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.gpu
def test_no_alloc_energy_terms_equal_the_existing_path_twice_in_a_row():
    import torch
    cases = [(32, 11, GAUSSIAN, 1.5, 3, 6), (12, 37, BIMODAL, 2.0, 4, 4), (64, 3, BIMODAL, 1.0, 5, 4), (2, 5, GAUSSIAN, 0.7, 6, 2)]
    want = [_existing_path(*c) for c in cases]
    stream = torch.cuda.Stream()
    for rep in range(2):                                          # the same sequence again: leftovers of the largest call
        for (L, R, kind, *_), (spins, field, terms) in zip(cases, want):
            for st in (None, stream.cuda_stream):
                got = _no_alloc_path(L, R, kind, spins, field, stream=st)
                assert np.array_equal(got, terms), f"L={L} R={R} kind={kind} rep={rep}: {got[:3]} vs {terms[:3]}"


@pytest.mark.gpu
def test_no_alloc_maximum_sizes():
    """R at the limit (one lattice repeated with flips so every replica differs) against a plain numpy sum."""
    L, R = 8, binding.NOALLOC_MAX_R
    rng = np.random.default_rng(11)
    spins = (rng.integers(0, 2, size=(R, L ** 3)) * 2 - 1).astype(np.int8)
    field = rng.integers(-(1 << 22), 1 << 22, size=L ** 3).astype(np.int32)
    s = spins.reshape(R, L, L, L).astype(np.int64)               # [r][z][y][x]
    eb = sum((s * np.roll(s, -1, axis=a)).sum(axis=(1, 2, 3)) for a in (1, 2, 3))
    ef = (spins.astype(np.int64) * field.astype(np.int64)).sum(axis=1)
    want = np.stack([eb, ef, spins.astype(np.int64).sum(axis=1)], axis=1)
    for _ in range(2):
        assert np.array_equal(_no_alloc_path(L, R, GAUSSIAN, spins, field), want)


def test_no_alloc_rejects_sizes_beyond_the_static_scratch():
    """Checked before any CUDA call: runs without a GPU."""
    for L, R, word in ((8, binding.NOALLOC_MAX_R + 1, "RFIM_PT_NOALLOC_MAX_R"), (binding.NOALLOC_MAX_L + 2, 4, "RFIM_PT_NOALLOC_MAX_L")):
        with pytest.raises(binding.RfimPtError) as e:
            binding.energy_terms_noalloc(L, R, BIMODAL, 256, 256, 256)
        assert e.value.code == -1 and word in str(e.value)
    for L, R, kind in ((7, 4, 0), (0, 4, 0), (8, 0, 0), (8, 4, 2)):
        with pytest.raises(binding.RfimPtError) as e:
            binding.energy_terms_noalloc(L, R, kind, 256, 256, 256)
        assert e.value.code == -1
    with pytest.raises(binding.RfimPtError):
        binding.energy_terms_noalloc(8, 4, 0, 0, 256, 256)
