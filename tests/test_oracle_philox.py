"""Pins for the oracle's Philox4x32-10 (north_star fixes the generator; the paper names none).

Two independent sources: the Random123 known-answer vectors (tests/golden) and PyTorch's
header-only at::philox_engine compiled here with g++.
"""
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def test_known_answer_vectors(oracle_mod):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        got = oracle_mod.philox4x32_10((v[4], v[5]), tuple(v[0:4]))
        assert got == v[6:10]


@pytest.fixture(scope="module")
def torch_philox(tmp_path_factory):
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    exe = str(tmp_path_factory.mktemp("tph") / "torch_philox")
    subprocess.run(["g++", "-O1", "-std=c++17", "-I" + inc, "-o", exe,
                    os.path.join(HERE, "helpers_torch_philox.cpp")], check=True)

    def run(seed, subsequence, offset, n):
        out = subprocess.run([exe, str(seed), str(subsequence), str(offset), str(n)],
                             check=True, capture_output=True, text=True).stdout.split()
        return [int(x) for x in out]
    return run


def test_against_torch_philox_engine(oracle_mod, torch_philox):
    # at::philox_engine(seed, subsequence, offset): key = (seed lo, seed hi),
    # counter = (offset lo, offset hi, subsequence lo, subsequence hi)  [PhiloxRNGEngine.h:79-96]
    rng = np.random.default_rng(12345)
    for _ in range(12):
        seed, sub, off = (int(x) for x in rng.integers(0, 2 ** 63, size=3, dtype=np.int64))
        words = torch_philox(seed, sub, off, 8)
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for q in range(2):
            o = off + q
            ctr = (o & 0xFFFFFFFF, (o >> 32) & 0xFFFFFFFF, sub & 0xFFFFFFFF, sub >> 32)
            assert oracle_mod.philox4x32_10(key, ctr) == words[4 * q:4 * q + 4]


def test_initial_spins_and_bimodal_field_follow_the_stream(oracle_mod):
    # reading S2: spins domain 3 (counter i>>2, replica slot in word 2), field domain 4; top bit decides
    L, R, seed = 4, 3, 0x1234567887654321
    o = oracle_mod.Oracle(L, R, 1.0, 1.0, 0, seed)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    f = o.get_field()
    for i in (0, 1, 17, 63):
        w = oracle_mod.philox4x32_10(key, (i, 0, 0, 4))
        assert f[i] == (1 if w[0] >> 31 else -1)
    for r in range(R):
        s = o.get_spins_slot(r)
        for i in (0, 5, 62, 63):
            w = oracle_mod.philox4x32_10(key, (i >> 2, 0, r, 3))
            assert s[i] == (1 if w[i & 3] >> 31 else -1)
    # different slots / seeds give different configurations; same seed reproduces
    assert not np.array_equal(o.get_spins_slot(0), o.get_spins_slot(1))
    o2 = oracle_mod.Oracle(L, R, 1.0, 1.0, 0, seed)
    assert np.array_equal(o2.get_spins_slot(2), o.get_spins_slot(2))
    assert np.array_equal(o2.get_field(), f)
