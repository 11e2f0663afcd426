"""-m "not gpu": the launch planning of rfim_pt_sweep (rfim_pt_plan_launch: host logic only, no CUDA call).

A persistent sweep kernel covers at most 127 sweeps per launch, stops at the first exchange step it reaches, or -- the resident
kernel on a single unsharded handle -- runs on through every whole exchange period that fits ("several
moves per launch").  Hand-derived cases, then the invariants of the whole call on random arguments."""
import numpy as np
import pytest


def _plan(*a):
    from paper_1508_06268_b200 import binding
    return binding.plan_launch(*a)


@pytest.mark.parametrize("args,expected", [
    ((0, 10, 10, 0), (10, 1)),            # one move per launch: to the next exchange step
    ((0, 10, 10, 1), (10, 1)),
    ((0, 10000, 10, 0), (10, 1)),
    ((0, 10000, 10, 1), (120, 12)),       # twelve whole periods fit in 127 sweeps
    ((120, 9880, 10, 1), (120, 12)),
    ((3, 100, 10, 1), (97, 10)),          # off a boundary: 7 sweeps to the first step, then nine periods
    ((3, 5, 10, 1), (5, 0)),              # ends before the next step: no exchange in this launch
    ((3, 7, 10, 1), (7, 1)),
    ((3, 16, 10, 1), (7, 1)),             # the second period does not fit whole: stop at the first step
    ((3, 17, 10, 1), (17, 2)),
    ((0, 300, 0, 1), (127, 0)),           # no exchange at all
    ((0, 130, 200, 1), (127, 0)),         # period longer than a launch
    ((0, 500, 127, 1), (127, 1)),
    ((5, 20, 5, 1), (20, 4)),
    ((5, 20, 5, 0), (5, 1)),
])
def test_launch_plan_cases(args, expected):
    assert _plan(*args) == expected


def test_launch_plan_bad_arguments():
    from paper_1508_06268_b200 import binding
    with pytest.raises(binding.RfimPtError):
        _plan(0, 0, 10, 1)
    with pytest.raises(binding.RfimPtError):
        _plan(0, 10, -1, 1)


def test_launch_plan_invariants_of_a_whole_call():
    rng = np.random.default_rng(7)
    for _ in range(400):
        s0 = int(rng.integers(0, 5000)); n = int(rng.integers(1, 3000)); k = int(rng.choice([0, 1, 2, 3, 5, 7, 10, 64, 127, 128, 1000]))
        multi = int(rng.integers(0, 2))
        s, left, steps, launches = s0, n, 0, 0
        while left > 0:
            sw, st = _plan(s, left, k, multi)
            assert 1 <= sw <= min(left, 127)
            if st:                                            # a launch that holds steps ends on one and covers whole periods after the first
                assert k > 0 and (s + sw) % k == 0
                first = k - s % k
                assert sw == first + (st - 1) * k
                assert multi or st == 1
            elif k > 0:                                       # no step inside: it did not reach a boundary
                assert (s // k) == ((s + sw) // k) or (s + sw) % k != 0
                assert ((s + sw) // k) == (s // k)
            s += sw; left -= sw; steps += st; launches += 1
        assert s == s0 + n
        assert steps == (0 if k == 0 else (s0 + n) // k - s0 // k)
        if multi and k and k <= 63 and n >= 4 * 127:
            assert launches <= -(-n // (127 - k)) + 1             # several periods per launch
