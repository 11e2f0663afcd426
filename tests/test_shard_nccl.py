"""-m gpu: the NCCL route of the replica-distribution gather on the one GPU the tests have (world_size 1).

`sharding.make_terms_gather` wraps the library's device array through __cuda_array_interface__ and runs
torch.distributed.all_gather_into_tensor on it from inside the library's callback.  With one rank the collective is a
copy, but the plumbing under test is the real one: NCCL accepts the aliased tensor, the call is ordered on the handle's
stream between the measuring kernel and the exchange kernel, and the run stays bit-identical to the oracle.  Runs in a
subprocess so that the process group does not leak into the other tests.
"""
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
torch.cuda.set_device(0)
dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
import oracle
from paper_1508_06268_b200 import binding, sharding
from paper_1508_06268_b200.workloads import geometric_ladder
L, R = 32, 6
T = geometric_ladder(0.9, 5.0, R)
calls = {"n": 0}
inner = sharding.make_terms_gather(0, 1)
def gather(ptr, off, nloc, ntot, stream):
    calls["n"] += 1
    t = torch.as_tensor(sharding._DevicePtr(ptr, ntot), device="cuda")
    mine = t.clone()
    dist.all_gather_into_tensor(t, mine)          # the real NCCL call on the aliased array (world 1)
    inner(ptr, off, nloc, ntot, stream)
g = binding.RfimPT(L, R, 1.0, 1.5, binding.GAUSSIAN, seed=9, shard=sharding.replica_window(R, 1, 0))
g.set_gather(gather)
g.set_temperatures(T)
o = oracle.Oracle(L, R, 1.0, 1.5, binding.GAUSSIAN, 9)
o.set_temperatures(T)
g.sweep(12, 3); o.sweep(12, 3)
assert calls["n"] == 4, calls
for r in range(R):
    assert np.array_equal(g.get_spins_slot(r), o.get_spins_slot(r)), r
assert np.array_equal(g.get_permutation(), o.get_permutation())
for a, b in zip(g.get_timeseries(), o.get_timeseries()):
    assert np.array_equal(a, b)
g.close()
dist.destroy_process_group()
print("shard-nccl-ok")
"""


def test_terms_gather_through_nccl_world_1():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r = subprocess.run([sys.executable, "-c", CHILD % ROOT], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "shard-nccl-ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]


CHILD_NATIVE = r"""
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch
torch.cuda.set_device(0)
import oracle
from paper_1508_06268_b200 import binding, sharding
from paper_1508_06268_b200.workloads import geometric_ladder
comm = sharding.NcclComm(0, 1)                    # the library's own communicator, world 1
for rr in (False, True):
    L, R, n0 = 32, 8, 5
    T = geometric_ladder(0.9, 5.0, n0)
    g = binding.RfimPT(L, R, 1.0, 1.5, binding.GAUSSIAN, seed=9, **({"shard_rr": (0, 1)} if rr else {"shard": sharding.replica_window(R, 1, 0)}))
    g.set_nccl(comm)                              # no Python callback: ncclAllGather / ncclBroadcast are called from C
    g.set_temperatures(T); g.set_adapt_params(3, 2)
    o = oracle.Oracle(L, R, 1.0, 1.5, binding.GAUSSIAN, 9)
    o.set_temperatures(T); o.set_adapt_params(3, 2)
    g.adapt_temperatures(30); o.adapt_temperatures(30)     # inserts two replicas: ncclBroadcast of their lattices
    g.sweep(12, 3); o.sweep(12, 3)                         # four exchange steps: ncclAllGather of the energy terms
    assert g.n == o.n == 7
    for r in range(g.n):
        assert np.array_equal(g.get_spins_slot(r), o.get_spins_slot(r)), r
    assert np.array_equal(g.get_permutation(), o.get_permutation())
    for a, b in zip(g.get_timeseries(), o.get_timeseries()):
        assert np.array_equal(a, b)
    g.close()
comm.close()
print("shard-nccl-native-ok")
"""


def test_native_nccl_route_world_1():
    r = subprocess.run([sys.executable, "-c", CHILD_NATIVE % ROOT], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "shard-nccl-native-ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
