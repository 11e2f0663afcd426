"""Rank sharding.  No method arithmetic lives here.  One process per GPU.

Two ways to use several GPUs:
  * independent disorder realisations per rank: rank r of W takes the realisations whose seeds are
    `rank_seeds(base_seeds, r)`; no data-path collective, only the reduction of timings (max over ranks) and, for
    drivers that want them, a gather of per-realisation observables;
  * ONE realisation, its R replica slots dealt to the ranks in contiguous windows (Eq. 6:
    m = ceil(M/D) replicas per GPU): `replica_window` gives rank r's window and `make_terms_gather` builds the one
    collective of the path, the all-gather of 24 bytes of integer energy terms per slot before every exchange step,
    after which every rank takes the same exchange decisions (lattices never move).
"""
from typing import Sequence

import torch
import torch.distributed as dist


def rank_seeds(base_seeds: Sequence[int], rank: int):
    """Seeds of the realisations rank `rank` runs: every rank gets its own disorder, same workload shape."""
    return [int(s) + int(rank) for s in base_seeds]


def max_over_ranks(values: Sequence[float], device="cpu"):
    """Element-wise MAX of `values` over all ranks (identity when torch.distributed is not initialised)."""
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_rate(units_per_rank: float, world: int, max_ms: float) -> float:
    """Whole-job throughput in units/ns: all ranks' units over the slowest rank's time."""
    return units_per_rank * world / (max_ms * 1e6)


def gather_by_rank(x: torch.Tensor):
    """all_gather of equally shaped per-rank observables -> list indexed by rank (list of one without a group)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [x]
    out = [torch.empty_like(x) for _ in range(dist.get_world_size())]
    dist.all_gather(out, x)
    return out


def replica_window(R: int, world: int, rank: int):
    """(slot0, nslots) of rank `rank`: contiguous windows of m = ceil(R / world) slots (Eq. 6).  The last
    windows may reach past R (padding, the paper's M' = D * m): those slots are never active."""
    m = -(-int(R) // int(world))
    if (world - 1) * m >= R:
        raise ValueError(f"{world} ranks of {m} slots leave a rank without any of the {R} slots: use fewer ranks")
    return rank * m, m


def replica_round_robin(R: int, world: int, rank: int):
    """Slots of rank `rank` when the R slots are dealt round-robin: rank, rank + world, ... ("replica i goes
    to GPU i mod k").  Pass (rank, world) as `shard_rr` to binding.RfimPT; returns the slot list for bookkeeping."""
    if rank >= R:
        raise ValueError(f"rank {rank} of {world} would store none of the {R} slots: use fewer ranks")
    return list(range(int(rank), int(R), int(world)))


def all_gather_rows(terms: torch.Tensor, rank: int, world: int, group=None):
    """In-place all-gather of a [world * m, 3] int64 array whose rows [rank*m, (rank+1)*m) are valid on this rank.
    Works on any device / backend (NCCL on CUDA tensors, gloo on CPU tensors); identity for world == 1."""
    assert terms.dim() == 2 and terms.shape[0] % world == 0
    if world == 1:
        return terms
    m = terms.shape[0] // world
    mine = terms[rank * m:(rank + 1) * m]
    if not terms.is_cuda:
        mine = mine.clone()                                # gloo: the send buffer must not alias the receive buffer
    # NCCL gathers in place when the send buffer is this rank's block of the receive buffer: no copy
    dist.all_gather_into_tensor(terms.view(-1), mine.view(-1), group=group)
    return terms


class _DevicePtr:
    """Expose a raw device pointer to torch through __cuda_array_interface__ (no copy, no ownership)."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes // 8,), "typestr": "<i8", "data": (int(ptr), False), "version": 3}


def make_terms_gather(rank: int, world: int, group=None):
    """The function to hand to RfimPT.set_gather: wraps the library's energy-term array (device memory the library
    owns) in a tensor and all-gathers it in place over torch.distributed.  The handle must run on torch's current
    stream (the binding's default), which is what orders the collective against the library's kernels."""
    def gather(terms_ptr, local_offset, local_bytes, total_bytes, stream_ptr):
        t = torch.as_tensor(_DevicePtr(terms_ptr, total_bytes), device="cuda").view(-1, 3)
        assert local_offset == rank * local_bytes and total_bytes == world * local_bytes, "windows must be equal and ordered by rank"
        all_gather_rows(t, rank, world, group)
    return gather


def make_lattice_broadcast(group=None):
    """The function to hand to RfimPT.set_broadcast: wraps the library's lattice buffer (device memory the library owns,
    L^3 / 8 bytes) in a tensor and broadcasts it from `root_rank` over torch.distributed on the current stream."""
    def bcast(buf_ptr, nbytes, root_rank, stream_ptr):
        if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
            return
        t = torch.as_tensor(_BytePtr(buf_ptr, nbytes), device="cuda")
        dist.broadcast(t, src=dist.get_global_rank(group, root_rank) if group is not None else root_rank, group=group)
    return bcast


class _BytePtr:
    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False), "version": 3}


class NcclComm:
    """An NCCL communicator of the library's own (torch's bundled libnccl through ctypes), for rfim_pt_set_nccl: the device
    library then issues ncclAllGather / ncclBroadcast itself on its stream, with no Python between the measuring kernel
    and the exchange kernel.  The unique id travels from rank 0 over torch.distributed (any backend); with world == 1 no
    process group is needed."""

    class _UniqueId(__import__("ctypes").Structure):
        _fields_ = [("internal", __import__("ctypes").c_char * 128)]

    def __init__(self, rank: int, world: int, group=None):
        import ctypes
        self._lib = ctypes.CDLL(self._find_libnccl())
        uid = NcclComm._UniqueId()
        if rank == 0:
            self._check(self._lib.ncclGetUniqueId(ctypes.byref(uid)), "ncclGetUniqueId")
        if world > 1:
            box = [bytes(uid.internal)] if rank == 0 else [None]
            dist.broadcast_object_list(box, src=0, group=group)
            ctypes.memmove(ctypes.byref(uid), box[0], 128)
        comm = ctypes.c_void_p()
        self._lib.ncclCommInitRank.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, NcclComm._UniqueId, ctypes.c_int]
        self._check(self._lib.ncclCommInitRank(ctypes.byref(comm), world, uid, rank), "ncclCommInitRank")
        self.comm = comm.value
        self.rank, self.world = rank, world
        self.fn_all_gather = ctypes.cast(self._lib.ncclAllGather, ctypes.c_void_p).value
        self.fn_broadcast = ctypes.cast(self._lib.ncclBroadcast, ctypes.c_void_p).value

    @staticmethod
    def _find_libnccl():
        import os
        for line in open("/proc/self/maps"):                 # the copy torch has loaded
            if "libnccl.so" in line:
                return line.split()[-1]
        import nvidia.nccl
        return os.path.join(list(nvidia.nccl.__path__)[0], "lib", "libnccl.so.2")

    @staticmethod
    def _check(rc, what):
        if rc != 0:
            raise RuntimeError(f"{what} failed with ncclResult_t {rc}")

    def close(self):
        if getattr(self, "comm", None):
            import ctypes
            self._lib.ncclCommDestroy.argtypes = [ctypes.c_void_p]
            self._lib.ncclCommDestroy(ctypes.c_void_p(self.comm))
            self.comm = None
