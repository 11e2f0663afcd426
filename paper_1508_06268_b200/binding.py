"""Thin ctypes binding over librfimpt.so (include/rfim_pt.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for the device
allocator (installed as the library's allocator hook) and for the current stream.  There is no CPU
fallback: if the library is missing or no CUDA device is present the calls raise.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("RFIM_PT_LIB") or os.path.join(_HERE, "librfimpt.so")   # RFIM_PT_LIB: another build of the same library (A/B timing)
_lib = None
_alloc_refs = {}

BIMODAL, GAUSSIAN = 0, 1
OK, EINVAL, ESTATE, ENOMEM, ECUDA = 0, -1, -2, -3, -4

_vp = ctypes.c_void_p
_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_i8p = ctypes.POINTER(ctypes.c_int8)
_i32p = ctypes.POINTER(ctypes.c_int32)
_i64p = ctypes.POINTER(ctypes.c_int64)
_u64p = ctypes.POINTER(ctypes.c_uint64)
_GATHER_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_size_t, ctypes.c_size_t,
                              ctypes.c_void_p)
_ALLOC_FN = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t)
_FREE_FN = ctypes.CFUNCTYPE(None, ctypes.c_void_p)
_BCAST_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_void_p)

# every symbol include/rfim_pt.h declares: name -> (restype, argtypes)
SIGNATURES = {
    "rfim_pt_create": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                      ctypes.c_int, ctypes.c_uint64]),
    "rfim_pt_create_batch": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                            ctypes.c_double, ctypes.c_int, ctypes.c_int, _u64p]),
    "rfim_pt_create_shard": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                            ctypes.c_int, ctypes.c_uint64, ctypes.c_int, ctypes.c_int]),
    "rfim_pt_create_shard_rr": (ctypes.c_int, [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                               ctypes.c_int, ctypes.c_uint64, ctypes.c_int, ctypes.c_int]),
    "rfim_pt_set_gather": (ctypes.c_int, [_vp, _GATHER_FN, _vp]),
    "rfim_pt_set_broadcast": (ctypes.c_int, [_vp, _BCAST_FN, _vp]),
    "rfim_pt_set_nccl": (ctypes.c_int, [_vp, _vp, _vp, _vp]),
    "rfim_pt_get_shard_layout": (ctypes.c_int, [_vp, _ip, _ip, _ip, _ip, _ip]),
    "rfim_pt_get_trial_rates": (ctypes.c_int, [_vp, ctypes.c_int, _dp, _ip]),
    "rfim_pt_get_shard": (ctypes.c_int, [_vp, _ip, _ip, ctypes.POINTER(_vp), ctypes.POINTER(ctypes.c_size_t)]),
    "rfim_pt_destroy": (ctypes.c_int, [_vp]),
    "rfim_pt_set_temperatures": (ctypes.c_int, [_vp, _dp, ctypes.c_int]),
    "rfim_pt_sweep": (ctypes.c_int, [_vp, ctypes.c_int64, ctypes.c_int]),
    "rfim_pt_adapt_temperatures": (ctypes.c_int, [_vp, ctypes.c_int64]),
    "rfim_pt_observables": (ctypes.c_int, [_vp, _dp, _dp, _dp]),
    "rfim_pt_get_spins": (ctypes.c_int, [_vp, ctypes.c_int, _i8p]),
    "rfim_pt_set_stream": (ctypes.c_int, [_vp, _vp]),
    "rfim_pt_synchronize": (ctypes.c_int, [_vp]),
    "rfim_pt_set_allocator": (ctypes.c_int, [_ALLOC_FN, _FREE_FN]),
    "rfim_pt_last_error": (ctypes.c_char_p, [_vp]),
    "rfim_pt_set_packing": (ctypes.c_int, [_vp, ctypes.c_int]),
    "rfim_pt_set_kernel_variant": (ctypes.c_int, [_vp, ctypes.c_int]),
    "rfim_pt_set_tuning": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "rfim_pt_set_adapt_params": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "rfim_pt_get_info": (ctypes.c_int, [_vp, _ip, _ip, _ip, _ip, _ip]),
    "rfim_pt_get_spins_member": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _i8p]),
    "rfim_pt_get_spins_slot": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _i8p]),
    "rfim_pt_set_spins_slot": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _i8p]),
    "rfim_pt_get_spins_all": (ctypes.c_int, [_vp, _i8p]),
    "rfim_pt_set_spins_all": (ctypes.c_int, [_vp, _i8p]),
    "rfim_pt_get_spins_all_bits": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_uint8)]),
    "rfim_pt_set_spins_all_bits": (ctypes.c_int, [_vp, ctypes.POINTER(ctypes.c_uint8)]),
    "rfim_pt_get_field": (ctypes.c_int, [_vp, ctypes.c_int, _i32p]),
    "rfim_pt_set_field": (ctypes.c_int, [_vp, ctypes.c_int, _i32p]),
    "rfim_pt_get_permutation": (ctypes.c_int, [_vp, ctypes.c_int, _i32p]),
    "rfim_pt_set_permutation": (ctypes.c_int, [_vp, ctypes.c_int, _i32p]),
    "rfim_pt_get_temperatures": (ctypes.c_int, [_vp, ctypes.c_int, _dp, _ip]),
    "rfim_pt_get_counters": (ctypes.c_int, [_vp, _u64p, _u64p]),
    "rfim_pt_set_counters": (ctypes.c_int, [_vp, ctypes.c_uint64, ctypes.c_uint64]),
    "rfim_pt_get_energy_terms": (ctypes.c_int, [_vp, ctypes.c_int, _i64p, _i64p, _i64p]),
    "rfim_pt_timeseries_steps": (ctypes.c_int64, [_vp]),
    "rfim_pt_get_timeseries": (ctypes.c_int, [_vp, ctypes.c_int, _i64p, _i64p, _i64p]),
    "rfim_pt_thermal_moments": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int64, _dp]),
    "rfim_pt_thermal_observables": (ctypes.c_int, [_vp, ctypes.c_int64, _dp, _dp, _dp]),
    "rfim_pt_get_exchange_counts": (ctypes.c_int, [_vp, ctypes.c_int, _u64p, _u64p]),
    "rfim_pt_get_bimodal_threshold": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _u64p]),
    "rfim_pt_get_diagnostics": (ctypes.c_int, [_vp, _u64p]),
    "rfim_pt_plan_adaptation": (ctypes.c_int, [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.POINTER(ctypes.c_int)]),
    "rfim_pt_plan_launch": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int)]),
    "rfim_pt_energy_terms_noalloc": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]),
    "rfim_pt_noalloc_last_error": (ctypes.c_char_p, []),
    "rfim_pt_bench_philox": (ctypes.c_int, [_vp, ctypes.c_int, _dp, _dp]),
    "rfim_pt_bench_issue": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _dp, _dp]),
    "rfim_pt_bench_stream": (ctypes.c_int, [_vp, ctypes.c_size_t, _dp, _dp]),
}


class RfimPtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"librfimpt error {code}: {msg}")
        self.code = code


def load():
    """dlopen the library and type every entry point (no GPU needed for this)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_1508_06268_b200.build` "
                               "(the CUDA extension is the product; there is no fallback)")
        L = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def use_torch_allocator():
    """Route the library's device allocations through PyTorch's CUDA caching allocator."""
    import torch
    lib = load()
    if "alloc" in _alloc_refs:            # installed once per process (handles may be created from several threads)
        return

    def _alloc(nbytes):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes))
        except Exception:
            return None

    def _free(ptr):
        try:
            if ptr:
                torch.cuda.caching_allocator_delete(ptr)
        except (AttributeError, TypeError):           # interpreter shutdown: torch is already torn down
            pass

    a, f = _ALLOC_FN(_alloc), _FREE_FN(_free)
    _alloc_refs["alloc"], _alloc_refs["free"] = a, f          # keep the thunks alive
    rc = lib.rfim_pt_set_allocator(a, f)
    if rc:
        raise RfimPtError(rc, "rfim_pt_set_allocator")


def _p(a, t):
    return a.ctypes.data_as(t)


class RfimPT:
    """Handle on D realisations x R replica slots of an L^3 lattice (see include/rfim_pt.h)."""

    def __init__(self, L, R, J, h, field_kind, seed=None, seeds=None, torch_allocator=True, torch_stream=True, shard=None, shard_rr=None):
        lib = load()
        if torch_allocator:
            import torch
            if not torch.cuda.is_available():
                raise RuntimeError("no CUDA device: librfimpt has no CPU fallback")
            torch.cuda.init()
            use_torch_allocator()
        self._h = _vp()
        self.shard = shard
        self._gather_ref = None
        self._bcast_ref = None
        if shard_rr is not None:          # (rank, world): this handle stores slots rank, rank + world, ...
            rc = lib.rfim_pt_create_shard_rr(ctypes.byref(self._h), L, R, J, h, field_kind, int(seed), int(shard_rr[0]), int(shard_rr[1]))
            self.D = 1
            shard = (int(shard_rr[0]), -(-R // int(shard_rr[1])))
            self.shard = shard
        elif shard is not None:           # (slot0, nslots): this handle stores that window of the R slots
            rc = lib.rfim_pt_create_shard(ctypes.byref(self._h), L, R, J, h, field_kind, int(seed), int(shard[0]), int(shard[1]))
            self.D = 1
        elif seeds is None:
            rc = lib.rfim_pt_create(ctypes.byref(self._h), L, R, J, h, field_kind, int(seed))
            self.D = 1
        else:
            s = np.ascontiguousarray(seeds, dtype=np.uint64)
            rc = lib.rfim_pt_create_batch(ctypes.byref(self._h), L, R, J, h, field_kind, len(s), _p(s, _u64p))
            self.D = len(s)
        if rc:
            raise RfimPtError(rc, "rfim_pt_create failed (bad argument, no CUDA device, or out of memory)")
        self.L, self.R, self.J, self.h, self.kind = L, R, J, h, field_kind
        self.N = L ** 3
        self.stored_slots = R if shard is None else int(shard[1])     # lattices this handle keeps in device memory
        self._torch_stream = torch_stream
        if torch_stream:
            self.use_current_torch_stream()

    # -- plumbing ---------------------------------------------------------------------------
    def _ck(self, rc):
        if rc:
            raise RfimPtError(rc, load().rfim_pt_last_error(self._h).decode())

    def use_current_torch_stream(self):
        import torch
        self._ck(load().rfim_pt_set_stream(self._h, _vp(torch.cuda.current_stream().cuda_stream)))

    def set_stream(self, cuda_stream_ptr):
        self._ck(load().rfim_pt_set_stream(self._h, _vp(cuda_stream_ptr)))

    def synchronize(self):
        self._ck(load().rfim_pt_synchronize(self._h))

    def close(self):
        if getattr(self, "_h", None):
            load().rfim_pt_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def n(self):
        n = ctypes.c_int()
        self._ck(load().rfim_pt_get_info(self._h, None, None, ctypes.byref(n), None, None))
        return n.value

    # -- the calls north_star names ---------------------------------------------------------------
    def set_temperatures(self, T):
        T = np.ascontiguousarray(T, dtype=np.float64)
        self._ck(load().rfim_pt_set_temperatures(self._h, _p(T, _dp), len(T)))

    def sweep(self, n_sweeps, exchange_every):
        self._ck(load().rfim_pt_sweep(self._h, int(n_sweeps), int(exchange_every)))

    def adapt_temperatures(self, trial_sweeps):
        self._ck(load().rfim_pt_adapt_temperatures(self._h, int(trial_sweeps)))

    def observables(self):
        n, D = self.n, self.D
        E = np.zeros((D, n)); M = np.zeros((D, n)); rate = np.zeros((D, max(n - 1, 0)))
        self._ck(load().rfim_pt_observables(self._h, _p(E, _dp), _p(M, _dp), _p(rate, _dp)))
        if D == 1:
            return E[0], M[0], rate[0]
        return E, M, rate

    def get_spins(self, temp_rank, d=0):
        out = np.zeros(self.N, dtype=np.int8)
        self._ck(load().rfim_pt_get_spins_member(self._h, d, temp_rank, _p(out, _i8p)))
        return out

    # -- extensions ------------------------------------------------------------------------------
    def set_gather(self, fn):
        """fn(terms_device_ptr, local_offset, local_bytes, total_bytes, stream_ptr) -> None: completes the energy-term
        array across ranks (include/rfim_pt.h, replica distribution).  Exceptions become a non-zero return code."""
        def _thunk(user, terms, off, nloc, ntot, stream):
            try:
                fn(terms, off, nloc, ntot, stream)
                return 0
            except Exception:                       # must not unwind through the C library
                import traceback
                traceback.print_exc()
                return 1
        self._gather_ref = _GATHER_FN(_thunk)       # keep the thunk alive as long as the handle
        self._ck(load().rfim_pt_set_gather(self._h, self._gather_ref, None))

    def set_broadcast(self, fn):
        """fn(buffer_device_ptr, nbytes, root_rank, stream_ptr) -> None: hands one bit-packed lattice from its owner to every
        rank (include/rfim_pt.h; used when an adaptation step inserts a replica on a shard)."""
        def _thunk(user, buf, nbytes, root, stream):
            try:
                fn(buf, nbytes, root, stream)
                return 0
            except Exception:
                import traceback
                traceback.print_exc()
                return 1
        self._bcast_ref = _BCAST_FN(_thunk)
        self._ck(load().rfim_pt_set_broadcast(self._h, self._bcast_ref, None))

    def set_nccl(self, comm):
        """comm: sharding.NcclComm (or None): the library then calls ncclAllGather / ncclBroadcast itself (rfim_pt_set_nccl)."""
        if comm is None:
            self._ck(load().rfim_pt_set_nccl(self._h, None, None, None))
        else:
            self._nccl_ref = comm                  # keep the communicator alive as long as the handle uses it
            self._ck(load().rfim_pt_set_nccl(self._h, _vp(comm.comm), _vp(comm.fn_all_gather), _vp(comm.fn_broadcast)))

    def get_shard_layout(self):
        v = [ctypes.c_int() for _ in range(5)]
        self._ck(load().rfim_pt_get_shard_layout(self._h, *[ctypes.byref(x) for x in v]))
        return dict(zip(("rank", "world", "first_slot", "stride", "nslots"), (x.value for x in v)))

    def stored_slot_ids(self):
        """Global slot indices of the lattices this handle stores, in storage order."""
        lay = self.get_shard_layout()
        return [lay["first_slot"] + j * lay["stride"] for j in range(lay["nslots"]) if lay["first_slot"] + j * lay["stride"] < self.R]

    def get_trial_rates(self, d=0):
        """Exchange rates measured by the trial run of the last adapt_temperatures call (the rates its update used)."""
        n = ctypes.c_int()
        self._ck(load().rfim_pt_get_trial_rates(self._h, d, None, ctypes.byref(n)))
        rate = np.zeros(n.value, dtype=np.float64)
        self._ck(load().rfim_pt_get_trial_rates(self._h, d, _p(rate, _dp), ctypes.byref(n)))
        return rate

    def get_shard(self):
        a, b, ptr, nb = ctypes.c_int(), ctypes.c_int(), _vp(), ctypes.c_size_t()
        self._ck(load().rfim_pt_get_shard(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(ptr), ctypes.byref(nb)))
        return a.value, b.value, ptr.value, nb.value

    def set_packing(self, bits):
        self._ck(load().rfim_pt_set_packing(self._h, bits))

    def set_kernel_variant(self, variant):
        self._ck(load().rfim_pt_set_kernel_variant(self._h, variant))

    def set_tuning(self, key, value):
        self._ck(load().rfim_pt_set_tuning(self._h, key, value))

    def set_adapt_params(self, exchange_every, insertions):
        self._ck(load().rfim_pt_set_adapt_params(self._h, exchange_every, insertions))

    def get_spins_slot(self, slot, d=0):
        out = np.zeros(self.N, dtype=np.int8)
        self._ck(load().rfim_pt_get_spins_slot(self._h, d, slot, _p(out, _i8p)))
        return out

    def set_spins_slot(self, slot, s, d=0):
        s = np.ascontiguousarray(s, dtype=np.int8)
        assert s.size == self.N
        self._ck(load().rfim_pt_set_spins_slot(self._h, d, slot, _p(s, _i8p)))

    def get_spins_all(self, out=None):
        if out is None:
            out = np.zeros((self.D, self.stored_slots, self.N), dtype=np.int8)
        self._ck(load().rfim_pt_get_spins_all(self._h, _p(out, _i8p)))
        return out

    def set_spins_all(self, s):
        assert s.dtype == np.int8 and s.size == self.D * self.stored_slots * self.N and s.flags.c_contiguous
        self._ck(load().rfim_pt_set_spins_all(self._h, _p(s, _i8p)))

    def get_spins_all_bits(self, out=None):
        """[D][stored slots][N/8] uint8: bit i&7 of byte i>>3 set iff s_i = +1 (natural site order)."""
        if out is None:
            out = np.zeros((self.D, self.stored_slots, self.N // 8), dtype=np.uint8)
        self._ck(load().rfim_pt_get_spins_all_bits(self._h, _p(out, ctypes.POINTER(ctypes.c_uint8))))
        return out

    def set_spins_all_bits(self, bits):
        assert bits.dtype == np.uint8 and bits.size == self.D * self.stored_slots * (self.N // 8) and bits.flags.c_contiguous
        self._ck(load().rfim_pt_set_spins_all_bits(self._h, _p(bits, ctypes.POINTER(ctypes.c_uint8))))

    def get_field(self, d=0):
        out = np.zeros(self.N, dtype=np.int32)
        self._ck(load().rfim_pt_get_field(self._h, d, _p(out, _i32p)))
        return out

    def set_field(self, f, d=0):
        f = np.ascontiguousarray(f, dtype=np.int32)
        assert f.size == self.N
        self._ck(load().rfim_pt_set_field(self._h, d, _p(f, _i32p)))

    def get_permutation(self, d=0):
        out = np.zeros(self.n, dtype=np.int32)
        self._ck(load().rfim_pt_get_permutation(self._h, d, _p(out, _i32p)))
        return out

    def set_permutation(self, t2r, d=0):
        t2r = np.ascontiguousarray(t2r, dtype=np.int32)
        assert t2r.size == self.n
        self._ck(load().rfim_pt_set_permutation(self._h, d, _p(t2r, _i32p)))

    def thermal_moments(self, skip=0, d=0):
        out = np.zeros((self.n, 5))
        self._ck(load().rfim_pt_thermal_moments(self._h, d, int(skip), _p(out, _dp)))
        return out

    def thermal_observables(self, skip=0):
        n = self.n
        absM, C, g = np.zeros(n), np.zeros(n), np.zeros(n)
        self._ck(load().rfim_pt_thermal_observables(self._h, int(skip), _p(absM, _dp), _p(C, _dp), _p(g, _dp)))
        return absM, C, g

    def get_temperatures(self, d=0):
        out = np.zeros(self.n)
        self._ck(load().rfim_pt_get_temperatures(self._h, d, _p(out, _dp), None))
        return out

    def get_counters(self):
        a, b = ctypes.c_uint64(), ctypes.c_uint64()
        self._ck(load().rfim_pt_get_counters(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def set_counters(self, sweep_index, exchange_step):
        self._ck(load().rfim_pt_set_counters(self._h, sweep_index, exchange_step))

    def get_energy_terms(self, d=0):
        n = self.n
        Eb = np.zeros(n, dtype=np.int64); Ef = np.zeros(n, dtype=np.int64); Ms = np.zeros(n, dtype=np.int64)
        self._ck(load().rfim_pt_get_energy_terms(self._h, d, _p(Eb, _i64p), _p(Ef, _i64p), _p(Ms, _i64p)))
        return Eb, Ef, Ms

    def get_timeseries(self, d=0):
        steps = int(load().rfim_pt_timeseries_steps(self._h))
        n = self.n
        Eb = np.zeros((steps, n), dtype=np.int64); Ef = np.zeros_like(Eb); Ms = np.zeros_like(Eb)
        if steps:
            self._ck(load().rfim_pt_get_timeseries(self._h, d, _p(Eb, _i64p), _p(Ef, _i64p), _p(Ms, _i64p)))
        return Eb, Ef, Ms

    def get_exchange_counts(self, d=0):
        n = self.n
        att = np.zeros(max(n - 1, 0), dtype=np.uint64); acc = np.zeros_like(att)
        self._ck(load().rfim_pt_get_exchange_counts(self._h, d, _p(att, _u64p), _p(acc, _u64p)))
        return att, acc

    def bimodal_threshold(self, rank, k, b, d=0):
        thr = ctypes.c_uint64()
        self._ck(load().rfim_pt_get_bimodal_threshold(self._h, d, rank, k, b, ctypes.byref(thr)))
        return thr.value

    def diagnostics(self):
        d = (ctypes.c_uint64 * 4)()
        self._ck(load().rfim_pt_get_diagnostics(self._h, d))
        return {"launches": int(d[0]), "exact_path": int(d[1]), "ulp_ambiguous": int(d[2]), "exchange_draws": int(d[3])}


def plan_adaptation(T, rate, R, a):
    """rfim_pt_plan_adaptation: the host-side planning step of the temperature adaptation, no handle, no GPU."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    rate = np.ascontiguousarray(rate, dtype=np.float64)
    out = np.zeros(R, dtype=np.float64)
    n = ctypes.c_int()
    rc = load().rfim_pt_plan_adaptation(_p(T, _dp), _p(rate, _dp), len(T), R, a, _p(out, _dp), ctypes.byref(n))
    if rc:
        raise RfimPtError(rc, "rfim_pt_plan_adaptation")
    return out[:n.value].copy()


def plan_launch(sweep_index, n_sweeps, exchange_every, several_moves):
    """rfim_pt_plan_launch: (sweeps, exchange steps) of the next launch of a persistent sweep kernel; no handle, no GPU."""
    sw, st = ctypes.c_int64(), ctypes.c_int()
    rc = load().rfim_pt_plan_launch(int(sweep_index), int(n_sweeps), int(exchange_every), int(bool(several_moves)), ctypes.byref(sw), ctypes.byref(st))
    if rc:
        raise RfimPtError(rc, "rfim_pt_plan_launch")
    return int(sw.value), int(st.value)


NOALLOC_MAX_R, NOALLOC_MAX_L = 256, 128      # RFIM_PT_NOALLOC_MAX_R / _MAX_L of include/rfim_pt.h


def energy_terms_noalloc(L, R, field_kind, spins_device, field_device, terms_device, stream=None):
    """rfim_pt_energy_terms_noalloc: (Eb, Ef, Msum) per replica from caller-owned DEVICE arrays, given as integer addresses
    (e.g. tensor.data_ptr()): spins int8 [R][L^3], field int32 [L^3], terms int64 [R][3].  Enqueues on `stream` (a raw
    cudaStream_t, default 0) and returns; the library allocates nothing (its scratch is a static device array)."""
    lib = load()
    rc = lib.rfim_pt_energy_terms_noalloc(_vp(stream or 0), int(L), int(R), int(field_kind), _vp(int(spins_device)),
                                          _vp(int(field_device)), _vp(int(terms_device)))
    if rc:
        raise RfimPtError(rc, (lib.rfim_pt_noalloc_last_error() or b"").decode())


def bench_philox(calls_per_thread=2000, stream=None):
    ms, att = ctypes.c_double(), ctypes.c_double()
    rc = load().rfim_pt_bench_philox(_vp(stream or 0), calls_per_thread, ctypes.byref(ms), ctypes.byref(att))
    if rc:
        raise RfimPtError(rc, "rfim_pt_bench_philox")
    return ms.value, att.value


PROBE_KINDS = {"LOP3": 1, "PRMT": 2, "I2FP (ALU)": 3, "I2F.RM (XU)": 4, "FFMA": 5, "FADD": 6, "MUFU.EX2": 7, "LDS.64": 8}


def bench_issue(kind, extra_per_call, stream=None):
    """rfim_pt_bench_issue -> (ms of one launch, warp-rows per SM sub-partition)."""
    ms, wr = ctypes.c_double(), ctypes.c_double()
    rc = load().rfim_pt_bench_issue(_vp(stream or 0), kind, extra_per_call, ctypes.byref(ms), ctypes.byref(wr))
    if rc:
        raise RfimPtError(rc, "rfim_pt_bench_issue")
    return ms.value, wr.value


def bench_stream(nbytes, stream=None):
    ms, moved = ctypes.c_double(), ctypes.c_double()
    rc = load().rfim_pt_bench_stream(_vp(stream or 0), nbytes, ctypes.byref(ms), ctypes.byref(moved))
    if rc:
        raise RfimPtError(rc, "rfim_pt_bench_stream")
    return ms.value, moved.value
