"""CPU oracle for the RFIM parallel-tempering hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of ``oracle/rfim_oracle.cpp`` (see that file's header for the
passages of PAPER.md it follows).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this
package.  It imports nothing from ``paper_1508_06268_b200``.
"""
import ctypes
import os

import numpy as np

from .build import LIB
from .build import build as _build_oracle

_lib = None

_c_void_pp = ctypes.POINTER(ctypes.c_void_p)
_dp = ctypes.POINTER(ctypes.c_double)
_i8p = ctypes.POINTER(ctypes.c_int8)
_i32p = ctypes.POINTER(ctypes.c_int32)
_i64p = ctypes.POINTER(ctypes.c_int64)
_u32p = ctypes.POINTER(ctypes.c_uint32)
_u64p = ctypes.POINTER(ctypes.c_uint64)


def lib():
    global _lib
    if _lib is None:
        _build_oracle()
        L = ctypes.CDLL(LIB)
        sig = {
            "oracle_philox4x32_10": (None, [ctypes.c_uint32] * 6 + [_u32p]),
            "oracle_threshold_from_x": (ctypes.c_uint64, [ctypes.c_double]),
            "oracle_create": (ctypes.c_int, [_c_void_pp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                             ctypes.c_double, ctypes.c_int, ctypes.c_uint64]),
            "oracle_destroy": (ctypes.c_int, [ctypes.c_void_p]),
            "oracle_set_threads": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
            "oracle_set_temperatures": (ctypes.c_int, [ctypes.c_void_p, _dp, ctypes.c_int]),
            "oracle_sweep": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int]),
            "oracle_adapt_temperatures": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int64]),
            "oracle_set_adapt_params": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]),
            "oracle_plan_adaptation": (ctypes.c_int, [_dp, _dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, ctypes.POINTER(ctypes.c_int)]),
            "oracle_observables": (ctypes.c_int, [ctypes.c_void_p, _dp, _dp, _dp]),
            "oracle_get_spins": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, _i8p]),
            "oracle_get_spins_slot": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, _i8p]),
            "oracle_set_spins_slot": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, _i8p]),
            "oracle_get_field": (ctypes.c_int, [ctypes.c_void_p, _i32p]),
            "oracle_set_field": (ctypes.c_int, [ctypes.c_void_p, _i32p]),
            "oracle_get_permutation": (ctypes.c_int, [ctypes.c_void_p, _i32p]),
            "oracle_set_permutation": (ctypes.c_int, [ctypes.c_void_p, _i32p]),
            "oracle_get_temperatures": (ctypes.c_int, [ctypes.c_void_p, _dp, ctypes.POINTER(ctypes.c_int)]),
            "oracle_get_counters": (ctypes.c_int, [ctypes.c_void_p, _u64p, _u64p]),
            "oracle_set_counters": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint64]),
            "oracle_get_energy_terms": (ctypes.c_int, [ctypes.c_void_p, _i64p, _i64p, _i64p]),
            "oracle_timeseries_steps": (ctypes.c_int64, [ctypes.c_void_p]),
            "oracle_get_timeseries": (ctypes.c_int, [ctypes.c_void_p, _i64p, _i64p, _i64p]),
            "oracle_get_exchange_counts": (ctypes.c_int, [ctypes.c_void_p, _u64p, _u64p]),
            "oracle_site_threshold": (ctypes.c_uint64, [ctypes.c_void_p] + [ctypes.c_int] * 4),
            "oracle_bimodal_threshold": (ctypes.c_uint64, [ctypes.c_void_p] + [ctypes.c_int] * 3),
            "oracle_energy_from_terms": (ctypes.c_double, [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64]),
            "oracle_thermal_moments": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int64, _dp]),
            "oracle_half_sweep": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_uint64]),
            "oracle_exchange_step": (ctypes.c_int, [ctypes.c_void_p]),
            "oracle_last_error": (ctypes.c_char_p, [ctypes.c_void_p]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def philox4x32_10(key, ctr):
    """key = (k0, k1), ctr = (c0, c1, c2, c3) -> four uint32 words."""
    out = (ctypes.c_uint32 * 4)()
    lib().oracle_philox4x32_10(key[0], key[1], ctr[0], ctr[1], ctr[2], ctr[3], out)
    return [int(v) for v in out]


def plan_adaptation(T, rate, R, a):
    """The planning step of the adaptation alone (S8): ladder T with interval exchange rates
    `rate`, capacity R, a insertions -> the new ladder."""
    T = np.ascontiguousarray(T, dtype=np.float64)
    rate = np.ascontiguousarray(rate, dtype=np.float64)
    assert len(rate) == len(T) - 1
    out = np.zeros(R, dtype=np.float64)
    n = ctypes.c_int()
    rc = lib().oracle_plan_adaptation(_ptr(T, _dp), _ptr(rate, _dp), len(T), R, a, _ptr(out, _dp), ctypes.byref(n))
    if rc:
        raise OracleError(f"oracle_plan_adaptation failed ({rc})")
    return out[:n.value].copy()


def threshold_from_x(x):
    return int(lib().oracle_threshold_from_x(float(x)))


def _ptr(a, t):
    return a.ctypes.data_as(t)


class OracleError(RuntimeError):
    pass


class Oracle:
    """One disorder realisation: R replica slots of an L^3 lattice."""

    BIMODAL, GAUSSIAN = 0, 1

    def __init__(self, L, R, J, h, field_kind, seed, threads=1):
        self._h = ctypes.c_void_p()
        rc = lib().oracle_create(ctypes.byref(self._h), L, R, J, h, field_kind, seed)
        if rc:
            raise OracleError(f"oracle_create failed ({rc})")
        self.L, self.R, self.J, self.h, self.kind, self.seed = L, R, J, h, field_kind, seed
        self.N = L ** 3
        if threads != 1:
            lib().oracle_set_threads(self._h, threads)

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc:
            raise OracleError(f"oracle call failed ({rc}): {lib().oracle_last_error(self._h).decode()}")

    # --- north_star calls -------------------------------------------------
    def set_temperatures(self, T):
        T = np.ascontiguousarray(T, dtype=np.float64)
        self._ck(lib().oracle_set_temperatures(self._h, _ptr(T, _dp), len(T)))

    def sweep(self, n_sweeps, exchange_every):
        self._ck(lib().oracle_sweep(self._h, n_sweeps, exchange_every))

    def adapt_temperatures(self, trial_sweeps):
        self._ck(lib().oracle_adapt_temperatures(self._h, trial_sweeps))

    def set_adapt_params(self, exchange_every, insertions):
        self._ck(lib().oracle_set_adapt_params(self._h, exchange_every, insertions))

    @property
    def n(self):
        n = ctypes.c_int()
        lib().oracle_get_temperatures(self._h, None, ctypes.byref(n))
        return n.value

    def observables(self):
        n = self.n
        E = np.zeros(n); M = np.zeros(n); rate = np.zeros(max(n - 1, 0))
        self._ck(lib().oracle_observables(self._h, _ptr(E, _dp), _ptr(M, _dp), _ptr(rate, _dp)))
        return E, M, rate

    def get_spins(self, temp_rank):
        out = np.zeros(self.N, dtype=np.int8)
        self._ck(lib().oracle_get_spins(self._h, temp_rank, _ptr(out, _i8p)))
        return out

    # --- test-only accessors ----------------------------------------------
    def get_spins_slot(self, slot):
        out = np.zeros(self.N, dtype=np.int8)
        self._ck(lib().oracle_get_spins_slot(self._h, slot, _ptr(out, _i8p)))
        return out

    def set_spins_slot(self, slot, s):
        s = np.ascontiguousarray(s, dtype=np.int8)
        assert s.size == self.N
        self._ck(lib().oracle_set_spins_slot(self._h, slot, _ptr(s, _i8p)))

    def get_field(self):
        out = np.zeros(self.N, dtype=np.int32)
        self._ck(lib().oracle_get_field(self._h, _ptr(out, _i32p)))
        return out

    def set_field(self, f):
        f = np.ascontiguousarray(f, dtype=np.int32)
        assert f.size == self.N
        self._ck(lib().oracle_set_field(self._h, _ptr(f, _i32p)))

    def thermal_moments(self, skip=0):
        """[n][5]: <e>, <e^2>, <|m|>, <m^2>, <m^4> per temperature rank over measurement steps [skip, steps)."""
        out = np.zeros((self.n, 5))
        self._ck(lib().oracle_thermal_moments(self._h, int(skip), _ptr(out, _dp)))
        return out

    def get_permutation(self):
        out = np.zeros(self.n, dtype=np.int32)
        self._ck(lib().oracle_get_permutation(self._h, _ptr(out, _i32p)))
        return out

    def set_permutation(self, t2r):
        t2r = np.ascontiguousarray(t2r, dtype=np.int32)
        assert t2r.size == self.n
        self._ck(lib().oracle_set_permutation(self._h, _ptr(t2r, _i32p)))

    def get_temperatures(self):
        out = np.zeros(self.n)
        n = ctypes.c_int()
        self._ck(lib().oracle_get_temperatures(self._h, _ptr(out, _dp), ctypes.byref(n)))
        return out

    def get_counters(self):
        a = ctypes.c_uint64(); b = ctypes.c_uint64()
        lib().oracle_get_counters(self._h, ctypes.byref(a), ctypes.byref(b))
        return a.value, b.value

    def set_counters(self, sweep_index, exchange_step):
        lib().oracle_set_counters(self._h, sweep_index, exchange_step)

    def get_energy_terms(self):
        n = self.n
        Eb = np.zeros(n, dtype=np.int64); Ef = np.zeros(n, dtype=np.int64); Ms = np.zeros(n, dtype=np.int64)
        self._ck(lib().oracle_get_energy_terms(self._h, _ptr(Eb, _i64p), _ptr(Ef, _i64p), _ptr(Ms, _i64p)))
        return Eb, Ef, Ms

    def get_timeseries(self):
        """(Eb, Ef, Msum), each int64 [steps, n], one row per exchange step since the last reset."""
        steps = int(lib().oracle_timeseries_steps(self._h))
        n = self.n
        Eb = np.zeros((steps, n), dtype=np.int64); Ef = np.zeros_like(Eb); Ms = np.zeros_like(Eb)
        if steps:
            self._ck(lib().oracle_get_timeseries(self._h, _ptr(Eb, _i64p), _ptr(Ef, _i64p), _ptr(Ms, _i64p)))
        return Eb, Ef, Ms

    def get_exchange_counts(self):
        n = self.n
        att = np.zeros(max(n - 1, 0), dtype=np.uint64); acc = np.zeros_like(att)
        lib().oracle_get_exchange_counts(self._h, _ptr(att, _u64p), _ptr(acc, _u64p))
        return att, acc

    def site_threshold(self, slot, x, y, z):
        return int(lib().oracle_site_threshold(self._h, slot, x, y, z))

    def bimodal_threshold(self, rank, k, b):
        return int(lib().oracle_bimodal_threshold(self._h, rank, k, b))

    def energy_from_terms(self, Eb, Ef):
        return float(lib().oracle_energy_from_terms(self._h, int(Eb), int(Ef)))

    def half_sweep(self, slot, colour, sweep_index):
        self._ck(lib().oracle_half_sweep(self._h, slot, colour, sweep_index))

    def exchange_step(self):
        self._ck(lib().oracle_exchange_step(self._h))


def thermal_observables(moments, T, N):
    """PAPER.md:249-260, Eq. 11-13 from the thermal moments of D disorder realisations at the same n temperatures.

    moments: [D][n][5] (Oracle.thermal_moments of each realisation), T: [D][n] or [n], N = L^3.
    Returns ([<|M|>], [C], [g]) per temperature: [.] = plain mean over the realisations;
    C_d = N / T^2 (<e^2> - <e>^2) per realisation (Eq. 12), g = (3 - [<M^4>] / [<M^2>]^2) / 2 (Eq. 13: the ratio is
    taken of the disorder averages, "an average at the disorder realization level")."""
    mom = np.asarray(moments, dtype=np.float64)
    if mom.ndim == 2:
        mom = mom[None]
    T = np.broadcast_to(np.asarray(T, dtype=np.float64), mom.shape[:2])
    absM = mom[:, :, 2].mean(axis=0)
    C = ((N / (T * T)) * (mom[:, :, 1] - mom[:, :, 0] * mom[:, :, 0])).mean(axis=0)
    g = 0.5 * (3.0 - mom[:, :, 4].mean(axis=0) / (mom[:, :, 3].mean(axis=0) ** 2))
    return absM, C, g
