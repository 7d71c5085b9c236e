"""ctypes wrapper around oracle/on_oracle.cpp (the O(N) model, multi-hit Metropolis) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it imports nothing from the
product package.  All numerics live in on_oracle.cpp; this file only marshals arguments.
Canonical field layout: float64 array of shape (V, N), lex site index = x0 + L0*(x1 + L1*(x2 + L2*x3)).
"""
import ctypes as C

import numpy as np

from .build import build_on_oracle

_LIB = None
COLD, HOT = 0, 1


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build_on_oracle())
        L.on_oracle_create.restype = C.c_void_p
        L.on_oracle_create.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int]
        L.on_oracle_destroy.argtypes = [C.c_void_p]
        L.on_oracle_set_fp32.argtypes = [C.c_void_p, C.c_int]
        L.on_oracle_set_seed.argtypes = [C.c_void_p, C.c_uint64]
        L.on_oracle_set_sweep_counter.argtypes = [C.c_void_p, C.c_uint32]
        L.on_oracle_get_sweep_counter.argtypes = [C.c_void_p]
        L.on_oracle_get_sweep_counter.restype = C.c_uint32
        L.on_oracle_get_field.argtypes = [C.c_void_p, C.c_void_p]
        L.on_oracle_set_field.argtypes = [C.c_void_p, C.c_void_p]
        L.on_oracle_counts.argtypes = [C.c_void_p, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong)]
        L.on_oracle_init.argtypes = [C.c_void_p, C.c_int, C.c_uint64]
        L.on_oracle_half_sweep.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int]
        L.on_oracle_sweep.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_int]
        L.on_oracle_action.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.on_oracle_action.restype = C.c_double
        L.on_oracle_measure.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p]
        L.on_oracle_block_numbers.argtypes = [C.c_uint64, C.c_long, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_void_p]
        L.on_oracle_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        _LIB = L
    return _LIB


def num_threads():
    return int(lib().on_oracle_num_threads())


def block_numbers(seed, lex, sweep, parity, hit, domain):
    out = np.zeros(5, dtype=np.uint32)
    lib().on_oracle_block_numbers(int(seed), int(lex), int(sweep), int(parity), int(hit), int(domain), out.ctypes.data)
    return out


def philox4x32_10(ctr, key):
    c, k = np.asarray(ctr, dtype=np.uint32).copy(), np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().on_oracle_philox(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


class OnOracle:
    def __init__(self, dims, N):
        self.dims = tuple(int(d) for d in dims)
        self.D, self.N = len(self.dims), int(N)
        self.V = int(np.prod(self.dims))
        arr = (C.c_int * self.D)(*self.dims)
        self._h = lib().on_oracle_create(self.D, arr, self.N)
        if not self._h:
            raise ValueError("on_oracle_create: invalid arguments %r N=%r" % (dims, N))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().on_oracle_destroy(self._h)
            self._h = None

    def set_fp32_shadow(self, on=True):
        lib().on_oracle_set_fp32(self._h, 1 if on else 0)

    def set_seed(self, seed):
        lib().on_oracle_set_seed(self._h, int(seed))

    @property
    def sweep_counter(self):
        return int(lib().on_oracle_get_sweep_counter(self._h))

    @sweep_counter.setter
    def sweep_counter(self, s):
        lib().on_oracle_set_sweep_counter(self._h, int(s))

    def init(self, start, seed):
        lib().on_oracle_init(self._h, int(start), int(seed))

    def get_field(self):
        out = np.zeros((self.V, self.N), dtype=np.float64)
        lib().on_oracle_get_field(self._h, out.ctypes.data)
        return out

    def set_field(self, phi):
        a = np.ascontiguousarray(phi, dtype=np.float64)
        assert a.shape == (self.V, self.N), a.shape
        lib().on_oracle_set_field(self._h, a.ctypes.data)

    def half_sweep(self, parity, kappa, lam, delta, nhit):
        lib().on_oracle_half_sweep(self._h, int(parity), float(kappa), float(lam), float(delta), int(nhit))

    def sweep(self, kappa, lam, delta, nhit):
        lib().on_oracle_sweep(self._h, float(kappa), float(lam), float(delta), int(nhit))

    def action(self, kappa, lam):
        return float(lib().on_oracle_action(self._h, float(kappa), float(lam)))

    def counts(self):
        a, t = C.c_ulonglong(0), C.c_ulonglong(0)
        lib().on_oracle_counts(self._h, C.byref(a), C.byref(t))
        return int(a.value), int(t.value)

    def measure(self):
        """(phi2, link energy, magnetisation vector)"""
        p2, lk = C.c_double(0.0), C.c_double(0.0)
        mag = np.zeros(self.N, dtype=np.float64)
        lib().on_oracle_measure(self._h, C.byref(p2), C.byref(lk), mag.ctypes.data)
        return p2.value, lk.value, mag
