"""ctypes wrapper around oracle/qcd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from the product package (paper_1310_7087_b200) and vice versa.
All numerics live in qcd_oracle.cpp; this file only marshals arguments (numpy arrays <-> pointers).
Canonical link layout: complex128 array of shape (V, D, N, N), lex site index = x0 + L0*(x1 + L1*(x2 + L2*x3)).
"""
import ctypes as C
import os

import numpy as np

from .build import build_oracle

_LIB = None

KIND_HB, KIND_OR = 0, 1
COLD, HOT = 0, 1
OPT_MAX_TRIALS, OPT_UNIFORM_MODE, OPT_STORE_FP32 = 0, 1, 2


class Field(C.Structure):
    """F = diag(exp(i*theta_c)) on every plaquette of plane (mu, nu), mu < nu (oracle-side definition)."""
    _fields_ = [("enabled", C.c_int), ("mu", C.c_int), ("nu", C.c_int), ("theta", C.c_double * 3)]


def make_field(mu, nu, theta):
    f = Field()
    f.enabled, f.mu, f.nu = 1, int(mu), int(nu)
    th = list(theta) + [0.0] * (3 - len(theta))
    for i in range(3):
        f.theta[i] = float(th[i])
    return f


def lib():
    global _LIB
    if _LIB is None:
        path = build_oracle()
        L = C.CDLL(path)
        L.oracle_create.restype = C.c_void_p
        L.oracle_create.argtypes = [C.c_int, C.POINTER(C.c_int), C.c_int]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.oracle_set_seed.argtypes = [C.c_void_p, C.c_uint64]
        L.oracle_set_sweep_counter.argtypes = [C.c_void_p, C.c_uint32]
        L.oracle_get_sweep_counter.argtypes = [C.c_void_p]
        L.oracle_get_sweep_counter.restype = C.c_uint32
        L.oracle_init.argtypes = [C.c_void_p, C.c_int, C.c_uint64]
        L.oracle_get_links.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_set_links.argtypes = [C.c_void_p, C.c_void_p]
        L.oracle_substep.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_substep_diag.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                          C.c_void_p]
        L.oracle_sweep.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_void_p]
        L.oracle_update_one_link.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_int, C.c_long, C.c_int, C.c_void_p,
                                             C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_staple.argtypes = [C.c_void_p, C.c_long, C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_measure.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_kp_samples.argtypes = [C.c_double, C.c_uint64, C.c_long, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.oracle_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_philox4x32_10_batch.argtypes = [C.c_void_p, C.c_void_p, C.c_long, C.c_void_p]
        L.oracle_keyed_block.argtypes = [C.c_uint64, C.c_long, C.c_uint32, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                         C.c_int, C.c_void_p]
        L.oracle_word_to_uniform.argtypes = [C.c_uint32, C.c_int]
        L.oracle_word_to_uniform.restype = C.c_double
        _LIB = L
    return _LIB


def num_threads():
    """OpenMP threads the oracle's site loops run on"""
    return int(lib().oracle_num_threads())


def _fptr(field):
    return C.byref(field) if field is not None else None


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def philox4x32_10_batch(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(c)
    lib().oracle_philox4x32_10_batch(c.ctypes.data, k.ctypes.data, len(c), out.ctypes.data)
    return out


def keyed_block(seed, lex, sweep, mu, parity, sg, hit, domain, draw):
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_keyed_block(seed, lex, sweep, mu, parity, sg, hit, domain, draw, out.ctypes.data)
    return out


def word_to_uniform(w, mode):
    return lib().oracle_word_to_uniform(int(w), int(mode))


def kp_samples(alpha, seed, n, max_trials=10, uniform_mode=0):
    g0 = np.zeros(n, dtype=np.float64)
    codes = np.zeros(n, dtype=np.uint8)
    lib().oracle_kp_samples(float(alpha), int(seed), int(n), int(max_trials), int(uniform_mode), g0.ctypes.data,
                            codes.ctypes.data)
    return g0, codes


class OracleLattice:
    def __init__(self, dims, Nc):
        self.dims = tuple(int(d) for d in dims)
        self.D = len(self.dims)
        self.N = int(Nc)
        self.V = int(np.prod(self.dims))
        arr = (C.c_int * self.D)(*self.dims)
        self._h = lib().oracle_create(self.D, arr, self.N)
        if not self._h:
            raise ValueError("oracle_create: invalid arguments %r Nc=%r" % (dims, Nc))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    # options
    def set_max_trials(self, n):
        assert lib().oracle_set_option(self._h, OPT_MAX_TRIALS, int(n)) == 0

    def set_fp32_shadow(self, on=True):
        """fp32 storage shadow: 23-bit uniforms in the heatbath and links rounded to float on every store."""
        lib().oracle_set_option(self._h, OPT_UNIFORM_MODE, 1 if on else 0)
        lib().oracle_set_option(self._h, OPT_STORE_FP32, 1 if on else 0)

    def set_seed(self, seed):
        lib().oracle_set_seed(self._h, int(seed))

    @property
    def sweep_counter(self):
        return int(lib().oracle_get_sweep_counter(self._h))

    @sweep_counter.setter
    def sweep_counter(self, s):
        lib().oracle_set_sweep_counter(self._h, int(s))

    # state
    def init(self, start, seed):
        lib().oracle_init(self._h, int(start), int(seed))

    def get_links(self):
        out = np.zeros((self.V, self.D, self.N, self.N), dtype=np.complex128)
        lib().oracle_get_links(self._h, out.ctypes.data)
        return out

    def set_links(self, links):
        a = np.ascontiguousarray(links, dtype=np.complex128)
        assert a.shape == (self.V, self.D, self.N, self.N), a.shape
        lib().oracle_set_links(self._h, a.ctypes.data)

    # updates
    def substep(self, beta, kind, hit, parity, mu, field=None, want_trials=False):
        trials = np.zeros((self.V, 3), dtype=np.uint8) if want_trials else None
        lib().oracle_substep(self._h, float(beta), int(kind), int(hit), int(parity), int(mu), _fptr(field),
                             trials.ctypes.data if want_trials else None)
        return trials

    def substep_diag(self, beta, kind, hit, parity, mu, field=None):
        """substep that also returns (trial codes (V,3), kmin (V,)): kmin = smallest subgroup projection norm k of each
        updated link (inf elsewhere) -- the conditioning of that update, used by the fp32 tolerance rule."""
        trials = np.zeros((self.V, 3), dtype=np.uint8)
        kmin = np.full(self.V, np.inf, dtype=np.float64)
        lib().oracle_substep_diag(self._h, float(beta), int(kind), int(hit), int(parity), int(mu), _fptr(field),
                                  trials.ctypes.data, kmin.ctypes.data)
        return trials, kmin

    def sweep(self, beta, n_hb, n_or, field=None):
        lib().oracle_sweep(self._h, float(beta), int(n_hb), int(n_or), _fptr(field))

    def update_one_link(self, beta, kind, hit, lex, mu, field=None):
        out = np.zeros((self.N, self.N), dtype=np.complex128)
        codes = np.zeros(3, dtype=np.uint8)
        kmin = C.c_double(0.0)
        lib().oracle_update_one_link(self._h, float(beta), int(kind), int(hit), int(lex), int(mu), _fptr(field),
                                     out.ctypes.data, codes.ctypes.data, C.byref(kmin))
        self.last_kmin = kmin.value
        return out, codes

    def staple(self, lex, mu, field=None):
        out = np.zeros((self.N, self.N), dtype=np.complex128)
        lib().oracle_staple(self._h, int(lex), int(mu), _fptr(field), out.ctypes.data)
        return out

    def measure(self, field=None):
        """returns (plaq_total, plaq_planes[D(D-1)/2], polyakov complex)"""
        npl = self.D * (self.D - 1) // 2
        tot = C.c_double(0.0)
        planes = np.zeros(npl, dtype=np.float64)
        poly = np.zeros(2, dtype=np.float64)
        lib().oracle_measure(self._h, _fptr(field), C.byref(tot), planes.ctypes.data, poly.ctypes.data)
        return tot.value, planes, complex(poly[0], poly[1])
