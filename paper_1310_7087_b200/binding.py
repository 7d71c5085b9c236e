"""Thin ctypes binding of include/qcd.h -- argument marshalling only; every step of the path runs in the CUDA
kernels of libqcd_b200.so.  There is no CPU fallback: if the library is missing or a call fails, this raises.

PyTorch is used only for device memory (a uint8 tensor handed to qcd_lattice_create) and for the stream.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libqcd_b200.so")

QCD_OK, QCD_ERR_INVALID_ARG, QCD_ERR_UNSUPPORTED, QCD_ERR_ALLOC, QCD_ERR_CUDA, QCD_ERR_STATE = 0, 1, 2, 3, 4, 5
QCD_FP32, QCD_FP64 = 0, 1
QCD_FLAG_COMPRESS12 = 1
QCD_COLD, QCD_HOT = 0, 1
QCD_KIND_HB, QCD_KIND_OR = 0, 1
QCD_OPT_KP_MAX_TRIALS, QCD_OPT_DEBUG_TRIALS, QCD_OPT_PROFILE, QCD_OPT_BULK_COPY, QCD_OPT_ALTERNATE_ORDER, QCD_OPT_EXCHANGE_ROWS01 = 0, 1, 2, 3, 4, 5
QCD_NOALLOC_MAX_PARTIALS = 1 << 20

# every symbol include/qcd.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "qcd_lattice_bytes", "qcd_lattice_create", "qcd_lattice_destroy", "qcd_init", "qcd_sweep", "qcd_measure",
    "qcd_get_links", "qcd_set_links", "qcd_get_sweep_counter", "qcd_set_sweep_counter", "qcd_get_seed", "qcd_set_seed",
    "qcd_set_option", "qcd_debug_substep", "qcd_debug_get_trials", "qcd_debug_philox", "qcd_debug_hb_math", "qcd_get_profile",
    "qcd_reset_profile", "qcd_get_launch_count", "qcd_measure_accumulate", "qcd_sweep_measure", "qcd_sweep_measure_accumulate", "qcd_accum_get", "qcd_accum_reset", "qcd_probe_fma_tflops", "qcd_probe_copy_gbs", "qcd_last_error",
    "qcd_version", "qcd_measure_plaquette_noalloc",
    "qcd_slab_bytes", "qcd_slab_create", "qcd_slab_halo_bytes", "qcd_slab_halo_pack", "qcd_slab_halo_unpack", "qcd_slab_measure_sums",
    "qcd_split_create", "qcd_split_destroy", "qcd_split_parts", "qcd_split_halo_bytes", "qcd_split_init", "qcd_split_sweep",
    "qcd_split_substep", "qcd_split_measure", "qcd_split_get_links", "qcd_split_set_links", "qcd_split_set_seed",
    "qcd_split_set_sweep_counter", "qcd_split_get_sweep_counter", "qcd_split_synchronize",
    "qcd_on_bytes", "qcd_on_create", "qcd_on_destroy", "qcd_on_init", "qcd_on_sweep", "qcd_on_half_sweep", "qcd_on_measure",
    "qcd_on_get_counts", "qcd_on_get_field", "qcd_on_set_field", "qcd_on_set_seed", "qcd_on_set_sweep_counter", "qcd_on_get_sweep_counter",
]


class qcd_field_t(C.Structure):
    _fields_ = [("enabled", C.c_int), ("mu", C.c_int), ("nu", C.c_int), ("theta", C.c_double * 3)]


class QcdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("qcd error %d: %s" % (code, msg))
        self.code = code


_lib = None


def lib():
    """Load libqcd_b200.so (built by paper_1310_7087_b200.build / __graft_entry__.build()).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libqcd_b200.so is not built: run `python -m paper_1310_7087_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    p, i, u, d, sz = C.c_void_p, C.c_int, C.c_uint, C.c_double, C.c_size_t
    ip, dp = C.POINTER(C.c_int), C.POINTER(C.c_double)
    fp = C.POINTER(qcd_field_t)
    L.qcd_lattice_bytes.restype = sz
    L.qcd_lattice_bytes.argtypes = [i, ip, i, i, u]
    L.qcd_lattice_create.argtypes = [i, ip, i, i, u, p, sz, p, C.POINTER(p)]
    L.qcd_lattice_destroy.argtypes = [p]
    L.qcd_init.argtypes = [p, i, C.c_uint64]
    L.qcd_sweep.argtypes = [p, d, i, i, fp]
    L.qcd_measure.argtypes = [p, fp, dp, dp, dp]
    L.qcd_measure_accumulate.argtypes = [p, fp]
    L.qcd_measure_plaquette_noalloc.argtypes = [p, fp, p]
    L.qcd_sweep_measure.argtypes = [p, d, i, i, fp, dp, dp, dp]
    L.qcd_sweep_measure_accumulate.argtypes = [p, d, i, i, fp]
    L.qcd_accum_get.argtypes = [p, C.POINTER(C.c_uint64), dp, dp, i]
    L.qcd_accum_reset.argtypes = [p]
    L.qcd_get_links.argtypes = [p, p, sz, i]
    L.qcd_set_links.argtypes = [p, p, sz, i]
    L.qcd_get_sweep_counter.argtypes = [p, C.POINTER(C.c_uint32)]
    L.qcd_set_sweep_counter.argtypes = [p, C.c_uint32]
    L.qcd_get_seed.argtypes = [p, C.POINTER(C.c_uint64)]
    L.qcd_set_seed.argtypes = [p, C.c_uint64]
    L.qcd_set_option.argtypes = [p, i, i]
    L.qcd_debug_substep.argtypes = [p, d, i, i, i, i, fp]
    L.qcd_debug_get_trials.argtypes = [p, p, sz]
    L.qcd_debug_philox.argtypes = [p, p, sz, p, i]
    L.qcd_debug_hb_math.argtypes = [p, sz, p]
    L.qcd_get_profile.argtypes = [p, i, dp, C.POINTER(C.c_uint64)]
    L.qcd_reset_profile.argtypes = [p]
    L.qcd_get_launch_count.argtypes = [p, C.POINTER(C.c_uint64)]
    L.qcd_probe_fma_tflops.argtypes = [i, dp]
    L.qcd_probe_copy_gbs.argtypes = [sz, i, dp]
    L.qcd_slab_bytes.restype = sz
    L.qcd_slab_bytes.argtypes = [i, ip, i, i, u, i, i]
    L.qcd_slab_create.argtypes = [i, ip, i, i, u, i, i, p, sz, p, C.POINTER(p)]
    L.qcd_slab_halo_bytes.restype = sz
    L.qcd_slab_halo_bytes.argtypes = [p]
    L.qcd_slab_halo_pack.argtypes = [p, i, i, i, p, sz]
    L.qcd_slab_halo_unpack.argtypes = [p, i, i, i, p, sz]
    L.qcd_slab_measure_sums.argtypes = [p, fp, dp, dp]
    L.qcd_split_create.argtypes = [i, ip, i, i, u, i, ip, ip, C.POINTER(p)]
    L.qcd_split_destroy.argtypes = [p]
    L.qcd_split_parts.argtypes = [p, ip, ip, ip, i]
    L.qcd_split_halo_bytes.argtypes = [p, C.POINTER(sz)]
    L.qcd_split_init.argtypes = [p, i, C.c_uint64]
    L.qcd_split_sweep.argtypes = [p, d, i, i, fp]
    L.qcd_split_substep.argtypes = [p, d, i, i, i, i, fp]
    L.qcd_split_measure.argtypes = [p, fp, dp, dp, dp]
    L.qcd_split_get_links.argtypes = [p, p, sz]
    L.qcd_split_set_links.argtypes = [p, p, sz]
    L.qcd_split_set_seed.argtypes = [p, C.c_uint64]
    L.qcd_split_set_sweep_counter.argtypes = [p, C.c_uint32]
    L.qcd_split_get_sweep_counter.argtypes = [p, C.POINTER(C.c_uint32)]
    L.qcd_split_synchronize.argtypes = [p]
    L.qcd_on_bytes.restype = sz
    L.qcd_on_bytes.argtypes = [i, ip, i, i]
    L.qcd_on_create.argtypes = [i, ip, i, i, p, sz, p, C.POINTER(p)]
    L.qcd_on_destroy.argtypes = [p]
    L.qcd_on_init.argtypes = [p, i, C.c_uint64]
    L.qcd_on_sweep.argtypes = [p, d, d, d, i]
    L.qcd_on_half_sweep.argtypes = [p, i, d, d, d, i]
    L.qcd_on_measure.argtypes = [p, dp, dp, dp]
    L.qcd_on_get_counts.argtypes = [p, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.qcd_on_get_field.argtypes = [p, p, sz, i]
    L.qcd_on_set_field.argtypes = [p, p, sz, i]
    L.qcd_on_set_seed.argtypes = [p, C.c_uint64]
    L.qcd_on_set_sweep_counter.argtypes = [p, C.c_uint32]
    L.qcd_on_get_sweep_counter.argtypes = [p, C.POINTER(C.c_uint32)]
    L.qcd_last_error.restype = C.c_char_p
    L.qcd_version.restype = C.c_char_p
    _lib = L
    return L


def _check(rc):
    if rc != QCD_OK:
        raise QcdError(rc, lib().qcd_last_error().decode())


def make_field(mu, nu, theta):
    f = qcd_field_t()
    f.enabled, f.mu, f.nu = 1, int(mu), int(nu)
    th = list(theta) + [0.0] * (3 - len(theta))
    for k in range(3):
        f.theta[k] = float(th[k])
    return f


def _fref(field):
    return C.byref(field) if field is not None else None


def qcd_lattice_bytes(dims, Nc, precision, flags=0):
    arr = (C.c_int * len(dims))(*[int(x) for x in dims])
    return int(lib().qcd_lattice_bytes(len(dims), arr, int(Nc), int(precision), int(flags)))


def qcd_probe_fma_tflops(precision):
    out = C.c_double(0.0)
    _check(lib().qcd_probe_fma_tflops(int(precision), C.byref(out)))
    return out.value


def qcd_probe_copy_gbs(nbytes, reps=10):
    out = C.c_double(0.0)
    _check(lib().qcd_probe_copy_gbs(int(nbytes), int(reps), C.byref(out)))
    return out.value


def qcd_debug_philox(ctr, key, impl=0):
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    assert len(ctr) == len(key)
    out = np.zeros_like(ctr)
    _check(lib().qcd_debug_philox(ctr.ctypes.data, key.ctypes.data, len(ctr), out.ctypes.data, int(impl)))
    return out


def qcd_debug_hb_math(words):
    """rows (ln u, cos^2 2 pi u, sin 2 pi u, cos 2 pi u, sqrt u, 1/sqrt u, 1/u), u = (w + 1/2) 2^-32, computed on the device"""
    words = np.ascontiguousarray(words, dtype=np.uint32).reshape(-1)
    out = np.zeros((len(words), 7), dtype=np.float64)
    _check(lib().qcd_debug_hb_math(words.ctypes.data, len(words), out.ctypes.data))
    return out


class Lattice:
    """One lattice handle.  Device memory comes from a torch uint8 tensor, the stream from torch.
    slab = (offset, extent): a part of the lattice of global extents `dims`, split along direction D-2 (qcd_slab_create);
    then dims / V describe the part's own block and global_dims the whole lattice.
    mem: a torch uint8 CUDA tensor to use as the lattice's memory (at least nbytes long) instead of allocating one."""

    def __init__(self, dims, Nc, precision=QCD_FP64, flags=0, device="cuda:0", library_alloc=False, slab=None, mem=None):
        import torch
        self.global_dims = tuple(int(x) for x in dims)
        self.D, self.Nc, self.precision, self.flags = len(self.global_dims), int(Nc), int(precision), int(flags)
        self.slab = None if slab is None else (int(slab[0]), int(slab[1]))
        self.dims = self.global_dims if slab is None else tuple(self.slab[1] if k == self.D - 2 else x for k, x in enumerate(self.global_dims))
        self.V = int(np.prod(self.dims))
        self._h = C.c_void_p()
        arr = (C.c_int * self.D)(*self.global_dims)
        if slab is None:
            nbytes = lib().qcd_lattice_bytes(self.D, arr, self.Nc, self.precision, self.flags)
        else:
            nbytes = lib().qcd_slab_bytes(self.D, arr, self.Nc, self.precision, self.flags, self.slab[0], self.slab[1])
        self._torch = torch
        self._mem = None
        self._device = torch.device(device)
        mem_ptr, stream_ptr = None, None
        self.nbytes = int(nbytes)
        if nbytes and not library_alloc:
            with torch.cuda.device(self._device):
                if mem is None:
                    self._mem = torch.empty(int(nbytes), dtype=torch.uint8, device=self._device)
                else:
                    assert mem.dtype == torch.uint8 and mem.is_cuda and mem.numel() >= int(nbytes) and mem.data_ptr() % 256 == 0
                    self._mem = mem
                mem_ptr = self._mem.data_ptr()
                stream_ptr = torch.cuda.current_stream().cuda_stream
        elif nbytes:
            torch.cuda.set_device(self._device)
        if slab is None:
            _check(lib().qcd_lattice_create(self.D, arr, self.Nc, self.precision, self.flags, mem_ptr, int(nbytes), stream_ptr,
                                            C.byref(self._h)))
        else:
            _check(lib().qcd_slab_create(self.D, arr, self.Nc, self.precision, self.flags, self.slab[0], self.slab[1], mem_ptr,
                                         int(nbytes), stream_ptr, C.byref(self._h)))
        self._rows = self.Nc                      # rows of a link in the exchange layout (2 with QCD_OPT_EXCHANGE_ROWS01)
        self.np_real = np.float32 if self.precision == QCD_FP32 else np.float64
        self.np_complex = np.complex64 if self.precision == QCD_FP32 else np.complex128

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().qcd_lattice_destroy(self._h)
            self._h = C.c_void_p()
        self._mem = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- the C ABI, same names
    def qcd_init(self, start, seed):
        _check(lib().qcd_init(self._h, int(start), int(seed)))

    def qcd_sweep(self, beta, n_hb, n_or, field=None):
        _check(lib().qcd_sweep(self._h, float(beta), int(n_hb), int(n_or), _fref(field)))

    def qcd_measure(self, field=None, plaquette=True, polyakov=True):
        npl = self.D * (self.D - 1) // 2
        tot = C.c_double(0.0)
        planes = (C.c_double * npl)()
        poly = (C.c_double * 2)()
        _check(lib().qcd_measure(self._h, _fref(field), C.byref(tot) if plaquette else None, planes if plaquette else None,
                                 poly if polyakov else None))
        return tot.value, np.array(planes[:]), complex(poly[0], poly[1])

    def qcd_measure_plaquette_noalloc(self, out, field=None):
        """Plane plaquettes (qcd_measure's `planes`) written to `out`, a float64 CUDA tensor of D(D-1)/2 elements that the
        caller owns, without any device allocation by the library -- for programs whose own allocator holds the GPU's memory
        or which cannot afford a cudaMalloc in their loop (include/qcd.h says who and why).  The partial sums live in one
        8 MiB array per GPU built into the library, shared by all calls: lattices beyond QCD_NOALLOC_MAX_PARTIALS partial sums
        are refused, and calls that may overlap on the GPU must be ordered by the caller.  Asynchronous on the lattice's
        stream; the lattice's device must be current.  Call it once during set-up before any stream capture."""
        assert out.is_cuda and out.dtype == self._torch.float64 and out.is_contiguous() and out.numel() >= self.D * (self.D - 1) // 2
        _check(lib().qcd_measure_plaquette_noalloc(self._h, _fref(field), out.data_ptr()))

    def qcd_sweep_measure(self, beta, n_hb, n_or, field=None):
        """one working sweep: qcd_sweep + the observables of the new configuration (plaquette fused into the last pass)"""
        npl = self.D * (self.D - 1) // 2
        tot = C.c_double(0.0)
        planes = (C.c_double * npl)()
        poly = (C.c_double * 2)()
        _check(lib().qcd_sweep_measure(self._h, float(beta), int(n_hb), int(n_or), _fref(field), C.byref(tot), planes, poly))
        return tot.value, np.array(planes[:]), complex(poly[0], poly[1])

    def qcd_sweep_measure_accumulate(self, beta, n_hb, n_or, field=None):
        _check(lib().qcd_sweep_measure_accumulate(self._h, float(beta), int(n_hb), int(n_or), _fref(field)))

    def qcd_measure_accumulate(self, field=None):
        _check(lib().qcd_measure_accumulate(self._h, _fref(field)))

    def qcd_accum_reset(self):
        _check(lib().qcd_accum_reset(self._h))

    def qcd_accum_get(self):
        """(count, sums, sums of squares) of the D(D-1)/2 plane plaquettes, Re L, Im L, |L|"""
        nq = self.D * (self.D - 1) // 2 + 3
        n = C.c_uint64(0)
        s1, s2 = (C.c_double * nq)(), (C.c_double * nq)()
        _check(lib().qcd_accum_get(self._h, C.byref(n), s1, s2, nq))
        return int(n.value), np.array(s1[:]), np.array(s2[:])

    def qcd_get_links(self):
        """canonical (V, D, N, N) complex array in the lattice's precision (host)"""
        out = np.zeros((self.V, self.D, self._rows, self.Nc), dtype=self.np_complex)
        _check(lib().qcd_get_links(self._h, out.ctypes.data, out.nbytes, 0))
        return out

    def qcd_set_links(self, links):
        a = np.ascontiguousarray(links, dtype=self.np_complex)
        assert a.shape == (self.V, self.D, self._rows, self.Nc), a.shape
        _check(lib().qcd_set_links(self._h, a.ctypes.data, a.nbytes, 0))

    def qcd_get_links_ptr(self, ptr, nbytes, is_device):
        _check(lib().qcd_get_links(self._h, int(ptr), int(nbytes), int(is_device)))

    def qcd_set_links_ptr(self, ptr, nbytes, is_device):
        _check(lib().qcd_set_links(self._h, int(ptr), int(nbytes), int(is_device)))

    @property
    def canonical_bytes(self):
        return self.V * self.D * self._rows * self.Nc * 2 * (4 if self.precision == QCD_FP32 else 8)

    def qcd_get_sweep_counter(self):
        out = C.c_uint32(0)
        _check(lib().qcd_get_sweep_counter(self._h, C.byref(out)))
        return out.value

    def qcd_set_sweep_counter(self, v):
        _check(lib().qcd_set_sweep_counter(self._h, int(v)))

    def qcd_get_seed(self):
        out = C.c_uint64(0)
        _check(lib().qcd_get_seed(self._h, C.byref(out)))
        return out.value

    def qcd_set_seed(self, seed):
        _check(lib().qcd_set_seed(self._h, int(seed)))

    def qcd_set_option(self, key, value):
        _check(lib().qcd_set_option(self._h, int(key), int(value)))
        if int(key) == QCD_OPT_EXCHANGE_ROWS01:
            self._rows = 2 if value else self.Nc

    def qcd_debug_substep(self, beta, kind, hit, parity, mu, field=None):
        _check(lib().qcd_debug_substep(self._h, float(beta), int(kind), int(hit), int(parity), int(mu), _fref(field)))

    def qcd_debug_get_trials(self):
        out = np.zeros((self.V, 3), dtype=np.uint8)
        _check(lib().qcd_debug_get_trials(self._h, out.ctypes.data, out.nbytes))
        return out

    # ---- slab primitives (a part of a divided lattice)
    def qcd_slab_halo_bytes(self):
        return int(lib().qcd_slab_halo_bytes(self._h))

    def qcd_slab_halo_pack(self, parity, mu, side, device_ptr, nbytes):
        _check(lib().qcd_slab_halo_pack(self._h, int(parity), int(mu), int(side), int(device_ptr), int(nbytes)))

    def qcd_slab_halo_unpack(self, parity, mu, side, device_ptr, nbytes):
        _check(lib().qcd_slab_halo_unpack(self._h, int(parity), int(mu), int(side), int(device_ptr), int(nbytes)))

    def qcd_slab_measure_sums(self, field=None):
        npl = self.D * (self.D - 1) // 2
        planes = (C.c_double * npl)()
        poly = (C.c_double * 2)()
        _check(lib().qcd_slab_measure_sums(self._h, _fref(field), planes, poly))
        return np.array(planes[:]), complex(poly[0], poly[1])

    def qcd_get_profile(self, kind):
        ms = C.c_double(0.0)
        n = C.c_uint64(0)
        _check(lib().qcd_get_profile(self._h, int(kind), C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def qcd_reset_profile(self):
        _check(lib().qcd_reset_profile(self._h))

    def qcd_get_launch_count(self):
        n = C.c_uint64(0)
        _check(lib().qcd_get_launch_count(self._h, C.byref(n)))
        return int(n.value)


class SplitLattice:
    """A lattice divided into parts along direction D-2, all parts in this process (qcd_split_*): one part per entry of
    `devices` (CUDA device ordinals; default: n_parts parts on the current device)."""

    def __init__(self, dims, Nc, precision=QCD_FP64, flags=0, n_parts=2, extents=None, devices=None):
        self.dims = tuple(int(x) for x in dims)
        self.D, self.Nc, self.precision, self.flags = len(self.dims), int(Nc), int(precision), int(flags)
        self.V = int(np.prod(self.dims))
        self._h = C.c_void_p()
        arr = (C.c_int * self.D)(*self.dims)
        ext = (C.c_int * n_parts)(*[int(e) for e in extents]) if extents is not None else None
        dev = (C.c_int * n_parts)(*[int(e) for e in devices]) if devices is not None else None
        _check(lib().qcd_split_create(self.D, arr, self.Nc, self.precision, self.flags, int(n_parts), ext, dev, C.byref(self._h)))
        self.np_complex = np.complex64 if self.precision == QCD_FP32 else np.complex128

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().qcd_split_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def qcd_split_parts(self):
        n = C.c_int(0)
        _check(lib().qcd_split_parts(self._h, C.byref(n), None, None, 0))
        off, ext = (C.c_int * n.value)(), (C.c_int * n.value)()
        _check(lib().qcd_split_parts(self._h, C.byref(n), off, ext, n.value))
        return list(off), list(ext)

    def qcd_split_halo_bytes(self):
        out = C.c_size_t(0)
        _check(lib().qcd_split_halo_bytes(self._h, C.byref(out)))
        return int(out.value)

    def qcd_split_init(self, start, seed):
        _check(lib().qcd_split_init(self._h, int(start), int(seed)))

    def qcd_split_sweep(self, beta, n_hb, n_or, field=None):
        _check(lib().qcd_split_sweep(self._h, float(beta), int(n_hb), int(n_or), _fref(field)))

    def qcd_split_substep(self, beta, kind, hit, parity, mu, field=None):
        _check(lib().qcd_split_substep(self._h, float(beta), int(kind), int(hit), int(parity), int(mu), _fref(field)))

    def qcd_split_measure(self, field=None):
        npl = self.D * (self.D - 1) // 2
        tot = C.c_double(0.0)
        planes = (C.c_double * npl)()
        poly = (C.c_double * 2)()
        _check(lib().qcd_split_measure(self._h, _fref(field), C.byref(tot), planes, poly))
        return tot.value, np.array(planes[:]), complex(poly[0], poly[1])

    def qcd_split_get_links(self):
        out = np.zeros((self.V, self.D, self.Nc, self.Nc), dtype=self.np_complex)
        _check(lib().qcd_split_get_links(self._h, out.ctypes.data, out.nbytes))
        return out

    def qcd_split_set_links(self, links):
        a = np.ascontiguousarray(links, dtype=self.np_complex)
        assert a.shape == (self.V, self.D, self.Nc, self.Nc), a.shape
        _check(lib().qcd_split_set_links(self._h, a.ctypes.data, a.nbytes))

    def qcd_split_set_seed(self, seed):
        _check(lib().qcd_split_set_seed(self._h, int(seed)))

    def qcd_split_set_sweep_counter(self, v):
        _check(lib().qcd_split_set_sweep_counter(self._h, int(v)))

    def qcd_split_get_sweep_counter(self):
        out = C.c_uint32(0)
        _check(lib().qcd_split_get_sweep_counter(self._h, C.byref(out)))
        return out.value

    def qcd_split_synchronize(self):
        _check(lib().qcd_split_synchronize(self._h))


class OnLattice:
    """The O(N) scalar model on lattice sites (qcd_on_*): N-vectors, multi-hit Metropolis on the checkerboard."""

    def __init__(self, dims, N, precision=QCD_FP64, device="cuda:0"):
        import torch
        self.dims = tuple(int(x) for x in dims)
        self.D, self.N, self.precision = len(self.dims), int(N), int(precision)
        self.V = int(np.prod(self.dims))
        self._h = C.c_void_p()
        arr = (C.c_int * self.D)(*self.dims)
        nbytes = lib().qcd_on_bytes(self.D, arr, self.N, self.precision)
        self._mem, mem_ptr, stream_ptr = None, None, None
        dev = torch.device(device)
        if nbytes:
            with torch.cuda.device(dev):
                self._mem = torch.empty(int(nbytes), dtype=torch.uint8, device=dev)
                mem_ptr = self._mem.data_ptr()
                stream_ptr = torch.cuda.current_stream().cuda_stream
        _check(lib().qcd_on_create(self.D, arr, self.N, self.precision, mem_ptr, int(nbytes), stream_ptr, C.byref(self._h)))
        self.np_real = np.float32 if self.precision == QCD_FP32 else np.float64

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().qcd_on_destroy(self._h)
            self._h = C.c_void_p()
        self._mem = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def qcd_on_init(self, start, seed):
        _check(lib().qcd_on_init(self._h, int(start), int(seed)))

    def qcd_on_sweep(self, kappa, lam, delta, nhit):
        _check(lib().qcd_on_sweep(self._h, float(kappa), float(lam), float(delta), int(nhit)))

    def qcd_on_half_sweep(self, parity, kappa, lam, delta, nhit):
        _check(lib().qcd_on_half_sweep(self._h, int(parity), float(kappa), float(lam), float(delta), int(nhit)))

    def qcd_on_measure(self):
        p2, lk = C.c_double(0.0), C.c_double(0.0)
        mag = (C.c_double * self.N)()
        _check(lib().qcd_on_measure(self._h, C.byref(p2), C.byref(lk), mag))
        return p2.value, lk.value, np.array(mag[:])

    def qcd_on_get_counts(self):
        a, t = C.c_uint64(0), C.c_uint64(0)
        _check(lib().qcd_on_get_counts(self._h, C.byref(a), C.byref(t)))
        return int(a.value), int(t.value)

    def qcd_on_get_field(self):
        out = np.zeros((self.V, self.N), dtype=self.np_real)
        _check(lib().qcd_on_get_field(self._h, out.ctypes.data, out.nbytes, 0))
        return out

    def qcd_on_set_field(self, phi):
        a = np.ascontiguousarray(phi, dtype=self.np_real)
        assert a.shape == (self.V, self.N), a.shape
        _check(lib().qcd_on_set_field(self._h, a.ctypes.data, a.nbytes, 0))

    def qcd_on_set_seed(self, seed):
        _check(lib().qcd_on_set_seed(self._h, int(seed)))

    def qcd_on_set_sweep_counter(self, v):
        _check(lib().qcd_on_set_sweep_counter(self._h, int(v)))

    def qcd_on_get_sweep_counter(self):
        out = C.c_uint32(0)
        _check(lib().qcd_on_get_sweep_counter(self._h, C.byref(out)))
        return out.value
