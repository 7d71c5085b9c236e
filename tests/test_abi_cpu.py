"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/qcd.h declares, validates arguments
before touching the device, and fails loudly (no CPU fallback) when there is no GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def q():
    import paper_1310_7087_b200 as q
    from paper_1310_7087_b200.build import build_cuda
    build_cuda()
    return q


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "qcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qcd_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(q):
    names = _declared_functions()
    assert len(names) >= 20
    lib = q.lib()
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(q.SYMBOLS)
    assert b"sm_100a" in lib.qcd_version()


def test_lattice_bytes(q):
    # internal layout: 2 parities x D directions x NP planes x roundup(V/2, 32) vectors
    assert q.qcd_lattice_bytes((32, 32, 32, 32), 3, q.QCD_FP32, q.QCD_FLAG_COMPRESS12) == 4 * 32 ** 4 * 48
    assert q.qcd_lattice_bytes((32, 32, 32, 32), 3, q.QCD_FP64, 0) == 4 * 32 ** 4 * 144
    assert q.qcd_lattice_bytes((48, 48, 48, 8), 2, q.QCD_FP32, 0) == 4 * 48 ** 3 * 8 * 16
    assert q.qcd_lattice_bytes((64, 64, 64, 64), 3, q.QCD_FP64, 0) == 4 * 64 ** 4 * 144
    # 128^4: each (parity, direction) array is addressed with 32 bits, the array bases are 64-bit: 51.5 GB of 12-real fp32
    # links and 154.6 GB of 18-real fp64 links (the largest lattice of one B200) are both within the indexing; V > 2^31 is not
    assert q.qcd_lattice_bytes((128, 128, 128, 128), 3, q.QCD_FP32, q.QCD_FLAG_COMPRESS12) == 4 * 128 ** 4 * 48
    assert q.qcd_lattice_bytes((128, 128, 128, 128), 3, q.QCD_FP64, 0) == 4 * 128 ** 4 * 144
    assert q.qcd_lattice_bytes((256, 256, 256, 128), 2, q.QCD_FP32, 0) == 4 * 2 ** 31 * 16
    assert q.qcd_lattice_bytes((256, 256, 256, 256), 2, q.QCD_FP32, 0) == 0
    assert q.qcd_lattice_bytes((6, 4), 2, q.QCD_FP64, 0) == 2 * 2 * 2 * 32 * 16       # V/2 = 12 padded to 32
    for bad in [((5, 4), 2, 1, 0), ((4,), 2, 1, 0), ((4, 4, 4, 4, 4), 2, 1, 0), ((4, 4), 4, 1, 0), ((4, 4), 2, 2, 0),
                ((4, 4), 2, 1, 1), ((0, 4), 2, 1, 0), ((4, 4), 3, 1, 2)]:
        assert q.qcd_lattice_bytes(*bad) == 0, bad


def test_create_rejects_bad_arguments_before_touching_the_device(q):
    lib = q.lib()
    h = C.c_void_p()
    dims = (C.c_int * 2)(5, 4)
    assert lib.qcd_lattice_create(2, dims, 2, 1, 0, None, 0, None, C.byref(h)) == q.QCD_ERR_INVALID_ARG
    assert b"dims" in lib.qcd_last_error()
    dims = (C.c_int * 2)(4, 4)
    assert lib.qcd_lattice_create(2, dims, 2, 1, 1, None, 0, None, C.byref(h)) == q.QCD_ERR_UNSUPPORTED
    assert lib.qcd_lattice_create(2, dims, 2, 1, 0, C.c_void_p(256), 16, None, C.byref(h)) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_lattice_create(2, dims, 2, 1, 0, C.c_void_p(8), 1 << 20, None, C.byref(h)) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_lattice_create(2, dims, 2, 1, 0, None, 0, None, None) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_init(None, 0, 0) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_sweep(None, 1.0, 1, 1, None) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_lattice_destroy(None) == q.QCD_OK


def test_no_gpu_means_loud_failure(q):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = q.lib()
    h = C.c_void_p()
    dims = (C.c_int * 2)(4, 4)
    rc = lib.qcd_lattice_create(2, dims, 2, 1, 0, None, 0, None, C.byref(h))
    assert rc in (q.QCD_ERR_ALLOC, q.QCD_ERR_CUDA) and not h.value
    assert len(lib.qcd_last_error()) > 0
    out = C.c_double(0.0)
    assert lib.qcd_probe_fma_tflops(0, C.byref(out)) != q.QCD_OK


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1310_7087_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "qcd_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1310_7087_b200" not in text and "from paper_1310_7087_b200" not in text and "libqcd_b200" not in text, f
