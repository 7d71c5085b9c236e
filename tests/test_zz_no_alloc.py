"""qcd_measure_plaquette_noalloc against qcd_measure (include/qcd.h).

The entry point exists for programs that cannot let this library allocate device memory: a process whose own allocator
(PyTorch's caching allocator, say) already owns the GPU's memory, so a cudaMalloc made behind its back may fail, or a
measurement loop that shares the GPU with other streams and cannot take the device-wide stall cudaMalloc / cudaFree may
cause.  It keeps its partial sums in one array built into the library (QCD_NOALLOC_MAX_PARTIALS doubles per GPU, shared by
every call), so what is worth testing is: the numbers equal the allocating path's, a call is not disturbed by what the
previous call left in the shared array, an oversized lattice is refused before anything is launched, and the free device
memory does not move.

This file is named so that pytest collects it LAST: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes on its own in a fresh process and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

from tests.tolerances import MEAS_TOL

VARIANTS = [(3, 0, 1), (3, 1, 0), (2, 0, 0)]          # (Nc, precision, flags): SU(3) fp32 x12, SU(3) fp64 x18, SU(2) fp32
VARIANT_IDS = ["su3-f32-x12", "su3-f64-x18", "su2-f32"]


def test_null_arguments_are_refused_without_a_device():
    import paper_1310_7087_b200 as q
    from paper_1310_7087_b200.build import build_cuda
    build_cuda()
    lib = q.lib()
    assert lib.qcd_measure_plaquette_noalloc(None, None, None) == q.QCD_ERR_INVALID_ARG
    assert lib.qcd_measure_plaquette_noalloc(None, None, C.c_void_p(256)) == q.QCD_ERR_INVALID_ARG
    assert len(lib.qcd_last_error()) > 0


@pytest.mark.gpu
@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_two_calls_in_a_row_match_qcd_measure(qcd, variant):
    """Call 1 on a large lattice fills many entries of the shared array; call 2, straight behind it on the same stream, is a
    small ragged lattice with a background field that uses only the first few entries; call 3 is the large lattice again after
    a sweep.  Each must equal what qcd_measure returns for the same links, to the bar the measurement tests use."""
    import torch
    Nc, prec, flags = variant
    big, small = (16, 16, 16, 8), (6, 4, 10, 2)         # boxed thread mapping / plain mapping with a ragged last CTA
    fld = qcd.make_field(1, 3, [0.4, -0.4] if Nc == 2 else [0.4, 0.3, -0.7])
    npl = 6
    with qcd.Lattice(big, Nc, prec, flags) as A, qcd.Lattice(small, Nc, prec, flags) as B, qcd.Lattice((4, 4, 4, 4), Nc, prec, flags) as W:
        A.qcd_init(qcd.QCD_HOT, 11)
        B.qcd_init(qcd.QCD_HOT, 12)
        W.qcd_init(qcd.QCD_HOT, 13)
        out = torch.full((3, npl), float("nan"), dtype=torch.float64, device="cuda")
        # set-up call (the first call on a device looks up the array's address; the first launch of a kernel loads its code)
        W.qcd_measure_plaquette_noalloc(torch.empty(npl, dtype=torch.float64, device="cuda"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        A.qcd_measure_plaquette_noalloc(out[0])
        B.qcd_measure_plaquette_noalloc(out[1], fld)
        torch.cuda.synchronize()
        # neither A nor B has been through qcd_measure yet, so no buffer of theirs existed before these two calls either:
        # the device's free memory must not have moved
        assert torch.cuda.mem_get_info()[0] == free_before
        A.qcd_sweep(5.7 if Nc == 3 else 2.3, 1, 1)
        A.qcd_measure_plaquette_noalloc(out[2])
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        ref_a2 = A.qcd_measure(polyakov=False)[1]
        ref_b = B.qcd_measure(fld, polyakov=False)[1]
        A.qcd_init(qcd.QCD_HOT, 11)
        ref_a1 = A.qcd_measure(polyakov=False)[1]
    assert np.all(np.isfinite(got))
    for k, ref in enumerate((ref_a1, ref_b, ref_a2)):
        assert np.max(np.abs(got[k] - ref)) < MEAS_TOL[prec], (k, got[k], ref)
    assert abs(ref_a1.mean() - ref_a2.mean()) > 1e-3      # the sweep did change what call 3 had to measure


@pytest.mark.gpu
def test_lattice_beyond_the_built_in_array_is_refused(qcd):
    import torch
    dims = (96, 64, 64, 64)                              # 6 planes x V / 128 = 1 179 648 partial sums > 2^20
    assert 6 * int(np.prod(dims)) // 128 > qcd.QCD_NOALLOC_MAX_PARTIALS
    out = torch.full((6,), -7.0, dtype=torch.float64, device="cuda")
    with qcd.Lattice(dims, 2, qcd.QCD_FP32, 0) as G:
        G.qcd_init(qcd.QCD_COLD, 1)
        with pytest.raises(qcd.QcdError) as err:
            G.qcd_measure_plaquette_noalloc(out)
        assert err.value.code == qcd.QCD_ERR_UNSUPPORTED and "QCD_NOALLOC_MAX_PARTIALS" in str(err.value)
        torch.cuda.synchronize()
        assert torch.all(out == -7.0)                    # nothing was launched
        assert np.all(G.qcd_measure(polyakov=False)[1] == 1.0)
    # the largest D = 4 lattice of the benchmark configurations that fits: 64^3 x 16 (config 5, fp32 x12) on a cold start
    with qcd.Lattice((64, 64, 64, 16), 3, qcd.QCD_FP32, qcd.QCD_FLAG_COMPRESS12) as G:
        G.qcd_init(qcd.QCD_COLD, 1)
        G.qcd_measure_plaquette_noalloc(out)
        torch.cuda.synchronize()
        assert torch.all(out == 1.0)
