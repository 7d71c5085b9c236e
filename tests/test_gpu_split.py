"""GPU tests of the divided lattice: qcd_split_* (all parts in one process, halo
layers written into the neighbour's memory by a kernel) and the qcd_slab_* primitives driven by the per-process bookkeeping
of paper_1310_7087_b200/split.py.  The Philox counters use the global site index, so a divided lattice must reproduce the
undivided one bit for bit wherever both run the same kernel instantiation, and the oracle per sub-step within the bars."""
import numpy as np
import pytest

import oracle
from tests.inputs import random_links, round_to_fp32
from tests.tolerances import MEAS_TOL, TOL

pytestmark = pytest.mark.gpu

# (Nc, precision, flags)
VARIANTS = [(3, 1, 0), (3, 0, 1), (3, 0, 0), (2, 1, 0), (2, 0, 0)]
VARIANT_IDS = ["su3-f64x18", "su3-f32x12", "su3-f32x18", "su2-f64", "su2-f32"]
# dims, part extents (None: equal parts), n_parts, field
SPLIT_CASES = [
    ((16, 8, 16, 4), None, 2, None),            # equal parts; the tiled fp32 OR kernel's boxes divide both the whole and the parts
    ((16, 8, 16, 4), [4, 12], 2, (0, 1)),       # unequal parts, field
    ((16, 8, 16, 4), None, 4, (2, 3)),          # four parts, field plane containing the split direction
    ((16, 8, 16, 4), None, 1, None),            # one part: the lattice is its own neighbour
    ((8, 12, 6), [4, 8], 2, (0, 2)),            # D = 3: split along direction 1
    ((6, 4, 8, 2), [2, 6], 2, None),            # thin part (2 layers), ragged CTAs
]


def _prep(dims, Nc, prec, seed=43):
    links = random_links(dims, Nc, seed, 0.35)
    return round_to_fp32(links) if prec == 0 else links


def _field(qcd, fld, Nc):
    if fld is None:
        return None, None
    th = [0.4, -0.4] if Nc == 2 else [0.4, 0.3, -0.7]
    return qcd.make_field(fld[0], fld[1], th), oracle.make_field(fld[0], fld[1], th)


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims,extents,n_parts,fld", SPLIT_CASES)
def test_split_sweep_is_bit_identical_to_the_undivided_sweep(qcd, variant, dims, extents, n_parts, fld):
    Nc, prec, flags = variant
    beta = 5.7 if Nc == 3 else 2.5
    fg, _ = _field(qcd, fld, Nc)
    links = _prep(dims, Nc, prec)
    with qcd.Lattice(dims, Nc, prec, flags) as G, qcd.SplitLattice(dims, Nc, prec, flags, n_parts=n_parts, extents=extents) as S:
        off, ext = S.qcd_split_parts()
        assert off[0] == 0 and sum(ext) == dims[len(dims) - 2] and all(e % 2 == 0 for e in ext)
        if extents is not None:
            assert ext == list(extents)
        # per (parity, mu) array two boundary layers per part, all planes
        layer_links = int(np.prod(dims)) // dims[len(dims) - 2] // 2
        link_bytes = {(3, 0, 1): 48, (3, 0, 0): 72, (3, 1, 0): 144, (2, 0, 0): 16, (2, 1, 0): 32}[variant]
        assert S.qcd_split_halo_bytes() == 2 * n_parts * layer_links * link_bytes
        for X in (G, S):
            (X.qcd_set_seed if X is G else X.qcd_split_set_seed)(2025)
        G.qcd_set_links(links)
        S.qcd_split_set_links(links)
        back = S.qcd_split_get_links().astype(np.complex128)
        cmp = slice(None) if flags == 0 else slice(0, 2)
        assert np.array_equal(back[..., cmp, :], links[..., cmp, :])
        for _ in range(2):
            G.qcd_sweep(beta, 1, 2, fg)
            S.qcd_split_sweep(beta, 1, 2, fg)
        assert S.qcd_split_get_sweep_counter() == G.qcd_get_sweep_counter() == 2
        a, b = G.qcd_get_links(), S.qcd_split_get_links()
        # the tiled fp32 x12 overrelaxation kernel runs where its boxes divide the visited extents: if whole and parts choose
        # differently (thin parts), the two kernels agree to rounding only
        same_kernel = not (variant == (3, 0, 1) and len(dims) == 4 and (dims[2] % 4 or any(e % 4 for e in ext) or dims[0] % 16))
        if same_kernel:
            assert np.array_equal(a, b)
        else:
            assert np.max(np.abs(a.astype(np.complex128) - b.astype(np.complex128))) < 1e-4
        ma, mb = G.qcd_measure(fg), S.qcd_split_measure(fg)
        tol = MEAS_TOL[prec] if same_kernel else 2e-5
        assert abs(ma[0] - mb[0]) < tol and np.max(np.abs(ma[1] - mb[1])) < tol and abs(ma[2] - mb[2]) < tol


@pytest.mark.parametrize("variant", [(3, 0, 1), (3, 1, 0)], ids=["su3-f32x12", "su3-f64x18"])
def test_split_measure_straight_behind_a_sweep(qcd, variant):
    """qcd_split_measure enqueued directly behind qcd_split_sweep, with no qcd_split_get_links / synchronise in between: the
    plaquette kernel of a part reads halo copies that the neighbours' last update kernels write from other streams, so the
    measurement has to wait for them itself.  Repeated, on four parts, against the undivided sweep + measure."""
    Nc, prec, flags = variant
    dims, beta = (16, 8, 16, 8), 5.7
    with qcd.Lattice(dims, Nc, prec, flags) as G, qcd.SplitLattice(dims, Nc, prec, flags, n_parts=4) as S:
        G.qcd_init(qcd.QCD_HOT, 77)
        S.qcd_split_init(qcd.QCD_HOT, 77)
        for it in range(25):
            G.qcd_sweep(beta, 1, 1)
            S.qcd_split_sweep(beta, 1, 1)
            ma, mb = G.qcd_measure(), S.qcd_split_measure()
            assert abs(ma[0] - mb[0]) < MEAS_TOL[prec] and np.max(np.abs(ma[1] - mb[1])) < MEAS_TOL[prec] and abs(ma[2] - mb[2]) < MEAS_TOL[prec], it
        assert np.array_equal(G.qcd_get_links(), S.qcd_split_get_links())


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_split_hot_start_and_substeps_match_the_oracle(qcd, variant):
    """hot start of the parts = the oracle's (global Philox counters); every (parity, mu) heatbath and overrelaxation sub-step
    of a three-part lattice from a common pre-state against the oracle's undivided sub-step"""
    Nc, prec, flags = variant
    dims, beta = (8, 4, 12, 4), (5.7 if Nc == 3 else 2.5)
    D = len(dims)
    O = oracle.OracleLattice(dims, Nc)
    O.init(oracle.HOT, 11)
    with qcd.SplitLattice(dims, Nc, prec, flags, n_parts=3, extents=[4, 2, 6]) as S:
        S.qcd_split_init(qcd.QCD_HOT, 11)
        hot = S.qcd_split_get_links().astype(np.complex128)
        assert np.max(np.abs(hot - O.get_links())) < (1e-13 if prec == 1 else 5e-7)
        m = S.qcd_split_measure()
        mo = O.measure()
        assert abs(m[0] - mo[0]) < MEAS_TOL[prec] * 5 and abs(m[2] - mo[2]) < MEAS_TOL[prec] * 5
        links = _prep(dims, Nc, prec, seed=47)
        worst = 0.0
        for kind in (oracle.KIND_HB, oracle.KIND_OR):
            for parity in (0, 1):
                for mu in range(D):
                    Oc = oracle.OracleLattice(dims, Nc)
                    if prec == 0:
                        Oc.set_fp32_shadow(True)
                    Oc.set_links(links)
                    Oc.set_seed(5)
                    Oc.sweep_counter = 3
                    Oc.substep(beta, kind, 1, parity, mu)
                    S.qcd_split_set_links(links)
                    S.qcd_split_set_seed(5)
                    S.qcd_split_set_sweep_counter(3)
                    S.qcd_split_substep(beta, kind, 1, parity, mu)
                    got = S.qcd_split_get_links().astype(np.complex128)
                    worst = max(worst, float(np.max(np.abs(got - Oc.get_links()))))
        # thermal-like links: well conditioned, no accept/reject disagreement expected at this size (it would show as O(1))
        assert worst < TOL[prec], worst                                      # the bar of the undivided sub-step tests, all storage forms


@pytest.mark.parametrize("variant", [(3, 1, 0), (3, 0, 1), (2, 0, 0)], ids=["su3-f64x18", "su3-f32x12", "su2-f32"])
def test_slab_primitives_with_the_per_process_bookkeeping(qcd, variant):
    """the path of one part per process (paper_1310_7087_b200/split.py: qcd_slab_create, qcd_debug_substep on the part,
    qcd_slab_halo_pack / unpack, qcd_slab_measure_sums) with the transport replaced by handing the packed device buffers over
    inside one process: three parts on one GPU must reproduce the undivided lattice bit for bit"""
    import torch
    from paper_1310_7087_b200 import split as sp
    Nc, prec, flags = variant
    dims, beta = (16, 8, 16, 4), (5.7 if Nc == 3 else 2.5)
    D = len(dims)
    parts = sp.partition(dims[D - 2], 3, [1, 2, 1])
    assert [e for _, e in parts] == [4, 8, 4]
    links = _prep(dims, Nc, prec, seed=53)
    grid = links.reshape(tuple(reversed(dims)) + links.shape[1:])
    P = [sp.GpuPart(qcd, dims, Nc, prec, flags, off, ext, "cuda:0") for off, ext in parts]
    try:
        for (off, ext), part in zip(parts, P):
            block = np.ascontiguousarray(grid[:, off:off + ext]).reshape(-1, D, Nc, Nc)      # axis 1 <-> direction D-2 (D = 4)
            part.lat.qcd_set_seed(9)
            part.lat.qcd_set_links(block)

        def refresh(parity, mu):
            packed = [{side: p.pack(parity, mu, side) for side in (0, 1)} for p in P]
            for r, p in enumerate(P):
                for side, dst, unpack_side in sp.halo_messages(r, len(P)):
                    P[dst].unpack(parity, mu, unpack_side, packed[r][side])

        for parity in (0, 1):
            for mu in range(D):
                refresh(parity, mu)
        for kind, hit, parity, mu in sp.sweep_schedule(D, 1, 2):
            for p in P:
                p.substep(beta, kind, hit, parity, mu)
            refresh(parity, mu)
        with qcd.Lattice(dims, Nc, prec, flags) as G:
            G.qcd_set_seed(9)
            G.qcd_set_links(links)
            G.qcd_sweep(beta, 1, 2)
            ref = G.qcd_get_links()
            m_ref = G.qcd_measure()
        got = np.zeros_like(ref).reshape(tuple(reversed(dims)) + ref.shape[1:])
        for (off, ext), part in zip(parts, P):
            got[:, off:off + ext] = part.lat.qcd_get_links().reshape((dims[3], ext, dims[1], dims[0]) + ref.shape[1:])
        assert np.array_equal(got.reshape(ref.shape), ref)
        sums = [p.measure_sums() for p in P]
        V = int(np.prod(dims))
        planes = sum(s[0] for s in sums) / V
        poly = sum(s[1] for s in sums) / (V // dims[-1])
        assert np.max(np.abs(planes - m_ref[1])) < MEAS_TOL[prec] and abs(poly - m_ref[2]) < MEAS_TOL[prec]
        # whole-lattice calls are refused on a part
        for call in (lambda: P[0].lat.qcd_sweep(beta, 1, 1), lambda: P[0].lat.qcd_measure()):
            with pytest.raises(qcd.QcdError) as e:
                call()
            assert e.value.code == qcd.QCD_ERR_UNSUPPORTED
    finally:
        for p in P:
            p.lat.close()


def test_split_error_paths(qcd):
    with pytest.raises(qcd.QcdError) as e:
        qcd.SplitLattice((8, 8), 2, 1, 0, n_parts=2)
    assert e.value.code == qcd.QCD_ERR_UNSUPPORTED                      # D = 2 has no direction D-2 >= 1 to split
    with pytest.raises(qcd.QcdError) as e:
        qcd.SplitLattice((8, 8, 8, 4), 3, 1, 0, n_parts=2, extents=[3, 5])
    assert e.value.code == qcd.QCD_ERR_INVALID_ARG
    with pytest.raises(qcd.QcdError) as e:
        qcd.SplitLattice((8, 8, 8, 4), 3, 1, 0, n_parts=5)
    assert e.value.code == qcd.QCD_ERR_INVALID_ARG
    with pytest.raises(qcd.QcdError) as e:
        qcd.Lattice((8, 8, 8, 4), 3, 1, 0, slab=(1, 4))
    assert e.value.code == qcd.QCD_ERR_INVALID_ARG
    with qcd.SplitLattice((8, 8, 8, 4), 3, 1, 0, n_parts=2) as S:
        with pytest.raises(qcd.QcdError) as e:
            S.qcd_split_sweep(5.7, 1, 1)
        assert e.value.code == qcd.QCD_ERR_STATE
        S.qcd_split_init(qcd.QCD_COLD, 1)
        tot, planes, poly = S.qcd_split_measure()
        assert tot == 1.0 and np.all(planes == 1.0) and poly == 1.0


@pytest.mark.parametrize("variant", [(3, 1, 0), (3, 0, 1), (2, 0, 0)], ids=["su3-f64x18", "su3-f32x12", "su2-f32"])
@pytest.mark.parametrize("dims,extents,fld", [((8, 6, 8, 4), [2, 4, 2], (1, 2)), ((8, 6, 8, 4), [8], None), ((6, 8, 4), [4, 4], None)])
def test_streamed_lattice_reproduces_the_undivided_sweep(qcd, variant, dims, extents, fld):
    """split.StreamedLattice: the parts live in pinned host memory and pass through one device buffer in every sub-step
    (the paper's use of the division when one device's memory is not enough).  From the same links and the
    same hot start it must reproduce qcd_sweep bit for bit (dims[0] = 8 or 6: every kernel is the ring kernel on both sides)
    and the observables within the measurement bars."""
    from paper_1310_7087_b200 import split
    Nc, prec, flags = variant
    beta = 5.7 if Nc == 3 else 2.5
    fg, _ = _field(qcd, fld, Nc)
    links = _prep(dims, Nc, prec)
    with qcd.Lattice(dims, Nc, prec, flags) as G, split.StreamedLattice(qcd, dims, Nc, prec, flags, extents=extents) as S:
        G.qcd_set_seed(77)
        S.set_seed(77)
        G.qcd_set_links(links)
        S.set_links(links)
        cmp = slice(None) if flags == 0 else slice(0, 2)
        assert np.array_equal(S.get_links().astype(np.complex128)[..., cmp, :], links[..., cmp, :])
        for _ in range(2):
            G.qcd_sweep(beta, 1, 1, fg)
            S.sweep(beta, 1, 1, fg)
        assert np.array_equal(G.qcd_get_links(), S.get_links())
        ma, mb = G.qcd_measure(fg), S.measure(fg)
        tol = MEAS_TOL[prec]
        assert abs(ma[0] - mb[0]) < tol and np.max(np.abs(ma[1] - mb[1])) < tol and abs(ma[2] - mb[2]) < tol
        # every sub-step moved every part to the device and the one array it wrote back: (1 + 1 / (2 D)) x the parts' bytes
        # <= 1.125 x (D = 4); set_links adds one full download
        parts_bytes = sum(L.nbytes for L in S.lat)
        D = len(dims)
        n_substeps = 2 * 2 * 2 * D
        assert S.bytes_moved == parts_bytes + n_substeps * (parts_bytes + parts_bytes // (2 * D))
        assert (S.bytes_moved - parts_bytes) / n_substeps <= (1.0 + 1.0 / 6.0) * parts_bytes
    # hot start through the parts = hot start of the whole lattice (Philox counters use the global site index)
    with qcd.Lattice(dims, Nc, prec, flags) as G, split.StreamedLattice(qcd, dims, Nc, prec, flags, extents=extents) as S:
        G.qcd_init(qcd.QCD_HOT, 5)
        S.init(qcd.QCD_HOT, 5)
        assert np.array_equal(G.qcd_get_links(), S.get_links())
        G.qcd_sweep(beta, 1, 0, fg)
        S.sweep(beta, 1, 0, fg)
        assert np.array_equal(G.qcd_get_links(), S.get_links())
