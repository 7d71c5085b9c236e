"""GPU-vs-oracle parity through the C ABI (SURVEY.md sec 8(c)-6 protocol T1..T5).  Run on the B200 box: -m gpu.

Tolerances (BASELINE.json north_star): Philox words bit-exact; links per element max abs 1e-12 (fp64) / 2e-5 (fp32);
heatbath accept/reject disagreements reported and <= 1e-6 of links; long-run <P> within 3 sigma.
Every oracle input is produced by oracle/ or tests/inputs.py, never by the CUDA path.
"""
import numpy as np
import pytest

import oracle
from tests import np_lattice as npl
from tests.inputs import random_links, round_to_fp32
# the bars and the arithmetic they come from (conditioning rule with its ceiling, Haar expectation, un-resynced bar)
from tests.tolerances import K_COND, MEAS_TOL, TOL, carry_bound, illcond_bound, link_tol, unresynced_bar

pytestmark = pytest.mark.gpu

# (Nc, precision, flags)
VARIANTS = [(3, 1, 0), (3, 0, 1), (3, 0, 0), (3, 1, 1), (2, 1, 0), (2, 0, 0)]
VARIANT_IDS = ["su3-f64x18", "su3-f32x12", "su3-f32x18", "su3-f64x12", "su2-f64", "su2-f32"]


def gpu_lattice(q, dims, Nc, precision, flags):
    return q.Lattice(dims, Nc, precision, flags)


def oracle_lattice(dims, Nc, precision, links=None):
    L = oracle.OracleLattice(dims, Nc)
    if precision == 0:
        L.set_fp32_shadow(True)
    if links is not None:
        L.set_links(links)
    return L


def prep_links(dims, Nc, precision, seed, spread=None):
    links = random_links(dims, Nc, seed, spread)
    return round_to_fp32(links) if precision == 0 else links


def field_pair(q, fld):
    if fld is None:
        return None, None
    return q.make_field(*fld), oracle.make_field(*fld)


# ----------------------------------------------------------------------------- T1: Philox
def test_philox_bit_exact_vs_oracle_and_curand(qcd):
    rng = np.random.Generator(np.random.PCG64(1))
    n = 1_000_000
    ctr = rng.integers(0, 2 ** 32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0], key[0] = 0, 0
    ctr[1], key[1] = 0xFFFFFFFF, 0xFFFFFFFF
    mine = qcd.qcd_debug_philox(ctr, key, impl=0)
    cur = qcd.qcd_debug_philox(ctr, key, impl=1)
    ref = oracle.philox4x32_10_batch(ctr, key)
    assert np.array_equal(mine, ref)
    assert np.array_equal(cur, ref)
    assert list(mine[0]) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]


# ----------------------------------------------------------------------------- layout / init / measure
@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims", [(4, 6), (6, 4, 2), (6, 4, 10, 2), (16, 16, 16, 4)])
def test_set_get_links_roundtrip(qcd, variant, dims):
    Nc, prec, flags = variant
    links = prep_links(dims, Nc, prec, seed=3)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_set_links(links)
        back = G.qcd_get_links().astype(np.complex128)
    if flags == 0:
        assert np.array_equal(back, links)
    else:
        assert np.array_equal(back[..., :2, :], links[..., :2, :])
        assert np.max(np.abs(back[..., 2, :] - links[..., 2, :])) < (5e-7 if prec == 0 else 4e-15)


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims", [(16, 16), (6, 4, 10), (6, 4, 10, 2), (16, 16, 16, 4)])
def test_hot_and_cold_start_match_oracle(qcd, variant, dims):
    Nc, prec, flags = variant
    O = oracle.OracleLattice(dims, Nc)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_init(qcd.QCD_COLD, 5)
        cold = G.qcd_get_links()
        assert np.array_equal(cold, np.broadcast_to(np.eye(Nc), cold.shape))
        tot, planes, poly = G.qcd_measure()
        assert tot == 1.0 and np.all(planes == 1.0) and poly == 1.0 + 0j
        G.qcd_init(qcd.QCD_HOT, 42)
        hot = G.qcd_get_links().astype(np.complex128)
        assert G.qcd_get_sweep_counter() == 0 and G.qcd_get_seed() == 42
    O.init(oracle.HOT, 42)
    ref = O.get_links()
    # fp32: rounding of the double result; compressed storage rebuilds row 2 in fp32 from the rounded rows 0,1
    tol = 1e-13 if prec == 1 else (6e-8 if flags == 0 else 5e-7)
    assert np.max(np.abs(hot - ref)) < tol


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims,fld", [((4, 6), None), ((6, 4, 10), None), ((6, 4, 10, 2), None), ((16, 16, 16, 4), None),
                                      ((6, 4, 10, 2), (0, 1, "std")), ((6, 4, 10, 2), (1, 3, "std")), ((6, 4, 10), (0, 2, "std"))])
def test_measure_matches_oracle(qcd, variant, dims, fld):
    Nc, prec, flags = variant
    if fld is not None:
        fld = (fld[0], fld[1], [0.4, -0.4] if Nc == 2 else [0.4, 0.3, -0.7])
    fg, fo = field_pair(qcd, fld)
    links = prep_links(dims, Nc, prec, seed=9)
    O = oracle_lattice(dims, Nc, prec, links)
    tot_o, planes_o, poly_o = O.measure(fo)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_set_links(links)
        tot, planes, poly = G.qcd_measure(fg)
        again = G.qcd_measure(fg)
    assert np.max(np.abs(planes - planes_o)) < MEAS_TOL[prec]
    assert abs(tot - tot_o) < MEAS_TOL[prec] and abs(poly - poly_o) < MEAS_TOL[prec]
    assert again[0] == tot and np.array_equal(again[1], planes) and again[2] == poly     # deterministic reduction


# ----------------------------------------------------------------------------- T2 / T3: per sub-step parity with resync
SUBSTEP_CASES = [
    # dims, field
    ((4, 6), None), ((6, 4, 10), None), ((6, 4, 10, 2), None), ((2, 2, 2, 2), None), ((16, 16, 16, 4), None), ((12, 6, 4, 8), None),
    ((6, 4, 10, 2), (0, 1)), ((6, 4, 10, 2), (1, 3)), ((6, 4, 10), (0, 2)), ((4, 6), (0, 1)),
    # lattices the CTA boxes of the tiled kernel (update_tiled.cuh: 8 half-indices x 4 x 4 x 1 and permutations) divide:
    # one box spans a whole direction (every face wraps onto the box itself) / several boxes per direction, with field
    ((16, 4, 4, 4), (0, 1)), ((16, 4, 8, 4), (1, 3)), ((32, 8, 4, 4), (0, 3)),
]


def _run_substeps(qcd, variant, dims, fld, kind, beta, spread, seed):
    """every (parity, mu) sub-step from a common pre-state; returns worst (link diff / link tolerance), disagreements,
    links compared, and how many links fell under the conditioning rule"""
    Nc, prec, flags = variant
    D = len(dims)
    if fld is not None:
        fld = (fld[0], fld[1], [0.4, -0.4] if Nc == 2 else [0.4, 0.3, -0.7])
    fg, fo = field_pair(qcd, fld)
    links = prep_links(dims, Nc, prec, seed=seed, spread=spread)
    worst, disagreements, compared, illcond = 0.0, 0, 0, 0
    site_par = np.stack(np.unravel_index(np.arange(int(np.prod(dims))), dims[::-1]), axis=-1).sum(axis=1) & 1   # lex -> parity
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
        G.qcd_set_seed(2024)
        for sweep_ctr, hit in [(0, 0), (7, 3)] if kind == 0 else [(0, 0)]:
            for parity in (0, 1):
                for mu in range(D):
                    O = oracle_lattice(dims, Nc, prec, links)
                    O.set_seed(2024)
                    O.sweep_counter = sweep_ctr
                    tr_o, kmin = O.substep_diag(beta, kind, hit, parity, mu, fo)
                    ref = O.get_links()
                    G.qcd_set_links(links)                      # resync to the common pre-state
                    G.qcd_set_sweep_counter(sweep_ctr)
                    G.qcd_debug_substep(beta, kind, hit, parity, mu, fg)
                    got = G.qcd_get_links().astype(np.complex128)
                    diff = np.max(np.abs(got - ref), axis=(-1, -2))            # (V, D)
                    # links of other (parity, mu) arrays must be bit-identical to the pre-state.  (Membership by index, not by
                    # "the oracle changed it": a link whose heatbath trials are all rejected keeps its value in the oracle
                    # but is re-normalised, i.e. may move by an ulp, on the GPU.)
                    untouched = np.ones_like(diff, dtype=bool)
                    untouched[site_par == parity, mu] = False
                    changed = ~untouched
                    cmp_links = got if flags == 0 else got[..., :2, :]
                    pre_links = links if flags == 0 else links[..., :2, :]
                    same = np.max(np.abs(cmp_links - pre_links), axis=(-1, -2)) == 0
                    assert np.all(same[untouched]), "a link outside the sub-step changed"
                    if kind == 0:
                        tr_g = G.qcd_debug_get_trials()
                        bad = np.any(tr_g != tr_o, axis=1)                       # (V,) accept/reject disagreements
                        disagreements += int(bad.sum())
                        diff[bad, :] = 0.0
                    tol = link_tol(prec, kmin)                                  # (V,)
                    illcond += int(np.sum(np.isfinite(kmin) & (kmin < K_COND))) if prec == 0 else 0
                    worst = max(worst, float((diff[:, mu] / tol).max()))
                    diff[:, mu] = 0.0
                    compared += int(changed.sum())
    return worst, disagreements, compared, illcond


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims,fld", SUBSTEP_CASES)
def test_overrelaxation_substeps(qcd, variant, dims, fld):
    worst, _, compared, illcond = _run_substeps(qcd, variant, dims, fld, kind=1, beta=5.7, spread=None, seed=13)
    assert compared > 0
    print("OR worst diff/tol %.3f; links under the conditioning rule: %d of %d" % (worst, illcond, compared))
    assert worst < 1.0, worst
    # Haar inputs: how many links may fall under the conditioning rule is bounded by the derived expectation
    assert illcond <= illcond_bound(variant[0], len(dims), compared), (illcond, compared)


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims,fld", SUBSTEP_CASES)
@pytest.mark.parametrize("spread", [None, 0.35], ids=["haar", "thermal"])
def test_heatbath_substeps(qcd, variant, dims, fld, spread):
    beta = 5.7 if variant[0] == 3 else 2.5
    worst, disagreements, compared, illcond = _run_substeps(qcd, variant, dims, fld, kind=0, beta=beta, spread=spread, seed=17)
    assert compared > 0
    print("HB worst diff/tol %.3f; links under the conditioning rule: %d of %d" % (worst, illcond, compared))
    assert worst < 1.0, worst
    if spread is not None:
        assert illcond == 0          # thermalised links are well conditioned: the plain north_star bar applied
    else:
        assert illcond <= illcond_bound(variant[0], len(dims), compared), (illcond, compared)
    # north_star: accept/reject disagreements at most 1e-6 of links (reported); on these small lattices that is zero
    print("heatbath disagreements: %d of %d links" % (disagreements, compared))
    assert disagreements <= max(0, int(1e-6 * compared)), (disagreements, compared)


def test_heatbath_trial_cap_and_exhaustion(qcd):
    # hot 2-D SU(2) at small beta: alpha is small, trials often fail; with T_max = 1 many links keep their value (R5)
    dims, Nc = (16, 16), 2
    links = prep_links(dims, Nc, 1, seed=23)
    O = oracle_lattice(dims, Nc, 1, links)
    O.set_seed(5)
    O.set_max_trials(1)
    tr_o = O.substep(0.8, oracle.KIND_HB, 0, 0, 1, want_trials=True)
    with gpu_lattice(qcd, dims, Nc, 1, 0) as G:
        G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
        G.qcd_set_option(qcd.QCD_OPT_KP_MAX_TRIALS, 1)
        G.qcd_set_seed(5)
        G.qcd_set_links(links)
        G.qcd_debug_substep(0.8, qcd.QCD_KIND_HB, 0, 0, 1)
        tr_g = G.qcd_debug_get_trials()
        got = G.qcd_get_links()
    assert np.array_equal(tr_g, tr_o)
    assert np.sum(tr_o[:, 0] == 0x81) > 10 and np.sum(tr_o[:, 0] == 1) > 10
    assert np.max(np.abs(got - O.get_links())) < 1e-12


# ----------------------------------------------------------------------------- whole sweeps without resync
def _unresynced_sequence(qcd, G, O, dims, Nc, prec, flags, beta, sequence, fg=None, fo=None):
    """Run `sequence` = [(kind, hit, parity, mu), ...] on both sides WITHOUT resync from the state both already hold.
    Heatbath accept/reject codes are compared per sub-step; a disagreement changes that link by O(1) and reaches, in later
    sub-steps, the links whose staples contain it: those links (the dependency cone, tests/np_lattice.staple_dependents) are
    fenced off.  Every other link must stay within ITS OWN bound, carried through the sequence from the oracle's conditioning
    number of every hit (tests/tolerances.carry_bound), and the median link within the typical bar (unresynced_bar).
    Returns (flips, fenced links, worst diff / bound outside the fence, median diff, median k, min k, GPU links)."""
    V, D = int(np.prod(dims)), len(dims)
    par = npl.site_parity(dims)
    fence = np.zeros((V, D), dtype=bool)
    bound = np.zeros((V, D))
    flips, kmed, kmin_all = 0, [], np.inf
    G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
    for kind, hit, parity, mu in sequence:
        tr_o, kmin = O.substep_diag(beta, kind, hit, parity, mu, fo)
        upd = par == parity
        kmed.append(float(np.median(kmin[upd])))
        kmin_all = min(kmin_all, float(kmin[upd].min()))
        G.qcd_debug_substep(beta, kind, hit, parity, mu, fg)
        bound = carry_bound(bound, npl.staple_rms(bound, dims, mu), kmin, TOL[prec], upd, mu)
        # links of this sub-step that read a fenced link join the fence
        dep = npl.staple_dependents(fence, dims, mu) & upd
        fence[dep, mu] = True
        if kind == 0:
            tr_g = G.qcd_debug_get_trials()
            bad = np.any(tr_g != tr_o, axis=1) & upd
            flips += int(bad.sum())
            fence[bad, mu] = True
    got = G.qcd_get_links().astype(np.complex128)
    diff = np.max(np.abs(got - O.get_links()), axis=(-1, -2))
    ok = ~fence & (bound > 0)
    worst = float((diff[ok] / bound[ok]).max()) if ok.any() else 0.0
    assert np.all(diff[~fence & (bound == 0)] == 0) or flags != 0     # links never updated did not move (x12: row 2 is rebuilt)
    return flips, int(fence.sum()), worst, float(np.median(diff[ok])), float(np.median(kmed)), kmin_all, got


def _sweep_sequence(D, n_hb, n_or):
    return [(0 if s < n_hb else 1, s if s < n_hb else 0, p, mu) for s in range(n_hb + n_or) for p in (0, 1) for mu in range(D)]


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_full_sweep_unresynced_from_thermal_state(qcd, variant):
    """One whole sweep (1 HB + 2 OR, 24 sub-steps) without resync, config-2 shape for SU(3) and a config-4-like shape for
    SU(2), from a thermal-like configuration (well conditioned: the plain bars apply).  Bar: every link-hit adds at most the
    single-sub-step bar and passes on what its 18 staple links carry with the RMS gain sqrt(18)/k (tests/tolerances.py).
    qcd_sweep itself must then reproduce, bit for bit, the sequence of debug sub-steps that was compared with the oracle."""
    Nc, prec, flags = variant
    dims = (16, 16, 16, 4) if Nc == 3 else (12, 12, 12, 8)
    beta = 5.7 if Nc == 3 else 2.5
    D = len(dims)
    links = prep_links(dims, Nc, prec, seed=29, spread=0.35)
    O = oracle_lattice(dims, Nc, prec, links)
    O.set_seed(7)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_set_seed(7)
        G.qcd_set_links(links)
        flips, fenced, worst, med, kmed, kmin, got = _unresynced_sequence(qcd, G, O, dims, Nc, prec, flags, beta, _sweep_sequence(D, 1, 2))
        bar = unresynced_bar(prec, 3, kmed)
        print("un-resynced sweep: flips %d, fenced links %d of %d, worst diff/bound %.3f, median diff %.3e (typical bar %.3e), k median %.2f min %.2f"
              % (flips, fenced, got.shape[0] * D, worst, med, bar, kmed, kmin))
        assert kmin > K_COND                       # no link under the conditioning rule on this state
        assert flips <= 1 and fenced <= 20000 * flips      # north_star: <= 1e-6 of links; one flip reaches < 20000 links in 2 passes
        assert worst < 1.0 and med < bar, (worst, med, bar)
        uni, det = npl.unitarity_defect(got)
        assert uni < (1e-12 if prec == 1 else 5e-6) and det < (1e-12 if prec == 1 else 5e-6)
        # qcd_sweep = the same 24 launches
        G.qcd_set_links(links)
        G.qcd_set_sweep_counter(0)
        G.qcd_sweep(beta, 1, 2)
        assert G.qcd_get_sweep_counter() == 1
        again = G.qcd_get_links().astype(np.complex128)
        assert np.array_equal(again, got)
        m_g, m_o = G.qcd_measure(), O.measure()
        if flips == 0:
            assert abs(m_g[0] - m_o[0]) < 10 * MEAS_TOL[prec]


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
def test_full_sweep_unresynced_from_hot_start(qcd, variant):
    """The same from the HOT start of config 2 (seed 7).  fp64: links agree to the un-resynced bar scaled by the worst
    conditioning met (k ~ 0.01 occurs among 65536 Haar links: 1e-12 * K_COND / k per hit).  fp32: links under the
    conditioning rule (tests/tolerances.expected_illcond_fraction: ~0.6 % per sub-step) lose digits at each of the 24
    sub-steps and pass that on, so link-by-link agreement of an un-resynced sweep is not defined from this state -- per
    sub-step parity from Haar inputs and un-resynced parity from a thermal state are the tests above; here the observables
    and the group property must agree."""
    Nc, prec, flags = variant
    dims = (16, 16, 16, 4) if Nc == 3 else (12, 12, 12, 8)
    beta = 5.7 if Nc == 3 else 2.5
    O = oracle.OracleLattice(dims, Nc)
    O.init(oracle.HOT, 7)
    start = O.get_links()
    if prec == 0:
        start = round_to_fp32(start)
        O.set_fp32_shadow(True)
        O.set_links(start)
    O.sweep(beta, 1, 2)
    ref = O.get_links()
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_init(qcd.QCD_HOT, 7)
        G.qcd_sweep(beta, 1, 2)
        got = G.qcd_get_links().astype(np.complex128)
        assert G.qcd_get_sweep_counter() == 1
        m_g = G.qcd_measure()
    m_o = O.measure()
    if prec == 1:
        diff = np.max(np.abs(got - ref), axis=(-1, -2))
        print("fp64 hot un-resynced sweep: worst link diff %.3e" % float(diff.max()))
        # Haar links: k is typically |sum of 6 Haar staples| ~ 1.5 (gain sqrt(18)/1.5 per hit) and the worst of the 2.6e5
        # link-hits is amplified by up to K_COND / K_FLOOR = 100 (the ceiling of the conditioning rule): 1.2e-9
        assert float(diff.max()) < unresynced_bar(1, 3, 1.5) * 100.0
    assert abs(m_g[0] - m_o[0]) < (1e-11 if prec == 1 else 1e-4)
    assert abs(m_g[2] - m_o[2]) < (1e-10 if prec == 1 else 2e-3)
    uni, det = npl.unitarity_defect(got)
    assert uni < (1e-12 if prec == 1 else 5e-6) and det < (1e-12 if prec == 1 else 5e-6)


@pytest.mark.parametrize("variant", [(3, 0, 1), (3, 1, 0), (3, 0, 0), (2, 0, 0)], ids=["su3-f32x12", "su3-f64x18", "su3-f32x18", "su2-f32"])
def test_substeps_back_to_back_in_any_order(qcd, variant):
    """An update kernel fetches, before it waits for the kernel launched just before it, only arrays that kernel does not
    write (prev_parity / prev_mu in the launch arguments).  qcd_sweep always launches (p, mu-1) before (p, mu); here the
    sub-steps follow each other WITHOUT a resync in orders a sweep never uses -- in particular (1-p, mu) right before
    (p, mu), whose output is the resident U_mu box of the tiled kernel, and (p, nu0) / (1-p, nu0) right before (p, mu),
    whose outputs are the first ring links, and the first sub-step right after qcd_set_links (every array just written) --
    and the result must equal the oracle's run of the same sequence."""
    Nc, prec, flags = variant
    dims, beta = (16, 8, 8, 4), 5.7                       # the CTA boxes of the tiled kernel divide this lattice
    links = prep_links(dims, Nc, prec, seed=21, spread=0.35)
    order = [(1, 2), (0, 2), (0, 0), (1, 1), (0, 1), (1, 0), (0, 1), (0, 0), (1, 3), (0, 3), (1, 0), (0, 1), (0, 1), (1, 1)]
    O = oracle_lattice(dims, Nc, prec, links)
    kmed = []
    for parity, mu in order:
        _, kmin = O.substep_diag(beta, oracle.KIND_OR, 0, parity, mu)
        kmed.append(float(np.median(kmin[np.isfinite(kmin)])))
        assert kmin.min() > K_COND
    ref = O.get_links()
    bar = unresynced_bar(prec, len(order), float(np.median(kmed)))     # dependency chains are at most len(order) hits deep
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        for rep in range(3):                              # timing-dependent hazards would not show every time
            G.qcd_set_links(links)
            for parity, mu in order:
                G.qcd_debug_substep(beta, qcd.QCD_KIND_OR, 0, parity, mu)
            got = G.qcd_get_links().astype(np.complex128)
            diff = float(np.max(np.abs(got - ref)))
            assert diff < bar, (rep, diff, bar)


@pytest.mark.parametrize("dims,Nc,fld", [((8, 8, 8, 4), 3, None), ((8, 8, 8, 4), 3, (0, 1)), ((16, 16), 2, None), ((6, 4, 10), 3, (0, 2))])
def test_measure_accumulate_matches_measure_and_oracle(qcd, dims, Nc, fld):
    """qcd_measure_accumulate / qcd_accum_get (on-device sums and sums of squares over configurations, no host
    synchronisation per measurement) against (i) the values qcd_measure returns for the same configurations, summed on the
    host in the same order, and (ii) the oracle's sweeps and measurements."""
    beta, n_meas = 5.7 if Nc == 3 else 2.0, 6
    if fld is not None:
        fld = (fld[0], fld[1], [0.4, 0.3, -0.7])
    fg, fo = field_pair(qcd, fld)
    D = len(dims)
    npl = D * (D - 1) // 2
    O = oracle.OracleLattice(dims, Nc)
    O.init(oracle.HOT, 11)
    host = np.zeros((2, npl + 3))
    orac = np.zeros((2, npl + 3))
    with gpu_lattice(qcd, dims, Nc, 1, 0) as G:
        G.qcd_init(qcd.QCD_HOT, 11)
        n0, s0, q0 = G.qcd_accum_get()
        assert n0 == 0 and not s0.any() and not q0.any()
        for _ in range(n_meas):
            O.sweep(beta, 1, 2, fo)
            G.qcd_set_links(O.get_links())                         # the oracle's configurations (sweeps are tested elsewhere;
            G.qcd_measure_accumulate(fg)                           # un-resynced trajectories separate chaotically)
            _, planes, poly = G.qcd_measure(fg)                    # same configuration, deterministic reductions
            v = np.concatenate([planes, [poly.real, poly.imag, abs(poly)]])
            host[0] += v
            host[1] += v * v
            _, planes_o, poly_o = O.measure(fo)
            vo = np.concatenate([planes_o, [poly_o.real, poly_o.imag, abs(poly_o)]])
            orac[0] += vo
            orac[1] += vo * vo
        n, s1, s2 = G.qcd_accum_get()
        assert n == n_meas
        assert np.max(np.abs(s1 - host[0])) < 1e-14 * n_meas and np.max(np.abs(s2 - host[1])) < 1e-14 * n_meas
        assert np.max(np.abs(s1 - orac[0])) < 1e-11 and np.max(np.abs(s2 - orac[1])) < 1e-11
        G.qcd_accum_reset()
        n, s1, s2 = G.qcd_accum_get()
        assert n == 0 and not s1.any() and not s2.any()


FUSED_CASES = [((4, 6), None, 1, 1), ((6, 4, 10), None, 1, 2), ((6, 4, 10, 2), None, 1, 2), ((16, 16, 16, 4), None, 1, 4), ((16, 8, 8, 4), (0, 1), 1, 2),
               ((6, 4, 10, 2), (1, 3), 2, 0), ((6, 4, 10), (0, 2), 0, 1), ((8, 4, 4, 4), (2, 3), 1, 1)]


@pytest.mark.parametrize("variant", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dims,fld,n_hb,n_or", FUSED_CASES)
def test_sweep_measure_fused_matches_separate_calls_and_oracle(qcd, variant, dims, fld, n_hb, n_or):
    """qcd_sweep_measure (plaquette folded into the last pass of the sweep: the sub-steps (parity 1, mu >= 1) see every
    plaquette of the planes (nu, mu), nu < mu, in its final state) against (i) qcd_sweep + qcd_measure on a second lattice
    from the same state -- same links bit for bit, observables to the measurement tolerance -- and (ii) the oracle's sweep
    and measurement.  Covers D = 2, 3, 4, field planes in every role, a heatbath as the last pass, lattices with a ragged
    last CTA (surplus threads of the measuring kernels) and the tiled overrelaxation kernel."""
    Nc, prec, flags = variant
    beta = 5.7 if Nc == 3 else 2.5
    if fld is not None:
        fld = (fld[0], fld[1], [0.4, -0.4] if Nc == 2 else [0.4, 0.3, -0.7])
    fg, fo = field_pair(qcd, fld)
    links = prep_links(dims, Nc, prec, seed=31, spread=0.35)
    O = oracle_lattice(dims, Nc, prec, links)
    O.set_seed(99)
    O.sweep(beta, n_hb, n_or, fo)
    tot_o, planes_o, poly_o = O.measure(fo)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as A, gpu_lattice(qcd, dims, Nc, prec, flags) as B:
        for G in (A, B):
            G.qcd_set_seed(99)
            G.qcd_set_links(links)
        tot_f, planes_f, poly_f = A.qcd_sweep_measure(beta, n_hb, n_or, fg)
        B.qcd_sweep(beta, n_hb, n_or, fg)
        tot_s, planes_s, poly_s = B.qcd_measure(fg)
        la, lb = A.qcd_get_links(), B.qcd_get_links()
        assert A.qcd_get_sweep_counter() == B.qcd_get_sweep_counter() == 1
        # the measuring kernels do the same link arithmetic; they are separate instantiations, in which the compiler may
        # contract multiply-adds differently: equal to a few units in the last place, not necessarily bit for bit
        assert np.max(np.abs(la - lb)) < (4e-15 if prec == 1 else 1e-6) * (n_hb + n_or)
        tol = MEAS_TOL[prec]
        assert np.max(np.abs(planes_f - planes_s)) < tol and abs(tot_f - tot_s) < tol, (planes_f, planes_s)
        assert abs(poly_f - poly_s) < tol
        # against the oracle (un-resynced sweep: fp32 links differ by ~1e-5, means over the lattice by much less)
        otol = 1e-11 if prec == 1 else 2e-5
        assert np.max(np.abs(planes_f - planes_o)) < otol and abs(poly_f - poly_o) < otol, (planes_f, planes_o)
        # repeatable, and the accumulating form adds the same numbers
        A.qcd_set_links(links)
        A.qcd_set_sweep_counter(0)
        again = A.qcd_sweep_measure(beta, n_hb, n_or, fg)
        assert again[0] == tot_f and np.array_equal(again[1], planes_f) and again[2] == poly_f
        A.qcd_set_links(links)
        A.qcd_set_sweep_counter(0)
        A.qcd_accum_reset()
        A.qcd_sweep_measure_accumulate(beta, n_hb, n_or, fg)
        n, s1, s2 = A.qcd_accum_get()
        want = np.concatenate([planes_f, [poly_f.real, poly_f.imag, abs(poly_f)]])
        assert n == 1 and np.max(np.abs(s1 - want)) < 1e-15 and np.max(np.abs(s2 - want * want)) < 1e-15


def test_sweep_measure_with_no_pass_measures_the_unchanged_configuration(qcd):
    links = prep_links((6, 4, 10, 2), 3, 1, seed=5)
    with gpu_lattice(qcd, (6, 4, 10, 2), 3, 1, 0) as G:
        G.qcd_set_links(links)
        a = G.qcd_sweep_measure(5.7, 0, 0)
        b = G.qcd_measure()
        assert a[0] == b[0] and np.array_equal(a[1], b[1]) and a[2] == b[2]
        assert np.array_equal(G.qcd_get_links(), links)


def test_bulk_copy_overrelaxation_kernel_matches_the_oracle(qcd):
    """QCD_OPT_BULK_COPY: the kernel that stages every operand with cp.async.bulk + mbarriers (update_bulk.cuh; slower,
    kept for the measurement of DESIGN.md sec 6.10) on lattices with dims[0] = 32: every (parity, mu) overrelaxation
    sub-step against the oracle, boxes that wrap onto themselves and several boxes per direction, and after qcd_set_links
    (no early fetch) as well as back to back"""
    for dims in [(32, 4, 2, 2), (32, 8, 4, 4), (32, 4, 6, 2)]:
        links = prep_links(dims, 3, 0, seed=61, spread=0.35)
        with gpu_lattice(qcd, dims, 3, 0, 1) as G:
            G.qcd_set_option(qcd.QCD_OPT_BULK_COPY, 1)
            worst = 0.0
            for parity in (0, 1):
                for mu in range(4):
                    O = oracle_lattice(dims, 3, 0, links)
                    O.substep(5.7, oracle.KIND_OR, 0, parity, mu)
                    G.qcd_set_links(links)
                    G.qcd_debug_substep(5.7, qcd.QCD_KIND_OR, 0, parity, mu)
                    worst = max(worst, float(np.max(np.abs(G.qcd_get_links().astype(np.complex128) - O.get_links()))))
            assert worst < TOL[0], (dims, worst)
            O = oracle_lattice(dims, 3, 0, links)
            G.qcd_set_links(links)
            for parity, mu in [(0, 1), (1, 1), (1, 0), (0, 0), (0, 3), (1, 2), (0, 2), (1, 3)]:
                O.substep(5.7, oracle.KIND_OR, 0, parity, mu)
                G.qcd_debug_substep(5.7, qcd.QCD_KIND_OR, 0, parity, mu)
            assert float(np.max(np.abs(G.qcd_get_links().astype(np.complex128) - O.get_links()))) < unresynced_bar(0, 8, 3.5)


def test_launch_order_does_not_change_any_result(qcd):
    """QCD_OPT_ALTERNATE_ORDER (consecutive update launches visit the lattice in opposite directions, for L2 reuse): the
    order in which CTAs take their boxes must not show in the links, the trial codes or the fused observables -- bit for bit,
    every storage format, tiled / ring / SU(2) kernels, a ragged last CTA and a divisible lattice"""
    cases = [((16, 16, 16, 4), 3, 0, 1), ((16, 16, 16, 4), 3, 1, 0), ((6, 4, 10, 2), 3, 0, 0), ((6, 4, 10, 2), 3, 1, 1),
             ((12, 6, 4, 8), 2, 0, 0), ((6, 4, 10), 3, 1, 0), ((4, 6), 2, 1, 0)]
    for dims, Nc, prec, flags in cases:
        out = []
        for alt in (1, 0):
            with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
                G.qcd_set_option(qcd.QCD_OPT_ALTERNATE_ORDER, alt)
                G.qcd_init(qcd.QCD_HOT, 11)
                G.qcd_sweep(5.7, 1, 2)
                obs = G.qcd_sweep_measure(5.7, 1, 1)
                out.append((G.qcd_get_links(), obs))
        (la, oa), (lb, ob) = out
        assert np.array_equal(la, lb), (dims, Nc, prec, flags)
        assert oa[0] == ob[0] and np.array_equal(oa[1], ob[1]) and oa[2] == ob[2], (dims, Nc, prec, flags)


def test_heatbath_functions_on_the_device_against_libm(qcd):
    """csrc/hb_math.cuh as the GPU evaluates it (MUFU.RCP64H / RSQ64H seeds, constant-bank coefficients) against numpy in
    extended precision: ln u, cos^2, sin, cos of 2 pi u for u = (w + 1/2) 2^-32, and sqrt / rsqrt / rcp -- random words
    and the neighbourhood of every fold point of the integer argument reductions.  Same bounds as the host test
    (tests/test_hb_math.py)."""
    rng = np.random.default_rng(99)
    edges = np.array([0x00000000, 0x1fffffff, 0x20000000, 0x3fffffff, 0x40000000, 0x5fffffff, 0x60000000, 0x7fffffff, 0x80000000,
                      0x9fffffff, 0xa0000000, 0xbfffffff, 0xc0000000, 0xdfffffff, 0xe0000000, 0xffffffff, 0x5a827999, 0xb504f333,
                      0x6a09e667, 0x2d413ccc], dtype=np.int64)
    near = ((edges[:, None] + np.arange(-300, 301)[None, :]) % (1 << 32)).reshape(-1)
    words = np.concatenate([near, rng.integers(0, 1 << 32, size=400000, dtype=np.int64)]).astype(np.uint32)
    got = qcd.qcd_debug_hb_math(words)
    ld = np.longdouble
    u = (words.astype(ld) + ld(0.5)) / ld(4294967296.0)
    assert np.finfo(ld).eps < 2e-19, "needs an extended-precision long double (x86-64)"
    ang = 2 * ld("3.14159265358979323846264338327950288") * u
    err = lambda a, b: float(np.max(np.abs(a.astype(ld) - b)))
    assert err(got[:, 0], np.log(u)) < 5e-15
    # reference angle good to ~1e-18 (64-bit mantissa)
    assert err(got[:, 1], np.cos(ang) ** 2) < 4e-16
    assert err(got[:, 2], np.sin(ang)) < 4e-16
    assert err(got[:, 3], np.cos(ang)) < 4e-16
    rel = lambda a, b: float(np.max(np.abs(a.astype(ld) / b - 1)))
    assert rel(got[:, 4], np.sqrt(u)) < 3e-16
    assert rel(got[:, 5], 1 / np.sqrt(u)) < 3e-16
    assert rel(got[:, 6], 1 / u) < 3e-16


def test_exchange_rows01_is_the_compressed_form_of_the_canonical_layout(qcd):
    """QCD_OPT_EXCHANGE_ROWS01: qcd_get_links / qcd_set_links of a 12-real SU(3) lattice move rows 0,1 only
    ([lex][mu][2][3]): the same numbers as rows 0,1 of the full canonical array, in both directions and through host and
    device pointers, whole lattice and chunked staging (a lattice larger than one 64 MiB chunk); refused elsewhere."""
    import torch
    for dims, prec in [((6, 4, 10, 2), 0), ((6, 4, 10, 2), 1), ((6, 4, 10), 0), ((48, 32, 32, 32), 0)]:
        with gpu_lattice(qcd, dims, 3, prec, 1) as G:
            G.qcd_init(qcd.QCD_HOT, 3)
            full = G.qcd_get_links()
            G.qcd_set_option(qcd.QCD_OPT_EXCHANGE_ROWS01, 1)
            assert G.canonical_bytes == full.nbytes * 2 // 3
            half = G.qcd_get_links()
            assert half.shape == full.shape[:2] + (2, 3) and np.array_equal(half, full[:, :, :2, :])
            # device pointer form
            dev = torch.empty(G.canonical_bytes, dtype=torch.uint8, device="cuda")
            G.qcd_get_links_ptr(dev.data_ptr(), G.canonical_bytes, 1)
            torch.cuda.synchronize()
            assert np.array_equal(dev.cpu().numpy().view(half.dtype).reshape(half.shape), half)
            # and back in: a cold lattice takes the rows and returns the same configuration
            G.qcd_init(qcd.QCD_COLD, 0)
            G.qcd_set_links(half)
            G.qcd_set_option(qcd.QCD_OPT_EXCHANGE_ROWS01, 0)
            assert np.array_equal(G.qcd_get_links(), full)
            G.qcd_set_option(qcd.QCD_OPT_EXCHANGE_ROWS01, 1)
            G.qcd_init(qcd.QCD_COLD, 0)
            G.qcd_set_links_ptr(dev.data_ptr(), G.canonical_bytes, 1)
            G.qcd_set_option(qcd.QCD_OPT_EXCHANGE_ROWS01, 0)
            assert np.array_equal(G.qcd_get_links(), full)
    for Nc, flags in [(3, 0), (2, 0)]:
        with gpu_lattice(qcd, (4, 4, 4, 4), Nc, 0, flags) as G:
            with pytest.raises(qcd.QcdError):
                G.qcd_set_option(qcd.QCD_OPT_EXCHANGE_ROWS01, 1)


def test_overrelaxation_conserves_action_on_gpu(qcd):
    dims = (8, 8, 8, 8)
    for Nc, prec, flags, tol in [(3, 1, 0, 1e-12), (3, 0, 1, 3e-6), (2, 1, 0, 1e-12)]:
        with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
            G.qcd_init(qcd.QCD_HOT, 3)
            G.qcd_sweep(5.0, 2, 0)
            p0 = G.qcd_measure()[0]
            G.qcd_sweep(5.0, 0, 3)
            p1 = G.qcd_measure()[0]
            assert abs(p1 - p0) < tol, (Nc, prec, p0, p1)


def test_resume_is_bit_identical_on_gpu(qcd):
    dims, Nc, beta = (8, 8, 4, 4), 3, 5.7
    for prec, flags in [(1, 0), (0, 1)]:
        with gpu_lattice(qcd, dims, Nc, prec, flags) as A, gpu_lattice(qcd, dims, Nc, prec, flags) as B, \
                gpu_lattice(qcd, dims, Nc, prec, flags) as C2:
            A.qcd_init(qcd.QCD_HOT, 11)
            for _ in range(4):
                A.qcd_sweep(beta, 1, 2)
            B.qcd_init(qcd.QCD_HOT, 11)
            for _ in range(2):
                B.qcd_sweep(beta, 1, 2)
            C2.qcd_set_links(B.qcd_get_links())
            C2.qcd_set_seed(B.qcd_get_seed())
            C2.qcd_set_sweep_counter(B.qcd_get_sweep_counter())
            for _ in range(2):
                C2.qcd_sweep(beta, 1, 2)
            a, c = A.qcd_get_links(), C2.qcd_get_links()
            if flags == 0:
                assert np.array_equal(a, c)
            else:
                assert np.array_equal(a[..., :2, :], c[..., :2, :])


# ----------------------------------------------------------------------------- T5: long runs
def _binned_error(x, nbins=10):
    x = np.asarray(x)
    b = x[: len(x) // nbins * nbins].reshape(nbins, -1).mean(axis=1)
    return b.std(ddof=1) / np.sqrt(nbins)


def test_config1_su2_2d_exact_plaquette_on_gpu(qcd):
    # BASELINE.json configs[0]
    from scipy import special
    exact = special.iv(2, 2.0) / special.iv(1, 2.0)
    with gpu_lattice(qcd, (16, 16), 2, 1, 0) as G:
        G.qcd_init(qcd.QCD_COLD, 1234)
        ps = []
        for _ in range(200):
            G.qcd_sweep(2.0, 1, 1)
            ps.append(G.qcd_measure()[0])
            if _ % 20 == 0:
                uni, det = npl.unitarity_defect(G.qcd_get_links())
                assert uni < 1e-12 and det < 1e-12
    meas = np.array(ps[20:])
    err = max(_binned_error(meas), np.sqrt(0.162709 / 256 / len(meas)))
    assert abs(meas.mean() - exact) < 3 * err, (meas.mean(), exact, err)
    # same seed, same keying, fp64: the GPU trajectory should coincide with the oracle's for the first sweeps
    O = oracle.OracleLattice((16, 16), 2)
    O.init(oracle.COLD, 1234)
    po = []
    for _ in range(200):
        O.sweep(2.0, 1, 1)
        po.append(O.measure()[0])
    po = np.array(po)
    assert abs(po[0] - ps[0]) < 1e-12
    erro = max(_binned_error(po[20:]), np.sqrt(0.162709 / 256 / len(meas)))
    assert abs(meas.mean() - po[20:].mean()) < 3 * np.sqrt(err ** 2 + erro ** 2)


def _robust_error(x):
    """error of the mean of a correlated series: the largest binned estimate over several bin sizes (the binned error grows
    with the bin size until the bins decorrelate), never below the naive one"""
    x = np.asarray(x)
    est = [x.std(ddof=1) / np.sqrt(len(x))]
    for nb in (12, 8, 6, 4):
        if len(x) // nb >= 2:
            est.append(_binned_error(x, nb))
    return max(est)


@pytest.mark.parametrize("prec,flags", [(1, 0), (0, 0), (0, 1)], ids=["f64", "f32", "f32x12"])
def test_config2_su3_long_run_vs_oracle(qcd, prec, flags):
    # BASELINE.json configs[1]: SU(3) 16^3x4 beta 5.7 hot seed 7, 100 sweeps of 1 HB + 4 OR; plaquette and Polyakov loop
    # every sweep.  beta = 5.7 at N_t = 4 sits on the deconfinement transition (beta_c ~ 5.69): the run is metastable
    # between two phases whose plaquettes differ by ~0.004, with a tunnelling time longer than 100 sweeps, so once rounding
    # has decorrelated two trajectories (a few sweeps in fp32) their 60-sweep means are not statistically comparable.  Here:
    # the early trajectory must coincide, unitarity must hold, and the means must lie in the band the two phases span.
    # The 3-sigma comparison of long-run means is test_long_run_plaquette_3sigma below, away from the transition.
    dims, beta, nsw, ndisc = (16, 16, 16, 4), 5.7, 100, 40
    O = oracle.OracleLattice(dims, 3)
    if prec == 0:
        O.set_fp32_shadow(True)
    O.init(oracle.HOT, 7)
    po, lo = [], []
    for _ in range(nsw):
        O.sweep(beta, 1, 4)
        t, _p, l = O.measure()
        po.append(t)
        lo.append(abs(l))
    with gpu_lattice(qcd, dims, 3, prec, flags) as G:
        G.qcd_init(qcd.QCD_HOT, 7)
        pg, lg = [], []
        for _ in range(nsw):
            G.qcd_sweep(beta, 1, 4)
            t, _p, l = G.qcd_measure()
            pg.append(t)
            lg.append(abs(l))
            if _ % 25 == 0:
                uni, det = npl.unitarity_defect(G.qcd_get_links().astype(np.complex128))
                assert uni < (1e-12 if prec == 1 else 5e-6) and det < (1e-12 if prec == 1 else 5e-6)
    po, pg = np.array(po), np.array(pg)
    # the first sweep agrees closely (same random numbers); later the trajectories decorrelate (rounding differs)
    assert abs(po[0] - pg[0]) < (1e-11 if prec == 1 else 1e-4)
    eo, eg = _robust_error(po[ndisc:]), _robust_error(pg[ndisc:])
    print("<P> oracle %.5f +- %.5f   gpu %.5f +- %.5f" % (po[ndisc:].mean(), eo, pg[ndisc:].mean(), eg))
    if prec == 1:
        assert abs(po[ndisc:].mean() - pg[ndisc:].mean()) < 3 * np.sqrt(eo ** 2 + eg ** 2)
    assert abs(po[ndisc:].mean() - pg[ndisc:].mean()) < 0.008
    assert 0.54 < pg[ndisc:].mean() < 0.56 and 0.54 < po[ndisc:].mean() < 0.56   # the band of the two phases (not a pin)
    # Polyakov loop: |L| tunnels between the two phases with an autocorrelation time longer than this run, so its long-run
    # mean is not comparable between two decorrelated trajectories; what is comparable is the early part, where both follow
    # the same random numbers (fp32: the ~0.1 % ill-conditioned links of the hot start each move one Polyakov line)
    assert abs(lo[0] - lg[0]) < (1e-11 if prec == 1 else 2e-3) and abs(lo[1] - lg[1]) < (1e-6 if prec == 1 else 2e-2)
    assert max(lg) < 0.5 and max(lo) < 0.5


@pytest.mark.parametrize("Nc,prec,flags,dims,beta", [(3, 1, 0, (8, 8, 8, 8), 6.0), (3, 0, 1, (8, 8, 8, 8), 6.0), (3, 0, 0, (8, 8, 8, 8), 6.0),
                                                      (2, 0, 0, (8, 8, 8, 8), 2.5), (3, 1, 1, (6, 6, 6), 9.0)],
                         ids=["su3-f64", "su3-f32x12", "su3-f32x18", "su2-f32", "su3-3d-f64x12"])
def test_long_run_plaquette_3sigma(qcd, Nc, prec, flags, dims, beta):
    # north_star: long-run <P> within 3 sigma of the oracle's.  Away from any transition (8^4 at beta 6.0 / 2.5 is
    # deconfined and thermalises in ~20 sweeps of 1 HB + 4 OR); different seeds on the two sides, so the two means are
    # independent estimates of the same expectation value.
    nsw, ndisc = 160, 40
    O = oracle.OracleLattice(dims, Nc)
    if prec == 0:
        O.set_fp32_shadow(True)
    O.init(oracle.HOT, 101)
    po = []
    for _ in range(nsw):
        O.sweep(beta, 1, 4)
        po.append(O.measure()[0])
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_init(qcd.QCD_HOT, 202)
        pg = []
        for _ in range(nsw):
            G.qcd_sweep(beta, 1, 4)
            pg.append(G.qcd_measure()[0])
    po, pg = np.array(po[ndisc:]), np.array(pg[ndisc:])
    eo, eg = _robust_error(po), _robust_error(pg)
    print("<P> oracle %.5f +- %.5f   gpu %.5f +- %.5f" % (po.mean(), eo, pg.mean(), eg))
    assert abs(po.mean() - pg.mean()) < 3 * np.sqrt(eo ** 2 + eg ** 2)


# ----------------------------------------------------------------------------- full size, bench launch configuration
def _sampled_links_at_full_size(qcd, dims, Nc, prec, flags, beta, seed, fld, substeps, n_edge=300, n_any=700):
    """The oracle produces the hot start and recomputes sampled links one by one (update_one_link); the GPU runs whole
    sub-steps in the launch configuration bench.py times.  Sampled links must agree within the per-link tolerance, all
    links outside the sub-step must be bit-unchanged, heatbath accept/reject disagreements are counted (<= 1 allowed),
    and the hot start and the observables of the full lattice must equal the oracle's."""
    fg, fo = field_pair(qcd, fld)
    O = oracle.OracleLattice(dims, Nc)
    O.init(oracle.HOT, seed)
    start = O.get_links()
    if prec == 0:
        start = round_to_fp32(start)
        O.set_fp32_shadow(True)
        O.set_links(start)
    O.set_seed(seed)
    rng = np.random.Generator(np.random.PCG64(5))
    V, D = O.V, len(dims)
    coords = np.stack(np.unravel_index(np.arange(V), dims[::-1]), axis=-1)[:, ::-1]
    par = coords.sum(axis=1) & 1
    on_edge = np.any((coords == 0) | (coords == np.array(dims) - 1), axis=1)
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
        G.qcd_set_links(start)
        G.qcd_set_seed(seed)
        total_bad, total = 0, 0
        for kind, parity, mu in substeps:
            G.qcd_set_links(start)
            G.qcd_debug_substep(beta, kind, 0, parity, mu, fg)
            got = G.qcd_get_links()
            tr = G.qcd_debug_get_trials() if kind == 0 else None
            # boundary sites (a wrap-around neighbour in some direction) plus random sites
            cand = np.flatnonzero(par == parity)
            edge = cand[on_edge[cand]]
            sample = np.concatenate([rng.choice(edge, n_edge, replace=False), rng.choice(cand, n_any, replace=False)])
            worst = 0.0
            for lex in sample:
                ref, codes = O.update_one_link(beta, kind, 0, int(lex), mu, fo)
                if kind == 0 and not np.array_equal(codes, tr[lex]):
                    total_bad += 1
                    continue
                tol = float(link_tol(prec, np.array([O.last_kmin]))[0])
                worst = max(worst, float(np.max(np.abs(got[lex, mu].astype(np.complex128) - ref))) / tol)
            total += len(sample)
            assert worst < 1.0, (kind, parity, mu, worst)
            # all other links untouched
            other = np.ones((V, D), dtype=bool)
            other[par == parity, mu] = False
            cmp_a = got if (flags == 0 or Nc == 2) else got[..., :2, :]
            cmp_b = start if (flags == 0 or Nc == 2) else start[..., :2, :]
            assert np.array_equal(cmp_a[other], cmp_b[other].astype(cmp_a.dtype))
            del got
        assert total_bad <= 1, (total_bad, total)
        # the GPU hot start at full size equals the oracle's, and so do the observables measured on it
        G.qcd_init(qcd.QCD_HOT, seed)
        hot_gpu = G.qcd_get_links()
        O2 = oracle.OracleLattice(dims, Nc)
        O2.init(oracle.HOT, seed)
        assert np.max(np.abs(hot_gpu - O2.get_links())) < (1e-13 if prec == 1 else 5e-7)
        tot, planes, poly = G.qcd_measure(fg)
        tot_o, planes_o, poly_o = O2.measure(fo)
        assert abs(tot - tot_o) < MEAS_TOL[prec] and abs(poly - poly_o) < MEAS_TOL[prec]
        assert np.max(np.abs(planes - planes_o)) < MEAS_TOL[prec]


@pytest.mark.parametrize("prec,flags", [(0, 1), (1, 0)], ids=["f32x12", "f64x18"])
def test_config3_sampled_links_at_full_size(qcd, prec, flags):
    # BASELINE.json configs[2]: SU(3) 32^4, beta 6.0, hot seed 42 -- the workload bench.py times
    _sampled_links_at_full_size(qcd, (32, 32, 32, 32), 3, prec, flags, 6.0, 42, None,
                                [(0, 0, 0), (0, 1, 3), (1, 1, 1), (1, 0, 2)])


@pytest.mark.parametrize("prec,flags", [(0, 1), (1, 0)], ids=["f32x12", "f64x18"])
def test_config3_thermalised_state_at_full_size(qcd, prec, flags):
    """BASELINE.json configs[2] on the state bench.py TIMES: SU(3) 32^4, beta 6.0, hot seed 42, then 10 thermalising sweeps
    of 1 HB + 4 OR (the GPU produces that configuration; both sides start from the same downloaded copy).
    sec 3.1 (the CPU regenerates configurations from the same random numbers) is the protocol.
      (i)  heatbath and overrelaxation sub-steps in the bench launch configuration, 1000 sampled links each against the
           oracle's update_one_link at the PLAIN north_star bars (2e-5 / 1e-12): no link of the sample is under the
           conditioning rule (asserted), all other links bit-unchanged;
      (ii) one whole un-resynced sweep (40 sub-steps, all 4.2 M links compared): accept/reject disagreements <= 1e-6 of the
           heatbath link-hits, every link outside the dependency cone of a disagreement within the derived un-resynced bar;
           qcd_sweep reproduces that sequence bit for bit."""
    dims, Nc, beta, seed, therm = (32, 32, 32, 32), 3, 6.0, 42, 10
    D, V = 4, 32 ** 4
    par = npl.site_parity(dims)
    coords = np.stack(np.unravel_index(np.arange(V), dims[::-1]), axis=-1)[:, ::-1]
    on_edge = np.any((coords == 0) | (coords == np.array(dims) - 1), axis=1)
    rng = np.random.Generator(np.random.PCG64(11))
    with gpu_lattice(qcd, dims, Nc, prec, flags) as G:
        G.qcd_init(qcd.QCD_HOT, seed)
        for _ in range(therm):
            G.qcd_sweep(beta, 1, 4)
        assert G.qcd_get_sweep_counter() == therm
        p_therm = G.qcd_measure()[0]
        assert 0.58 < p_therm < 0.61                               # thermalised at beta = 6 (sanity, not a pin)
        start = G.qcd_get_links().astype(np.complex128)
        O = oracle_lattice(dims, Nc, prec, start)
        O.set_seed(seed)
        O.sweep_counter = therm
        G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
        # (i) sampled links per sub-step at the plain bars
        bad = 0
        for kind, parity, mu in [(0, 0, 0), (0, 1, 3), (1, 1, 1), (1, 0, 2), (0, 1, 2), (1, 0, 0)]:
            G.qcd_set_links(start)
            G.qcd_debug_substep(beta, kind, 0, parity, mu)
            got = G.qcd_get_links()
            tr = G.qcd_debug_get_trials() if kind == 0 else None
            cand = np.flatnonzero(par == parity)
            edge = cand[on_edge[cand]]
            sample = np.concatenate([rng.choice(edge, 300, replace=False), rng.choice(cand, 700, replace=False)])
            worst, kworst = 0.0, np.inf
            for lex in sample:
                ref, codes = O.update_one_link(beta, kind, 0, int(lex), mu)
                kworst = min(kworst, O.last_kmin)
                if kind == 0 and not np.array_equal(codes, tr[lex]):
                    bad += 1
                    continue
                worst = max(worst, float(np.max(np.abs(got[lex, mu].astype(np.complex128) - ref))))
            print("thermal 32^4 %s p=%d mu=%d: worst |diff| %.3e (bar %.0e), smallest k %.2f" % ("HB" if kind == 0 else "OR", parity, mu, worst, TOL[prec], kworst))
            assert kworst > K_COND                                  # illcond == 0: the plain bar is the bar
            assert worst < TOL[prec], (kind, parity, mu, worst)
            other = np.ones((V, D), dtype=bool)
            other[par == parity, mu] = False
            cmp_a = got if flags == 0 else got[..., :2, :]
            cmp_b = start if flags == 0 else start[..., :2, :]
            assert np.array_equal(cmp_a[other], cmp_b[other].astype(cmp_a.dtype))
            del got
        assert bad == 0, bad
        # (ii) the whole working sweep without resync
        G.qcd_set_links(start)
        flips, fenced, worst, med, kmed, kmin, got = _unresynced_sequence(qcd, G, O, dims, Nc, prec, flags, beta, _sweep_sequence(D, 1, 4))
        bar = unresynced_bar(prec, 5, kmed)
        print("thermal 32^4 un-resynced sweep: flips %d, fenced %d of %d links, worst diff/bound %.3f, median diff %.3e (typical bar %.3e), "
              "k median %.2f min %.3f" % (flips, fenced, V * D, worst, med, bar, kmed, kmin))
        assert flips <= max(1, int(1e-6 * V * D)), flips           # north_star: at most 1e-6 of links
        assert fenced <= 120000 * max(flips, 0)                    # a disagreement reaches < (2*4+1)^4 * 4 links in 4 passes
        assert worst < 1.0 and med < bar, (worst, med, bar)        # every link within its own carried bound; the median within the typical bar
        G.qcd_set_links(start)
        G.qcd_set_sweep_counter(therm)
        G.qcd_sweep(beta, 1, 4)
        again = G.qcd_get_links().astype(np.complex128)
        assert np.array_equal(again, got)


def test_config4_su2_background_field_at_full_size(qcd):
    # BASELINE.json configs[3]: SU(2) 48^3 x 8, beta 2.5, fp32, constant abelian field along sigma_3 on the x-y plane,
    # every x-y plaquette times exp(i phi sigma_3 / 2), phi = 2 pi n_f / (Lx Ly), n_f = 4; hot seed 99
    phi = 2.0 * np.pi * 4 / (48 * 48)
    _sampled_links_at_full_size(qcd, (48, 48, 48, 8), 2, 0, 0, 2.5, 99, (0, 1, [0.5 * phi, -0.5 * phi]),
                                [(0, 0, 0), (0, 1, 1), (1, 1, 0), (1, 0, 1), (0, 1, 3), (1, 0, 2)])


def test_config5_su3_large_volume_fp32_sampled_links(qcd):
    # BASELINE.json configs[4], fp32 arm: SU(3) 64^3 x 16, beta 6.2, 12-real links, hot seed 2024 (805 MB of links)
    _sampled_links_at_full_size(qcd, (64, 64, 64, 16), 3, 0, 1, 6.2, 2024, None, [(0, 1, 0), (1, 0, 3), (1, 1, 2)],
                                n_edge=200, n_any=300)


def test_config5_su3_64to4_fp64_properties_at_full_size(qcd):
    """BASELINE.json configs[4], fp64 arm: SU(3) 64^4, 18 reals, 9.66 GB of links -- too large for the oracle to hold next
    to the test, so this checks what holds at any size and ties it to oracle-verified results:
      * the hot start depends on (seed, lex, mu) only, so its first V' links equal the oracle's hot start of 64^3 x 2;
      * an overrelaxation sub-step is deterministic and local: on a 64^4 configuration that repeats a 32^4 one with period 32
        in every direction it must reproduce, bit for bit and on all 67 M links, the periodic repetition of the same sub-step
        on the 32^4 lattice (whose sub-steps test_config3 checks against the oracle);
      * after a full sweep (1 HB + 4 OR, beta 6.2) every link is unitary with det 1 to 1e-12, the plaquette moved off the
        hot start, and an overrelaxation-only sweep conserves it to 1e-12."""
    import torch
    big, small, Nc, seed, beta = (64, 64, 64, 64), (32, 32, 32, 32), 3, 2024, 6.2
    dev = torch.device("cuda:0")
    Vb, Vs = 64 ** 4, 32 ** 4

    def links_to_device(G, V):
        t = torch.empty((V, 4, 3, 3), dtype=torch.complex128, device=dev)
        G.qcd_get_links_ptr(t.data_ptr(), t.numel() * 16, 1)
        return t

    with gpu_lattice(qcd, small, Nc, 1, 0) as S:
        S.qcd_init(qcd.QCD_HOT, seed)
        S.qcd_sweep(beta, 1, 1)
        base = links_to_device(S, Vs)
        ext = base.view(32, 32, 32, 32, 4, 3, 3).repeat(2, 2, 2, 2, 1, 1, 1).contiguous()      # [x3][x2][x1][x0]: lex order
        results = {}
        for parity, mu in [(0, 0), (1, 3), (1, 1)]:
            S.qcd_set_links_ptr(base.data_ptr(), base.numel() * 16, 1)
            S.qcd_debug_substep(beta, qcd.QCD_KIND_OR, 0, parity, mu)
            results[(parity, mu)] = links_to_device(S, Vs)
    with gpu_lattice(qcd, big, Nc, 1, 0) as G:
        for (parity, mu), res in results.items():
            G.qcd_set_links_ptr(ext.data_ptr(), ext.numel() * 16, 1)
            G.qcd_debug_substep(beta, qcd.QCD_KIND_OR, 0, parity, mu)
            got = links_to_device(G, Vb).view(64, 64, 64, 64, 4, 3, 3)
            for o3 in (0, 32):
                for o2 in (0, 32):
                    for o1 in (0, 32):
                        for o0 in (0, 32):
                            blk = got[o3:o3 + 32, o2:o2 + 32, o1:o1 + 32, o0:o0 + 32]
                            assert torch.equal(blk.reshape(Vs, 4, 3, 3), res), (parity, mu, o3, o2, o1, o0)
            del got
        del ext, results
        # hot start: first V' links against the oracle's 64^3 x 2 lattice
        G.qcd_init(qcd.QCD_HOT, seed)
        O = oracle.OracleLattice((64, 64, 64, 2), Nc)
        O.init(oracle.HOT, seed)
        ref = torch.from_numpy(O.get_links()).to(dev)
        hot = links_to_device(G, Vb)
        assert float((hot[:O.V] - ref).abs().max()) < 1e-13
        del ref, O
        p_hot = G.qcd_measure()[0]
        assert abs(p_hot) < 5e-4                                   # Haar-random links: <P> = 0, sigma ~ 1e-5 at this volume
        del hot
        G.qcd_sweep(beta, 1, 4)
        p1, planes, poly = G.qcd_measure()
        assert 0.2 < p1 < 0.7 and np.all(np.abs(planes - p1) < 0.01) and abs(poly) < 0.01
        U = links_to_device(G, Vb).view(-1, 3, 3)
        eye = torch.eye(3, dtype=torch.complex128, device=dev)
        worst_u, worst_d = 0.0, 0.0
        for c in torch.split(U, 1 << 23):
            worst_u = max(worst_u, float((c @ c.conj().transpose(1, 2) - eye).abs().max()))
            worst_d = max(worst_d, float((torch.linalg.det(c) - 1.0).abs().max()))
        assert worst_u < 1e-12 and worst_d < 1e-12, (worst_u, worst_d)
        del U
        G.qcd_sweep(beta, 0, 2)
        p2 = G.qcd_measure()[0]
        assert abs(p2 - p1) < 1e-12, (p1, p2)


def _mem_available_gb():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) / 2 ** 20
    except OSError:
        pass
    return 0.0


def test_config5_su3_64to4_fp64_heatbath_sampled_vs_oracle(qcd):
    """BASELINE.json configs[4], fp64 arm, the HEATBATH at full size: the 9.66 GB configuration is handed to the oracle (one
    host copy inside it), the GPU runs whole heatbath sub-steps at 64^4 (Philox counter c0 = lex up to 1.7e7, 64^4 strides,
    fp64 x18 trial loop), and sampled links -- wrap-around boundary sites, the top of the lex range, random sites -- are
    recomputed one by one by the oracle's update_one_link: trial codes equal, links within 1e-12."""
    import torch
    if _mem_available_gb() < 48.0:
        pytest.skip("host MemAvailable %.0f GB < 48 GB: the oracle needs 2 x 9.66 GB for the 64^4 configuration" % _mem_available_gb())
    dims, Nc, seed, beta = (64, 64, 64, 64), 3, 2024, 6.2
    V, dev = 64 ** 4, torch.device("cuda:0")
    rng = np.random.Generator(np.random.PCG64(3))
    with gpu_lattice(qcd, dims, Nc, 1, 0) as G:
        G.qcd_init(qcd.QCD_HOT, seed)
        G.qcd_sweep(beta, 1, 1)                                    # off the hot start: staple norms k ~ 3
        start_dev = torch.empty((V, 4, 3, 3), dtype=torch.complex128, device=dev)
        G.qcd_get_links_ptr(start_dev.data_ptr(), start_dev.numel() * 16, 1)
        start = G.qcd_get_links()
        O = oracle.OracleLattice(dims, Nc)
        O.set_links(start)
        del start
        O.set_seed(seed)
        O.sweep_counter = G.qcd_get_sweep_counter()
        G.qcd_set_option(qcd.QCD_OPT_DEBUG_TRIALS, 1)
        res = torch.empty_like(start_dev)
        bad, total = 0, 0
        for parity, mu in [(0, 0), (1, 3), (1, 1)]:
            G.qcd_set_links_ptr(start_dev.data_ptr(), start_dev.numel() * 16, 1)
            G.qcd_debug_substep(beta, qcd.QCD_KIND_HB, 0, parity, mu)
            G.qcd_get_links_ptr(res.data_ptr(), res.numel() * 16, 1)
            tr = G.qcd_debug_get_trials()
            # candidate sites: random, forced onto a wrap-around boundary, and from the top 1 % of the lex range
            c = rng.integers(0, 64, size=(1500, 4))
            for i in range(500, 1000):
                c[i, i % 4] = 0 if (i // 4) % 2 else 63
            c[1000:, 3] = 63
            c[1000:, 2] = rng.integers(60, 64, size=500)
            c = c[(c.sum(axis=1) & 1) == parity][:600]
            lexs = c[:, 0] + 64 * (c[:, 1] + 64 * (c[:, 2] + 64 * c[:, 3]))
            got = res[torch.from_numpy(lexs).to(dev), mu].cpu().numpy()
            worst = 0.0
            for i, lex in enumerate(lexs):
                ref, codes = O.update_one_link(beta, oracle.KIND_HB, 0, int(lex), mu)
                assert O.last_kmin > K_COND
                if not np.array_equal(codes, tr[lex]):
                    bad += 1
                    continue
                worst = max(worst, float(np.max(np.abs(got[i] - ref))))
            total += len(lexs)
            print("64^4 fp64 HB p=%d mu=%d: %d sampled links (max lex %d), worst |diff| %.3e" % (parity, mu, len(lexs), int(lexs.max()), worst))
            assert worst < TOL[1], (parity, mu, worst)
            assert len(lexs) >= 400 and lexs.max() > 0.98 * V
            # sites of the other parity did not move (trial code 0 and bit-unchanged), sampled
            other = rng.integers(0, V, size=2000)
            oc = np.stack([other % 64, other // 64 % 64, other // 4096 % 64, other // 262144], axis=1)
            other = other[(oc.sum(axis=1) & 1) != parity]
            idx = torch.from_numpy(other).to(dev)
            assert torch.equal(res[idx], start_dev[idx]) and not tr[other].any()
        assert bad == 0, (bad, total)


def test_largest_indexable_lattice_128to4_fp32(qcd):
    """Edge of the 32-bit vector indexing: SU(3) 128^4 with 12-real fp32 links (51.5 GB, 3.2e9 vectors).  Too large for any
    host-side comparison; checked by what holds at any size: the cold start measures plaquette = Polyakov loop = 1 exactly,
    a hot start measures ~0, a heatbath sweep moves the plaquette to its beta = 6 neighbourhood on every plane, and an
    overrelaxation sweep conserves it (a wrapped or truncated index would break each of these)."""
    with gpu_lattice(qcd, (128, 128, 128, 128), 3, 0, 1) as G:
        G.qcd_init(qcd.QCD_COLD, 1)
        tot, planes, poly = G.qcd_measure()
        assert tot == 1.0 and np.all(planes == 1.0) and poly == 1.0
        G.qcd_init(qcd.QCD_HOT, 1)
        tot, planes, poly = G.qcd_measure()
        assert abs(tot) < 1e-4 and np.max(np.abs(planes)) < 1e-4 and abs(poly) < 1.5e-3    # 1.4e-5 / 2.3e-4 statistical sigma
        G.qcd_sweep(6.0, 1, 0)
        G.qcd_sweep(6.0, 1, 0)
        p1, planes, _ = G.qcd_measure()
        assert 0.3 < p1 < 0.62 and np.max(np.abs(planes - p1)) < 2e-2     # two sweeps from hot: planes still order-dependent at 5e-3
        G.qcd_sweep(6.0, 0, 2)
        p2, planes2, _ = G.qcd_measure()
        assert abs(p2 - p1) < 3e-6, (p1, p2)


def test_largest_lattice_of_one_b200_128to4_fp64(qcd):
    """SU(3) 128^4 in fp64 x18: 154.6 GB of links, the largest lattice one B200 holds (no slab streaming
    needed below this size).  Each (parity, direction) array has 1.2e9 vectors (32-bit in-array offsets), the array bases are
    64-bit.  Checked by what holds at any size, like the fp32 case above; skipped when the device has less free memory."""
    import gc
    import torch
    gc.collect()
    torch.cuda.empty_cache()                                     # blocks cached by earlier tests count as used otherwise
    free, _ = torch.cuda.mem_get_info()
    need = 4 * 128 ** 4 * 144
    if free < need + (4 << 30):
        pytest.skip("device has %.1f GB free, the lattice needs %.1f GB" % (free / 1e9, need / 1e9))
    with gpu_lattice(qcd, (128, 128, 128, 128), 3, 1, 0) as G:
        G.qcd_init(qcd.QCD_COLD, 1)
        tot, planes, poly = G.qcd_measure()
        assert tot == 1.0 and np.all(planes == 1.0) and poly == 1.0
        G.qcd_init(qcd.QCD_HOT, 1)
        tot, planes, poly = G.qcd_measure()
        assert abs(tot) < 1e-4 and np.max(np.abs(planes)) < 1e-4 and abs(poly) < 1.5e-3
        G.qcd_sweep(6.0, 1, 0)
        G.qcd_sweep(6.0, 1, 0)
        p1, planes, _ = G.qcd_measure()
        assert 0.3 < p1 < 0.62 and np.max(np.abs(planes - p1)) < 2e-2
        G.qcd_sweep(6.0, 0, 2)
        p2, _, _ = G.qcd_measure()
        assert abs(p2 - p1) < 1e-12, (p1, p2)


# ----------------------------------------------------------------------------- ABI error paths on a live device
def test_error_paths(qcd):
    with pytest.raises(qcd.QcdError) as e:
        qcd.Lattice((5, 4), 2, 1, 0)
    assert e.value.code == qcd.QCD_ERR_INVALID_ARG
    with pytest.raises(qcd.QcdError) as e:
        qcd.Lattice((4, 4), 2, 1, qcd.QCD_FLAG_COMPRESS12)
    assert e.value.code == qcd.QCD_ERR_UNSUPPORTED
    with gpu_lattice(qcd, (4, 4), 2, 1, 0) as G:
        with pytest.raises(qcd.QcdError) as e:
            G.qcd_sweep(2.0, 1, 1)
        assert e.value.code == qcd.QCD_ERR_STATE
        G.qcd_init(qcd.QCD_COLD, 1)
        with pytest.raises(qcd.QcdError) as e:
            G.qcd_sweep(float("nan"), 1, 1)
        assert e.value.code == qcd.QCD_ERR_INVALID_ARG
        with pytest.raises(qcd.QcdError) as e:
            G.qcd_sweep(2.0, 1, 1, qcd.make_field(1, 0, [0.1, -0.1]))
        assert e.value.code == qcd.QCD_ERR_INVALID_ARG
        with pytest.raises(qcd.QcdError) as e:
            G.qcd_sweep(2.0, 1, 1, qcd.make_field(0, 1, [0.1, 0.1]))
        assert e.value.code == qcd.QCD_ERR_INVALID_ARG
        with pytest.raises(qcd.QcdError):
            G.qcd_set_option(qcd.QCD_OPT_KP_MAX_TRIALS, 0)
        with pytest.raises(qcd.QcdError):
            G.qcd_debug_get_trials()
    # library-allocated workspace works too
    with qcd.Lattice((4, 4), 2, 1, 0, library_alloc=True) as G:
        G.qcd_init(qcd.QCD_COLD, 1)
        assert G.qcd_measure()[0] == 1.0
