"""CPU checks of the tolerance rules the GPU parity tests apply (tests/tolerances.py): the ceiling of the
fp32 conditioning rule, and the derived Haar expectation of how many links fall under it, against the conditioning numbers
the oracle reports."""
import numpy as np
import pytest

import oracle
from tests import tolerances as T
from tests.inputs import random_links


def test_conditioning_rule_has_a_ceiling():
    k = np.array([np.inf, 4.0, 0.25, 0.2, 0.025, 2.5e-3, 1e-4, 1e-9, 0.0])
    t32 = T.link_tol(0, k)
    assert np.all(t32[:3] == 2e-5) and t32[3] == pytest.approx(2.5e-5) and t32[4] == pytest.approx(2e-4)
    assert np.all(t32[5:] == pytest.approx(T.TOL_CEIL)) and t32.max() <= T.TOL_CEIL       # never "no bar at all"
    assert np.all(T.link_tol(1, k) == 1e-12)                                               # fp64: the plain bar, always


@pytest.mark.parametrize("Nc,dims", [(3, (16, 16)), (3, (8, 8, 8)), (3, (8, 8, 8, 4)), (2, (16, 16)), (2, (8, 8, 8)), (2, (8, 8, 8, 4))])
def test_haar_expectation_of_illconditioned_links(Nc, dims):
    """the fraction of Haar-input link updates with k_min < K_COND stays under the bound derived in tests/tolerances.py"""
    D = len(dims)
    links = random_links(dims, Nc, 5)
    total, ill = 0, 0
    for kind in (oracle.KIND_HB, oracle.KIND_OR):
        for parity in (0, 1):
            for mu in range(D):
                O = oracle.OracleLattice(dims, Nc)
                O.set_links(links)
                O.set_seed(3)
                _, kmin = O.substep_diag(5.7 if Nc == 3 else 2.5, kind, 0, parity, mu)
                f = np.isfinite(kmin)
                total += int(f.sum())
                ill += int((kmin[f] < T.K_COND).sum())
    assert ill <= T.illcond_bound(Nc, D, total), (ill, total, T.expected_illcond_fraction(Nc, D))
    # and the estimate is not vacuous: it is within a factor of ~4 of what is seen where counts allow a statement
    if ill >= 20:
        assert ill >= 0.25 * T.expected_illcond_fraction(Nc, D) * total


def test_thermal_inputs_are_well_conditioned():
    links = random_links((8, 8, 8, 4), 3, 17, 0.35)
    O = oracle.OracleLattice((8, 8, 8, 4), 3)
    O.set_links(links)
    _, kmin = O.substep_diag(5.7, oracle.KIND_OR, 0, 0, 1)
    k = kmin[np.isfinite(kmin)]
    assert k.min() > T.K_COND and np.median(k) > 3.0
    assert T.unresynced_bar(0, 5, float(np.median(k))) < 2e-4 and T.unresynced_bar(1, 5, float(np.median(k))) < 1e-11


def test_staple_dependents_matches_the_oracles_staple_by_brute_force():
    """tests/np_lattice.staple_dependents (the fence around a heatbath disagreement in the un-resynced GPU tests): marking one
    link must flag exactly the sites whose staple sum, or own link, the oracle sees change when that link is replaced"""
    from tests import np_lattice as npl
    dims, D = (4, 6, 4, 2), 4
    V = int(np.prod(dims))
    links = random_links(dims, 3, 1)
    O = oracle.OracleLattice(dims, 3)
    O.set_links(links)
    base = {(x, mu): O.staple(x, mu) for x in range(V) for mu in range(D)}
    rng = np.random.default_rng(0)
    for _ in range(5):
        lx, lm = int(rng.integers(V)), int(rng.integers(D))
        l2 = links.copy()
        l2[lx, lm] = l2[lx, lm] @ links[(lx + 1) % V, 0]
        O2 = oracle.OracleLattice(dims, 3)
        O2.set_links(l2)
        mask = np.zeros((V, D), dtype=bool)
        mask[lx, lm] = True
        for mu in range(D):
            dep = npl.staple_dependents(mask, dims, mu)
            changed = np.array([np.max(np.abs(O2.staple(x, mu) - base[(x, mu)])) > 0 for x in range(V)])
            changed[lx] |= (mu == lm)
            assert np.array_equal(dep, changed)
    par = npl.site_parity(dims)
    assert par[0] == 0 and par[1] == 1 and par[dims[0]] == 1 and par.sum() == V // 2
