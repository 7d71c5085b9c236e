"""Pins for the O(N)-model oracle (oracle/on_oracle.cpp) against what mathematics fixes (CPU only).
None of the expected values comes from the oracle or from the CUDA path: known-answer vectors, an independent numpy
recomputation from the definition of the action, closed forms (radial quadrature, the free lattice propagator), limits."""
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import on

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers_and_number_packing():
    # the published Philox4x32-10 vectors (tests/golden/philox4x32_10_kat.txt): this oracle restates the function itself
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert list(on.philox4x32_10(v[0:4], v[4:6])) == v[6:10]
    # R18: counter packing and the five 23-bit numbers, hand-packed here from the block
    rng = np.random.default_rng(1)
    for _ in range(200):
        seed = int(rng.integers(0, 2 ** 63))
        lex, sweep, parity, hit, domain = int(rng.integers(0, 2 ** 31)), int(rng.integers(0, 2 ** 32)), int(rng.integers(0, 2)), int(rng.integers(0, 65536)), int(rng.integers(2, 4))
        w = on.philox4x32_10([lex, sweep, (parity << 4) | (hit << 8) | (domain << 24), 0], [seed & 0xFFFFFFFF, seed >> 32]).astype(np.uint64)
        k = on.block_numbers(seed, lex, sweep, parity, hit, domain)
        assert list(k[:4]) == [int(x) & 0x7FFFFF for x in w]
        assert int(k[4]) == (int(w[0]) >> 23) | ((int(w[1]) >> 23) << 9) | (((int(w[2]) >> 23) & 31) << 18)
        assert all(int(x) < 2 ** 23 for x in k)


def test_numbers_are_uniform_and_independent():
    ks = np.array([on.block_numbers(7, lex, 3, lex & 1, lex % 50, 2) for lex in range(40000)], dtype=np.float64)
    u = (ks + 0.5) / 2 ** 23
    for a in range(5):
        obs = np.histogram(u[:, a], bins=64, range=(0, 1))[0]
        chi2 = np.sum((obs - len(u) / 64) ** 2 / (len(u) / 64))
        assert chi2 < 63 + 5 * np.sqrt(126), (a, chi2)
    c = np.corrcoef(u.T)
    assert np.max(np.abs(c - np.eye(5))) < 5 / np.sqrt(len(u))


def _np_action(phi, dims, kappa, lam):
    """S = sum_x [ -2 kappa sum_mu phi(x).phi(x+mu) + phi.phi + lam (phi.phi - 1)^2 ]  (reading R16), numpy roll"""
    D = len(dims)
    g = phi.reshape(tuple(reversed(dims)) + (phi.shape[1],))
    pp = (g * g).sum(-1)
    S = (pp + lam * (pp - 1.0) ** 2).sum()
    for mu in range(D):
        S -= 2.0 * kappa * (g * np.roll(g, -1, axis=D - 1 - mu)).sum()
    return S


@pytest.mark.parametrize("dims,N", [((4, 6), 1), ((4, 4, 2), 3), ((4, 2, 6, 2), 4), ((2, 2, 2, 2), 2)])
def test_action_and_one_hit_against_the_definition(dims, N):
    """total action = the definition; one try per site (NHIT = 1) = accept iff u < exp(-(global action difference)) with the
    proposal phi + delta (2u - 1): recomputed here site by site from the definition, not from the oracle's local formula"""
    kappa, lam, delta = 0.13, 0.7, 0.8
    V = int(np.prod(dims))
    rng = np.random.default_rng(3)
    phi = rng.uniform(-1.5, 1.5, size=(V, N))
    O = on.OnOracle(dims, N)
    O.set_field(phi)
    assert abs(O.action(kappa, lam) - _np_action(phi, dims, kappa, lam)) < 1e-10
    # O(N) invariance of the action (global rotation)
    q, _ = np.linalg.qr(rng.standard_normal((N, N)))
    O.set_field(phi @ q.T)
    assert abs(O.action(kappa, lam) - _np_action(phi, dims, kappa, lam)) < 1e-10
    O.set_field(phi)
    O.set_seed(99)
    O.sweep_counter = 5
    par = np.stack(np.unravel_index(np.arange(V), dims[::-1]), axis=-1).sum(1) & 1
    for parity in (0, 1):
        before = O.get_field()
        O.half_sweep(parity, kappa, lam, delta, 1)
        after = O.get_field()
        S0 = _np_action(before, dims, kappa, lam)
        n_acc = 0
        for lex in np.flatnonzero(par == parity):
            k = on.block_numbers(99, lex, 5, parity, 0, 2).astype(np.float64)
            u = (k + 0.5) / 2 ** 23
            trial = before.copy()
            trial[lex] = before[lex] + delta * (2.0 * u[:N] - 1.0)
            dS = _np_action(trial, dims, kappa, lam) - S0            # sites of one parity do not interact
            want = trial[lex] if u[4] < np.exp(-dS) else before[lex]
            n_acc += int(u[4] < np.exp(-dS))
            assert np.allclose(after[lex], want, rtol=0, atol=1e-14), (lex, dS)
        assert np.array_equal(after[par != parity], before[par != parity])
        assert 0 < n_acc < V // 2


@pytest.mark.parametrize("dims,N", [((4, 6), 1), ((4, 4, 2), 3), ((4, 2, 6, 2), 4), ((2, 2, 2, 2), 2), ((6, 4, 2), 4)])
def test_measure_against_the_definitions(dims, N):
    """R19 on a fixed random field, element-wise: phi2 = (1/V) sum_x phi.phi, link = (1/(V D)) sum_x sum_mu phi(x).phi(x+mu),
    mag_a = (1/V) sum_x phi_a, each recomputed here with numpy (roll for the neighbour).  The field has a non-zero mean in
    every component, distinct per component, and the extents differ, so a wrong normalisation (V D for V, a dropped 1/D),
    a swapped component or a wrong neighbour changes the number."""
    D, V = len(dims), int(np.prod(dims))
    rng = np.random.default_rng(17)
    phi = rng.uniform(-1.0, 1.0, size=(V, N)) + 0.3 * (1.0 + np.arange(N))
    O = on.OnOracle(dims, N)
    O.set_field(phi)
    p2, lk, mag = O.measure()
    g = phi.reshape(tuple(reversed(dims)) + (N,))
    assert abs(p2 - (g * g).sum() / V) < 1e-13
    link = sum((g * np.roll(g, -1, axis=D - 1 - mu)).sum() for mu in range(D)) / (V * D)
    assert abs(lk - link) < 1e-13
    assert mag.shape == (N,) and np.max(np.abs(mag - phi.mean(axis=0))) < 1e-13
    assert np.min(np.abs(np.diff(phi.mean(axis=0)))) > 0.1 if N > 1 else True
    # the backward neighbour gives the same link sum (periodic lattice); a constant field gives phi2 = link = |c|^2, mag = c
    link_b = sum((g * np.roll(g, +1, axis=D - 1 - mu)).sum() for mu in range(D)) / (V * D)
    assert abs(lk - link_b) < 1e-13
    c = 0.25 * (1.0 + np.arange(N))
    O.set_field(np.broadcast_to(c, (V, N)).copy())
    p2, lk, mag = O.measure()
    assert abs(p2 - c @ c) < 1e-14 and abs(lk - c @ c) < 1e-14 and np.max(np.abs(mag - c)) < 1e-15


def _radial_moment(N, lam):
    w = lambda r: r ** (N - 1) * np.exp(-r * r - lam * (r * r - 1.0) ** 2)
    z = integrate.quad(w, 0, np.inf)[0]
    return integrate.quad(lambda r: r * r * w(r), 0, np.inf)[0] / z


@pytest.mark.parametrize("N,lam", [(1, 0.0), (2, 0.5), (4, 0.5), (4, 2.0), (3, 10.0)])
def test_decoupled_sites_against_radial_quadrature(N, lam):
    """kappa = 0: every site is an independent chain with density exp(-phi^2 - lam (phi^2 - 1)^2) on R^N:
    <phi^2> = int r^(N+1) w / int r^(N-1) w.  Pins the on-site terms and the Metropolis rule (lam = 0, N = 1: <phi^2> = 1/2)."""
    dims = (8, 8, 4)
    O = on.OnOracle(dims, N)
    O.init(on.HOT, 11)
    delta = 1.0 if lam < 5 else 0.4
    per_site = []
    for s in range(60):
        O.sweep(0.0, lam, delta, 10)
        if s >= 10:
            per_site.append((O.get_field() ** 2).sum(1))
    x = np.mean(per_site, axis=0)                       # one time average per independent site
    exact = _radial_moment(N, lam)
    assert abs(x.mean() - exact) < 4.5 * x.std(ddof=1) / np.sqrt(len(x)), (x.mean(), exact)
    if lam == 0.0:
        assert abs(exact - 0.5 * N) < 1e-9


@pytest.mark.parametrize("dims,N,kappa", [((16, 16), 1, 0.2), ((6, 6, 6), 2, 0.12), ((4, 4, 4, 4), 4, 0.1)])
def test_free_field_against_the_lattice_propagator(dims, N, kappa):
    """lam = 0: S = sum_p |phi_p|^2 (1 - 2 kappa sum_mu cos p_mu) per component, so
    <phi.phi> = (N/V) sum_p 1 / (2 (1 - 2 kappa sum cos p)),  <phi(x).phi(x+mu)> = (N/V) sum_p cos p_mu / (2 (1 - 2 kappa sum cos p)).
    Pins the hopping term (sign, the factor 2 kappa, both neighbours in every direction)."""
    D = len(dims)
    grids = np.meshgrid(*[2 * np.pi * np.arange(L) / L for L in dims], indexing="ij")
    csum = sum(np.cos(g) for g in grids)
    denom = 2.0 * (1.0 - 2.0 * kappa * csum)
    assert denom.min() > 0
    V = int(np.prod(dims))
    phi2_exact = N * np.sum(1.0 / denom) / V
    link_exact = N * np.sum(csum / D / denom) / V
    O = on.OnOracle(dims, N)
    O.init(on.HOT, 5)
    p2, lk = [], []
    for s in range(700):
        O.sweep(kappa, 0.0, 1.2, 4)
        if s >= 100:
            a, b, _ = O.measure()
            p2.append(a)
            lk.append(b)

    def err(x, nb=20):
        b = np.asarray(x)[: len(x) // nb * nb].reshape(nb, -1).mean(1)
        return b.std(ddof=1) / np.sqrt(nb)

    assert abs(np.mean(p2) - phi2_exact) < 4.5 * err(p2), (np.mean(p2), phi2_exact, err(p2))
    assert abs(np.mean(lk) - link_exact) < 4.5 * err(lk), (np.mean(lk), link_exact, err(lk))
    assert link_exact > 0.01                                  # a dropped or sign-flipped hopping term would give <= 0


def test_strong_self_coupling_pins_the_length():
    # lambda -> infinity: phi.phi -> 1 (the non-linear sigma model limit): fluctuation of phi^2 ~ 1/sqrt(2 lambda)
    O = on.OnOracle((4, 4, 4), 3)
    O.init(on.COLD, 1)
    for _ in range(30):
        O.sweep(0.1, 2e4, 0.01, 20)
    r2 = (O.get_field() ** 2).sum(1)
    assert abs(r2.mean() - 1.0) < 5e-3 and r2.std() < 0.02


def test_starts_bookkeeping_and_resume():
    dims, N = (4, 6, 4), 4
    V = int(np.prod(dims))
    O = on.OnOracle(dims, N)
    O.init(on.COLD, 3)
    assert np.array_equal(O.get_field(), np.tile([1.0, 0, 0, 0], (V, 1))) and O.sweep_counter == 0
    big = on.OnOracle((16, 16, 16), 3)
    big.init(on.HOT, 3)
    f = big.get_field()
    assert np.all(np.abs(f) < 1.0) and abs(f.mean()) < 4.5 / np.sqrt(3 * f.size) and abs(f.var() - 1.0 / 3) < 0.01
    O.init(on.HOT, 3)
    start = O.get_field()
    O.sweep(0.1, 0.5, 0.5, 0)                                  # no tries: nothing moves, the counter still advances
    assert np.array_equal(O.get_field(), start) and O.sweep_counter == 1 and O.counts() == (0, 0)
    O.sweep(0.1, 0.5, 0.5, 7)
    acc, tried = O.counts()
    assert tried == V * 7 and 0 < acc < tried and O.sweep_counter == 2
    # same seed reproduces, another seed does not; 2k sweeps = k + state transfer + k
    A, B, C2 = on.OnOracle(dims, N), on.OnOracle(dims, N), on.OnOracle(dims, N)
    A.init(on.HOT, 8)
    B.init(on.HOT, 8)
    for _ in range(4):
        A.sweep(0.12, 0.5, 0.6, 5)
    for _ in range(2):
        B.sweep(0.12, 0.5, 0.6, 5)
    C2.set_field(B.get_field())
    C2.set_seed(8)
    C2.sweep_counter = B.sweep_counter
    for _ in range(2):
        C2.sweep(0.12, 0.5, 0.6, 5)
    assert np.array_equal(A.get_field(), C2.get_field())
    B.init(on.HOT, 9)
    assert not np.array_equal(B.get_field(), start)
    # fp32 shadow: the stored field is float-representable
    S = on.OnOracle(dims, N)
    S.set_fp32_shadow(True)
    S.init(on.HOT, 8)
    S.sweep(0.12, 0.5, 0.6, 5)
    g = S.get_field()
    assert np.array_equal(g, g.astype(np.float32).astype(np.float64))
