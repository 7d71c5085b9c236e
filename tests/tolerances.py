"""Tolerances of the GPU-vs-oracle parity tests and the arithmetic they are derived from.

north_star: links per element max abs 1e-12 (fp64) / 2e-5 (fp32) per sub-step from a common pre-state.  Holds no method
arithmetic: only the bars, and the statistics of the conditioning number k the oracle reports.
"""
import numpy as np

TOL = {0: 2e-5, 1: 1e-12}          # per-element max abs, by precision (0 = fp32, 1 = fp64)
MEAS_TOL = {0: 2e-6, 1: 1e-12}     # observables (means over the lattice)

# Conditioning rule, fp32 only.  A subgroup hit maps the projected staple v (k = |v|) to v / k; that map has Lipschitz
# constant 1/k, and fp32 rounding of v is ~3e-7 absolute whatever k is.  For k >= K_COND the plain north_star bar applies.
# A link whose smallest subgroup norm is k < K_COND (met on Haar-random inputs only: thermalised links have k ~ 4) gets
# the bar TOL * K_COND / k, and the rule has a CEILING: the bar never exceeds TOL_CEIL (k is floored at
# K_FLOOR = K_COND * TOL / TOL_CEIL = 2.5e-3; below that a link must still agree to 2e-3, which an O(1) error fails).
K_COND = 0.25
TOL_CEIL = 2e-3
K_FLOOR = K_COND * TOL[0] / TOL_CEIL


def link_tol(prec, kmin):
    """per-link tolerance array from the oracle's conditioning numbers kmin (inf where the link was not updated)"""
    t = np.full(np.shape(kmin), TOL[prec])
    if prec == 0:
        small = np.asarray(kmin) < K_COND
        t[small] = np.minimum(TOL_CEIL, TOL[prec] * K_COND / np.maximum(np.asarray(kmin)[small], K_FLOOR))
    return t


def expected_illcond_fraction(Nc, D):
    """Expected fraction of link updates with k_min < K_COND on HAAR-random links.

    W = U A with A the sum of n = 2(D-1) staples, each Haar-distributed and independent, so the quaternion projection v of a
    2 x 2 block of W has 4 real components of variance sigma^2 = n/12 each (SU(3): E|M_ij|^2 = 1/3, a component is half the sum
    of two real or imaginary parts) or n/4 (SU(2): a unit quaternion).  For n >= 4 v is close to a 4-d Gaussian:
        P(|v| < K) = 1 - exp(-x) (1 + x),  x = K^2 / (2 sigma^2)      (chi-square with 4 degrees of freedom)
    times the number of subgroup hits (3 for SU(3), taken as independent: an upper estimate).  For SU(2) in D = 2 (two unit
    quaternions at angle psi, density (2/pi) sin^2 psi, |v| = 2 cos(psi/2)):  P = (2/pi) K^3 / 3 to leading order."""
    n = 2 * (D - 1)
    if Nc == 2 and D == 2:
        return (2.0 / np.pi) * K_COND ** 3 / 3.0
    sigma2 = n * (1.0 / 12 if Nc == 3 else 1.0 / 4)
    x = K_COND ** 2 / (2.0 * sigma2)
    return (3 if Nc == 3 else 1) * (1.0 - np.exp(-x) * (1.0 + x))


def illcond_bound(Nc, D, n_links):
    """upper bound asserted on the COUNT of links under the conditioning rule among n_links Haar-input updates:
    twice the expectation plus 6 Poisson sigmas (and a floor of 6 links for tiny lattices)"""
    e = expected_illcond_fraction(Nc, D) * n_links
    return 2.0 * e + 6.0 * np.sqrt(e) + 6.0


def unresynced_bar(prec, n_hits, k_typ=3.5):
    """bar for a link after n_hits un-resynced link-hits on a THERMALISED configuration: every hit adds at
    most the single-sub-step bar TOL, and the error already carried by the 18 neighbour links of a staple sum is passed on
    with the RMS gain g = sqrt(18) / k (independent errors; k >= k_typ is asserted from the oracle's conditioning numbers):
        bar = TOL * sum_{i<n} g^i"""
    g = np.sqrt(18.0) / k_typ
    return TOL[prec] * sum(g ** i for i in range(n_hits))


def carry_bound(B, rms_nbr, k, tol, updated, mu):
    """Per-link error bound after one more un-resynced sub-step.  B: (V, D) bounds so far; rms_nbr: (V,)
    RMS-combined bounds of the 18 staple links (tests/np_lattice.staple_rms); k: (V,) the oracle's smallest subgroup norm of
    this hit; `updated`: (V,) bool, the sites of this sub-step.  A hit computes U' = a(v) U with v = proj(U A), |v| = k:
        * its own rounding: at most the single-sub-step bar tol (north_star);
        * the staple sum inherits sqrt(sum B_nbr^2) (independent errors, every factor unitary), the old link its own B and
          moves v by at most |A| B_own <= 6 B_own (A is a sum of 6 unitary matrices); the normalisation v -> v/k passes a
          perturbation of v on with gain 1/k, and U itself enters U' once more directly:
              B' = tol + (rms_nbr + 6 B_own) / k + B_own."""
    out = B.copy()
    own = B[:, mu]
    new = tol + (rms_nbr + 6.0 * own) / np.where(updated, k, 1.0) + own
    out[updated, mu] = new[updated]
    return out
