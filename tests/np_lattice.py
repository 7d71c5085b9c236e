"""Independent numpy helpers for the tests (np.roll-based indexing; shares nothing with oracle/ or the CUDA path).

Used to pin conventions: lex order, direction order, plaquette orientation, Polyakov direction, gauge
transformations and lattice translations.  Canonical links: (V, D, N, N) complex, lex = x0 + L0*(x1 + ...).
"""
import numpy as np


def to_grid(links, dims):
    """(V, D, N, N) -> (L_{D-1}, ..., L_1, L_0, D, N, N): numpy axis a <-> lattice direction D-1-a."""
    D = len(dims)
    return links.reshape(tuple(reversed(dims)) + links.shape[1:])


def from_grid(grid, dims):
    V = int(np.prod(dims))
    return np.ascontiguousarray(grid.reshape((V,) + grid.shape[len(dims):]))


def shift(grid, dims, mu, step=1):
    """field at x + step*mu_hat, periodic: result[x] = grid[x + step*mu]"""
    D = len(dims)
    return np.roll(grid, -step, axis=D - 1 - mu)


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


def plaquettes(links, dims, field=None):
    """per-plane means of (1/N) Re Tr [F] U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+, order (0,1),(0,2),...;
    field = (mu, nu, theta) dresses that plane with F = diag(exp(i theta))."""
    D = len(dims)
    N = links.shape[-1]
    g = to_grid(links, dims)
    out = []
    for mu in range(D):
        for nu in range(mu + 1, D):
            Um, Un = g[..., mu, :, :], g[..., nu, :, :]
            P = Um @ shift(Un, dims, mu) @ dag(shift(Um, dims, nu)) @ dag(Un)
            if field is not None and field[0] == mu and field[1] == nu:
                F = np.diag(np.exp(1j * np.asarray(field[2][:N], dtype=float)))
                P = F @ P
            out.append(np.mean(np.trace(P, axis1=-2, axis2=-1).real) / N)
    return np.array(out)


def polyakov(links, dims):
    D = len(dims)
    N = links.shape[-1]
    g = to_grid(links, dims)[..., D - 1, :, :]          # axis 0 is time
    P = g[0]
    for t in range(1, dims[D - 1]):
        P = P @ g[t]
    return np.mean(np.trace(P, axis1=-2, axis2=-1)) / N


def gauge_transform(links, dims, omega):
    """U_mu(x) -> Omega(x) U_mu(x) Omega(x+mu)^+ ; omega: (V, N, N)"""
    D = len(dims)
    g = to_grid(links, dims).copy()
    og = omega.reshape(tuple(reversed(dims)) + omega.shape[1:])
    for mu in range(D):
        g[..., mu, :, :] = og @ g[..., mu, :, :] @ dag(shift(og, dims, mu))
    return from_grid(g, dims)


def translate(links, dims, mu):
    """configuration moved by one site along mu: U'(x) = U(x + mu_hat)"""
    return from_grid(shift(to_grid(links, dims), dims, mu), dims)


def unitarity_defect(links):
    N = links.shape[-1]
    uu = links @ dag(links) - np.eye(N)
    return float(np.max(np.abs(uu))), float(np.max(np.abs(np.linalg.det(links) - 1.0)))


def staple_dependents(mask, dims, mu):
    """Sites whose U_mu update reads a marked link.  mask: (V, D) bool of marked links; returns (V,) bool: True at x if the
    own link U_mu(x) or any of the 6(D-1) links of its staples -- U_nu(x), U_nu(x+mu), U_mu(x+nu), U_nu(x-nu), U_mu(x-nu),
    U_nu(x+mu-nu) for nu != mu -- is marked.  (Pure index bookkeeping: used to fence off the links a heatbath accept/reject
    disagreement can reach in later, un-resynced sub-steps.)"""
    D = len(dims)
    g = mask.reshape(tuple(reversed(dims)) + (D,))
    dep = g[..., mu].copy()
    for nu in range(D):
        if nu == mu:
            continue
        gn, gm = g[..., nu], g[..., mu]
        dep |= gn | shift(gn, dims, mu) | shift(gm, dims, nu)
        dep |= shift(gn, dims, nu, -1) | shift(gm, dims, nu, -1) | shift(shift(gn, dims, mu), dims, nu, -1)
    return dep.reshape(-1)


def site_parity(dims):
    """(V,) parity (sum of coordinates) & 1 in lex order"""
    V = int(np.prod(dims))
    return np.stack(np.unravel_index(np.arange(V), tuple(reversed(dims))), axis=-1).sum(axis=1) & 1


def staple_rms(B, dims, mu):
    """For every site x: sqrt of the sum of squares of B over the 6(D-1) links of the staples of U_mu(x) (same index
    bookkeeping as staple_dependents).  B: (V, D) float.  Used to carry per-link error BOUNDS through un-resynced sub-steps."""
    D = len(dims)
    g = (B * B).reshape(tuple(reversed(dims)) + (D,))
    acc = np.zeros(g.shape[:-1])
    for nu in range(D):
        if nu == mu:
            continue
        gn, gm = g[..., nu], g[..., mu]
        acc += gn + shift(gn, dims, mu) + shift(gm, dims, nu)
        acc += shift(gn, dims, nu, -1) + shift(gm, dims, nu, -1) + shift(shift(gn, dims, mu), dims, nu, -1)
    return np.sqrt(acc.reshape(-1))
