"""Seeded synthetic input generators shared by the oracle-side and the CUDA-side tests.

Holds none of the method's arithmetic (no staples, no heatbath, no Philox): only random SU(N) link
configurations drawn with numpy's PCG64, in the canonical layout (V, D, N, N) complex128,
lex = x0 + L0*(x1 + L1*(x2 + L2*x3)).
"""
import numpy as np


def random_sun(rng, n_mats, N):
    """n_mats Haar-distributed SU(N) matrices (QR of complex Ginibre, phases fixed, det -> 1)."""
    z = rng.standard_normal((n_mats, N, N)) + 1j * rng.standard_normal((n_mats, N, N))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=1, axis2=2)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    q = q * (det ** (-1.0 / N))[:, None, None]
    return q


def random_links(dims, N, seed, spread=None):
    """Random SU(N) configuration.  spread=None: Haar.  spread=s: exp(i s H) near the identity
    (H random Hermitian traceless), which mimics a thermalised large-beta configuration."""
    rng = np.random.Generator(np.random.PCG64(seed))
    V, D = int(np.prod(dims)), len(dims)
    if spread is None:
        u = random_sun(rng, V * D, N)
    else:
        h = rng.standard_normal((V * D, N, N)) + 1j * rng.standard_normal((V * D, N, N))
        h = 0.5 * (h + np.conj(np.swapaxes(h, 1, 2)))
        h = h - (np.trace(h, axis1=1, axis2=2) / N)[:, None, None] * np.eye(N)
        w, v = np.linalg.eigh(h)
        u = (v * np.exp(1j * spread * w)[:, None, :]) @ np.conj(np.swapaxes(v, 1, 2))
    if N == 2:
        # exact quaternion form [[a, b], [-conj(b), conj(a)]] so that the 4-real SU(2) storage round-trips bit for bit
        u[:, 1, 0] = -np.conj(u[:, 0, 1])
        u[:, 1, 1] = np.conj(u[:, 0, 0])
    return np.ascontiguousarray(u.reshape(V, D, N, N))


def round_to_fp32(links):
    """Round a complex128 configuration to fp32-representable values (still complex128)."""
    return links.astype(np.complex64).astype(np.complex128)
