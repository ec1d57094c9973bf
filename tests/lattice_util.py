"""numpy helpers for the tests only (shifts, gauge transforms, per-link norms).

np.roll based and independent of both the oracle's and the CUDA path's indexing code.
Canonical layout: fields are [V, ...] with s = x + Lx*(y + Ly*(z + Lz*t)); reshaped to
[Lt, Lz, Ly, Lx, ...] the direction mu lives on numpy axis 3 - mu.
"""
import numpy as np
from scipy.linalg import expm as scipy_expm


def grid(field, dims):
    Lx, Ly, Lz, Lt = dims
    return field.reshape((Lt, Lz, Ly, Lx) + field.shape[1:])


def flat(field, dims):
    V = int(np.prod(dims))
    return field.reshape((V,) + field.shape[4:])


def shift(field, dims, mu, d=+1):
    """Returns f'(x) = f(x + d*mu_hat) (periodic)."""
    g = grid(field, dims)
    return flat(np.roll(g, -d, axis=3 - mu), dims)


def coord(dims, mu):
    """Coordinate x_mu of every site, shape [V]."""
    Lx, Ly, Lz, Lt = dims
    idx = np.arange(Lx * Ly * Lz * Lt)
    c = [idx % Lx, (idx // Lx) % Ly, (idx // (Lx * Ly)) % Lz, idx // (Lx * Ly * Lz)]
    return c[mu]


def dagger(M):
    return M.conj().swapaxes(-1, -2)


def random_su3(n, rng):
    G = rng.standard_normal((n, 3, 3)) + 1j * rng.standard_normal((n, 3, 3))
    H = 0.5 * (G + dagger(G))
    w, v = np.linalg.eigh(H)
    g = (v * np.exp(1j * w)[:, None, :]) @ dagger(v)
    return g / np.linalg.det(g)[:, None, None] ** (1.0 / 3.0)


def gauge_transform_links(U, g, dims):
    """U_mu(x) -> g(x) U_mu(x) g^dag(x+mu)."""
    out = np.empty_like(U)
    for mu in range(4):
        out[:, mu] = g @ U[:, mu] @ dagger(shift(g, dims, mu))
    return out


def gauge_transform_spinor(psi, g):
    """psi(x) -> g(x) psi(x) acting on colour."""
    return np.einsum("sab,sib->sia", g, psi)


def link_rel_err(F, F_ref):
    """Eq. 8 of the paper per link, with the floor of DESIGN.md reading A-16.
    Returns (eps_floored_max, eps_plain_max)."""
    d = np.sqrt(np.sum(np.abs(F - F_ref) ** 2, axis=(-1, -2)))
    n = np.sqrt(np.sum(np.abs(F_ref) ** 2, axis=(-1, -2)))
    rms = np.sqrt(np.mean(n ** 2))
    floored = d / np.maximum(n, 1e-3 * rms) if rms > 0 else d
    with np.errstate(divide="ignore", invalid="ignore"):
        plain = np.where(n > 0, d / n, 0.0)
    return float(floored.max()), float(plain.max())


def link_rel_quantiles(F, F_ref, qs=(0.5, 0.9, 0.99, 0.999, 1.0)):
    """The distribution behind the paper's Fig. 2: plain Eq. 8 over all links, no floor, at the
    cumulative fractions qs."""
    d = np.sqrt(np.sum(np.abs(F - F_ref) ** 2, axis=(-1, -2))).ravel()
    n = np.sqrt(np.sum(np.abs(F_ref) ** 2, axis=(-1, -2))).ravel()
    assert (n > 0).all()
    return [float(v) for v in np.quantile(d / n, qs)]


def numpy_dslash(U, psi, dims, kappa, bc, gam, dag=False):
    """Second, vectorised statement of the Wilson-Dirac operator of BASELINE.json configs[0]
    (np.roll shifts, einsum products); used to cross-check the oracle's indexing."""
    sg = -1.0 if dag else 1.0
    out = psi.copy()
    for mu in range(4):
        sign = np.where(coord(dims, mu) == dims[mu] - 1, float(bc[mu]), 1.0)
        Us = U[:, mu] * sign[:, None, None]
        fw = np.einsum("sab,sib->sia", Us, shift(psi, dims, mu, +1))
        fw = fw - sg * np.einsum("ij,sja->sia", gam[mu], fw)
        bwU = shift(Us, dims, mu, -1)
        bw = np.einsum("sba,sib->sia", bwU.conj(), shift(psi, dims, mu, -1))
        bw = bw + sg * np.einsum("ij,sja->sia", gam[mu], bw)
        out -= kappa * (fw + bw)
    return out


__all__ = [n for n in dir() if not n.startswith("_")]
