"""Seeded synthetic input fields (BASELINE.json configs).

This module only MAKES inputs: random links, momenta and spinors in the canonical
layout (numpy complex128, site index s = x + Lx*(y + Ly*(z + Lz*t))).  It holds none
of the method's arithmetic (no Dirac operator, force, projector or link update) and is
the one module both the CUDA path's callers and the oracle's callers may share.
The same arrays are handed to both sides, so nothing depends on reproducing an RNG
on the device.  Stand-in for the paper's own (unavailable) 16^4 / 24^4 SU(3)
configurations.
"""
import numpy as np

# Workloads of BASELINE.json configs[0..4] with the seeds SURVEY.md section 8(d) assigns.
CONFIGS = {
    0: dict(dims=(4, 4, 4, 4), links="warm", eps=0.2, beta=5.5, kappa=0.10, bc=(1, 1, 1, -1),
            seed_links=1001, seed_eta=1002, cg_tol=1e-14),
    1: dict(dims=(8, 8, 8, 8), links="haar", beta=6.0, kappa=0.0, bc=(1, 1, 1, 1),
            seed_links=1101, seed_mom=1102, nsteps=50, dt=0.02),
    2: dict(dims=(16, 16, 16, 16), links="warm", eps=0.3, beta=0.0, kappa=0.12, bc=(1, 1, 1, -1),
            seed_links=1201, seed_eta=1202, cg_tol=1e-12),
    3: dict(dims=(32, 32, 32, 32), links="warm", eps=0.3, beta=5.6, kappa=0.12, bc=(1, 1, 1, -1),
            seed_links=1301, seed_mom=1302, seed_eta=1303, cg_tol=1e-12, dt=0.01),
    4: dict(dims=(48, 48, 48, 96), links="warm", eps=0.3, beta=5.6, kappa=0.12, bc=(1, 1, 1, -1),
            seed_links=1401, seed_eta=1402, cg_tol=1e-10),
}

_CHUNK = 1 << 18  # matrices per batch, bounds host memory at 32^4 and 48^3x96


def volume(dims):
    return int(np.prod([int(d) for d in dims]))


def gell_mann():
    """lambda^a, a = 0..7, shape [8,3,3]."""
    lam = np.zeros((8, 3, 3), np.complex128)
    lam[0, 0, 1] = lam[0, 1, 0] = 1
    lam[1, 0, 1], lam[1, 1, 0] = -1j, 1j
    lam[2, 0, 0], lam[2, 1, 1] = 1, -1
    lam[3, 0, 2] = lam[3, 2, 0] = 1
    lam[4, 0, 2], lam[4, 2, 0] = -1j, 1j
    lam[5, 1, 2] = lam[5, 2, 1] = 1
    lam[6, 1, 2], lam[6, 2, 1] = -1j, 1j
    lam[7] = np.diag([1, 1, -2]) / np.sqrt(3.0)
    return lam


def _complex_gaussian(rng, shape):
    g = rng.standard_normal(tuple(shape) + (2,))
    return g[..., 0] + 1j * g[..., 1]


def warm_links(dims, eps, seed):
    """U = exp(i eps H), H = traceless Hermitian part of a complex Gaussian matrix
    (entries a + ib with a, b ~ N(0,1)); reading A-17.  Shape [V,4,3,3]."""
    V = volume(dims)
    rng = np.random.default_rng(seed)
    U = np.empty((V * 4, 3, 3), np.complex128)
    eye = np.eye(3)
    for lo in range(0, V * 4, _CHUNK):
        hi = min(V * 4, lo + _CHUNK)
        G = _complex_gaussian(rng, (hi - lo, 3, 3))
        H = 0.5 * (G + G.conj().swapaxes(-1, -2))
        H -= (np.trace(H, axis1=-2, axis2=-1) / 3.0)[:, None, None] * eye
        w, v = np.linalg.eigh(H)  # H = v diag(w) v^dag
        U[lo:hi] = (v * np.exp(1j * eps * w)[:, None, :]) @ v.conj().swapaxes(-1, -2)
    return U.reshape(V, 4, 3, 3)


def haar_links(dims, seed):
    """Haar-random SU(3): complex Gaussian 3x3, Gram-Schmidt on the rows in order, third
    row times conj(det) so that det = 1; reading A-18.  Shape [V,4,3,3]."""
    V = volume(dims)
    rng = np.random.default_rng(seed)
    U = np.empty((V * 4, 3, 3), np.complex128)
    for lo in range(0, V * 4, _CHUNK):
        hi = min(V * 4, lo + _CHUNK)
        G = _complex_gaussian(rng, (hi - lo, 3, 3))
        r0 = G[:, 0]
        r0 = r0 / np.linalg.norm(r0, axis=-1, keepdims=True)
        r1 = G[:, 1] - np.sum(r0.conj() * G[:, 1], axis=-1, keepdims=True) * r0
        r1 = r1 / np.linalg.norm(r1, axis=-1, keepdims=True)
        r2 = G[:, 2] - np.sum(r0.conj() * G[:, 2], axis=-1, keepdims=True) * r0
        r2 = r2 - np.sum(r1.conj() * r2, axis=-1, keepdims=True) * r1
        r2 = r2 / np.linalg.norm(r2, axis=-1, keepdims=True)
        Q = np.stack([r0, r1, r2], axis=1)
        Q[:, 2] *= np.linalg.det(Q).conj()[:, None]
        U[lo:hi] = Q
    return U.reshape(V, 4, 3, 3)


def unit_links(dims):
    V = volume(dims)
    U = np.zeros((V, 4, 3, 3), np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1.0
    return U


def gaussian_momenta(dims, seed):
    """Pi = sum_a pi^a tau^a, tau^a = i lambda^a/2, pi^a ~ N(0,1) (reading A-14):
    traceless anti-Hermitian, shape [V,4,3,3]."""
    V = volume(dims)
    rng = np.random.default_rng(seed)
    pi = rng.standard_normal((V * 4, 8))
    tau = 0.5j * gell_mann()
    return np.einsum("na,aij->nij", pi, tau).reshape(V, 4, 3, 3)


def gaussian_spinor(dims, seed):
    """Unit complex Gaussian: Re, Im ~ N(0, 1/2), so E|eta|^2 = 1 per component
    (reading A-9); 12 complex = 24 real numbers per site (reading A-8).  Shape [V,4,3]."""
    V = volume(dims)
    rng = np.random.default_rng(seed)
    return _complex_gaussian(rng, (V, 4, 3)) * np.sqrt(0.5)


def config_links(cfg):
    c = CONFIGS[cfg] if isinstance(cfg, int) else cfg
    if c["links"] == "warm":
        return warm_links(c["dims"], c["eps"], c["seed_links"])
    if c["links"] == "haar":
        return haar_links(c["dims"], c["seed_links"])
    raise ValueError(c["links"])
