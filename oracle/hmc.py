"""CPU oracle for the HMC layer around the MD step -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

SURVEY.md 8(f)2: momentum and pseudofermion heat baths, Metropolis accept/reject, and the integrators the paper
names (second-order leapfrog PAPER.md:152; "Sexton-Weingarten" with inner gauge steps and the multi-time-scale
set-up of PAPER.md:154, 164) plus the Omelyan second-order minimum-norm scheme.  Only tests/ may import this module.
It shares no code with paper_2602_20516_b200: plain numpy on top of the pinned oracle functions
(oracle.kick / oracle.drift / oracle.hamiltonian / oracle.dslash).

Random numbers (reading A-25).  Both sides implement the same counter-based generator, Philox4x32-10
(Salmon, Moraes, Dror, Shaw, SC'11), so that a heat bath is a pure function of (seed, trajectory, element):
    key     = (seed mod 2^32, seed div 2^32)
    counter = (element index, draw index j, stream, trajectory)        stream 1 = momenta, 2 = pseudofermion, 3 = Metropolis
    output words x0..x3  ->  u1 = ((x0 + 2^32 x1) div 2^11 + 1/2) 2^-53,  u2 likewise from (x2, x3)   (both in (0,1))
    Box-Muller: g0 = sqrt(-2 ln u1) cos(2 pi u2),  g1 = sqrt(-2 ln u1) sin(2 pi u2)
  momenta:       element = link 4 s + mu, j = 0..3, (g0, g1) = (pi^(2j+1), pi^(2j+2)),  Pi = sum_a pi^a tau^a,
                 tau^a = i lambda^a / 2  (reading A-14: pi^a ~ N(0,1), weight exp(-K), K = sum ||Pi||_F^2 = sum (pi^a)^2 / 2)
  pseudofermion: element = site s, j = 0..11 = component 3 alpha + a, eta = (g0 + i g1) / sqrt 2  (weight exp(-eta^dag eta)),
                 phi = D^dag eta  (S_F = phi^dag (D^dag D)^-1 phi = eta^dag eta at the start of a trajectory)
  Metropolis:    element 0, j = 0, u = u1; accept iff u < exp(-dH).

Pins (tests/test_oracle_hmc_pins.py): the three published known-answer vectors of Philox4x32-10; moments of the
heat-bath fields and K / dof; integrators: Omelyan with lambda = 1/4 equals two leapfrog steps of dt/2, Sexton-Weingarten
on a gauge-only action equals leapfrog with m n steps of dt/m, both are reversible and have |dH| ~ dt^2; Metropolis
restores the links on rejection.
"""
import numpy as np

import oracle

OMELYAN_LAMBDA = 0.1931833275037836  # minimum-norm value of the second-order scheme (Omelyan, Mryglod, Folk 2003)
STREAM_MOMENTA, STREAM_PSEUDOFERMION, STREAM_METROPOLIS = 1, 2, 3

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = np.uint64(0x9E3779B9), np.uint64(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox4x32 with 10 rounds.  Counter words: arrays (or scalars) of values < 2^32; key words: scalars.
    Returns the four output words as uint64 arrays holding 32-bit values."""
    c = [np.atleast_1d(np.asarray(v, dtype=np.uint64)) & _MASK for v in (c0, c1, c2, c3)]
    c = list(np.broadcast_arrays(*c))
    k0, k1 = np.uint64(int(k0) & 0xFFFFFFFF), np.uint64(int(k1) & 0xFFFFFFFF)
    for _ in range(10):
        p0 = _M0 * c[0]  # 64-bit products of 32-bit values: no overflow
        p1 = _M1 * c[2]
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c = [hi1 ^ c[1] ^ k0, lo1, hi0 ^ c[3] ^ k1, lo0]
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c


def _uniforms(x):
    a = (x[1] << _S32) | x[0]
    b = (x[3] << _S32) | x[2]
    two53 = 2.0 ** -53
    u1 = ((a >> np.uint64(11)).astype(np.float64) + 0.5) * two53
    u2 = ((b >> np.uint64(11)).astype(np.float64) + 0.5) * two53
    return u1, u2


def gaussian_pairs(seed, trajectory, stream, element, j):
    """Two independent N(0,1) numbers per (element, j) of the given stream."""
    x = philox4x32_10(element, j, stream, trajectory, int(seed) & 0xFFFFFFFF, int(seed) >> 32)
    u1, u2 = _uniforms(x)
    r = np.sqrt(-2.0 * np.log(u1))
    return r * np.cos(2.0 * np.pi * u2), r * np.sin(2.0 * np.pi * u2)


def _gell_mann():
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


def momentum_heatbath(dims, seed, trajectory):
    """Pi[V,4,3,3] = sum_a pi^a tau^a with pi^a ~ N(0,1) from stream 1; also returns pi[V*4, 8]."""
    V = int(np.prod(dims))
    link = np.arange(4 * V, dtype=np.uint64)[:, None]
    j = np.arange(4, dtype=np.uint64)[None, :]
    g0, g1 = gaussian_pairs(seed, trajectory, STREAM_MOMENTA, link, j)
    pi = np.empty((4 * V, 8))
    pi[:, 0::2] = g0
    pi[:, 1::2] = g1
    tau = 0.5j * _gell_mann()
    return np.einsum("na,aij->nij", pi, tau).reshape(V, 4, 3, 3), pi


def pseudofermion_noise(dims, seed, trajectory):
    """eta[V,4,3], Re and Im ~ N(0, 1/2), from stream 2."""
    V = int(np.prod(dims))
    site = np.arange(V, dtype=np.uint64)[:, None]
    j = np.arange(12, dtype=np.uint64)[None, :]
    g0, g1 = gaussian_pairs(seed, trajectory, STREAM_PSEUDOFERMION, site, j)
    return ((g0 + 1j * g1) * np.sqrt(0.5)).reshape(V, 4, 3)


def metropolis_uniform(seed, trajectory):
    x = philox4x32_10(0, 0, STREAM_METROPOLIS, trajectory, int(seed) & 0xFFFFFFFF, int(seed) >> 32)
    return float(_uniforms(x)[0][0])


# ---------------------------------------------------------------------------------------------- integrators
LEAPFROG, OMELYAN, SEXTON_WEINGARTEN = 0, 1, 2


def integrate(dims, beta, kappa, bc, U, phi, P, nsteps, dt, integrator=LEAPFROG, n_inner=1, lam=OMELYAN_LAMBDA,
              tol=1e-12, max_iter=100000):
    """MD trajectory of nsteps steps of size dt (U <- exp(eps Pi) U, Pi <- Pi - eps F), adjacent
    kicks merged.  Returns (U, P, cg_iters).
      LEAPFROG:           K(dt/2) {D(dt) K(dt)}^(n-1) D(dt) K(dt/2)
      OMELYAN:            per step K(lam dt) D(dt/2) K((1 - 2 lam) dt) D(dt/2) K(lam dt)
      SEXTON_WEINGARTEN:  per step Kf(dt/2) I(dt) Kf(dt/2), fermion force outside, and inside the gauge leapfrog
                          I(dt) = Kg(h/2) {D(h) Kg(h)}^(m-1) D(h) Kg(h/2), h = dt / m, m = n_inner
    K = kick with both forces, Kg / Kf = gauge / fermion part only, D = link drift."""
    fermions = phi is not None and kappa != 0.0
    its = [0]

    def K(U, P, eps, b=beta, k=kappa):
        P, it, ok = oracle.kick(dims, b, k, bc, U, phi if (fermions and k != 0.0) else None, P, eps, tol, max_iter)
        assert ok
        its[0] += it
        return P

    def D(U, P, eps):
        return oracle.drift(dims, eps, P, U)

    if nsteps <= 0:
        return U.copy(), P.copy(), 0
    if integrator == LEAPFROG:
        P = K(U, P, 0.5 * dt)
        for n in range(nsteps):
            U = D(U, P, dt)
            P = K(U, P, 0.5 * dt if n == nsteps - 1 else dt)
    elif integrator == OMELYAN:
        P = K(U, P, lam * dt)
        for n in range(nsteps):
            U = D(U, P, 0.5 * dt)
            P = K(U, P, (1.0 - 2.0 * lam) * dt)
            U = D(U, P, 0.5 * dt)
            P = K(U, P, lam * dt if n == nsteps - 1 else 2.0 * lam * dt)
    elif integrator == SEXTON_WEINGARTEN:
        m = int(n_inner)
        h = dt / m
        if fermions:
            P = K(U, P, 0.5 * dt, b=0.0)
        for n in range(nsteps):
            P = K(U, P, 0.5 * h, k=0.0)
            for i in range(m):
                U = D(U, P, h)
                P = K(U, P, 0.5 * h if i == m - 1 else h, k=0.0)
            if fermions:
                P = K(U, P, 0.5 * dt if n == nsteps - 1 else dt, b=0.0)
    else:
        raise ValueError("unknown integrator")
    return U, P, its[0]


def hmc_trajectory(dims, beta, kappa, bc, U, seed, trajectory, nsteps, dt, integrator=LEAPFROG, n_inner=1,
                   tol=1e-12, max_iter=100000):
    """One HMC trajectory: heat baths, MD integration, Metropolis test with u < exp(-dH).
    Returns dict(U=links after the test, accepted, dH, H0, H1, P0, eta, phi, U_proposed, u, cg_iters)."""
    P0, _ = momentum_heatbath(dims, seed, trajectory)
    eta = phi = None
    SF0 = 0.0
    if kappa != 0.0:
        eta = pseudofermion_noise(dims, seed, trajectory)
        phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
        SF0 = float(np.sum(np.abs(eta) ** 2))  # = phi^dag (D^dag D)^-1 phi exactly
    K0 = oracle.kinetic(dims, P0)
    Sg0, _ = oracle.gauge_action(dims, beta, U)
    H0 = K0 + Sg0 + SF0
    U1, P1, its = integrate(dims, beta, kappa, bc, U, phi, P0, nsteps, dt, integrator, n_inner, OMELYAN_LAMBDA, tol, max_iter)
    H1 = oracle.hamiltonian(dims, beta, kappa, bc, U1, phi, P1, tol, max_iter)[0]
    dH = H1 - H0
    u = metropolis_uniform(seed, trajectory)
    accepted = bool(u < np.exp(-dH))
    return dict(U=U1 if accepted else U.copy(), accepted=accepted, dH=dH, H0=H0, H1=H1, P0=P0, eta=eta, phi=phi,
                U_proposed=U1, u=u, cg_iters=its)
