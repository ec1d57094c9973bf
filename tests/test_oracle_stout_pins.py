"""Pins for the stout-smearing oracle (oracle/stout.py), no GPU.

T1  the smeared fermion force is the derivative of the smeared action: Richardson central differences along every
    generator on sampled links (incl. one crossing the antiperiodic boundary), one and two levels, rho = 0.3
T2  Phi_{-A} (differential of exp, adjoint) against the block-triangular exponential of scipy's expm
T3  the smearing is gauge covariant, rho = 0 is the identity, the unit field is a fixed point, smeared links are
    SU(3) and smoother (plaquette goes up)
T4  W's force (plaquette loops with one insertion of G) against a finite difference of the pinned gauge force
    along G, and its pieces: linear in G, zero for G = 0
T5  the ref. [6] form U' = exp(iQ) U, Q from Omega = C U^dag with C = rho * (sum of staples), written out with np.roll
"""
import numpy as np
from scipy.linalg import expm as scipy_expm

import oracle
from oracle import stout
from paper_2602_20516_b200 import synth
from lattice_util import dagger, gauge_transform_links, link_rel_err, random_su3, shift

DIMS = (4, 4, 4, 4)
BC = (1, 1, 1, -1)
RHO = 0.3
TAU = [oracle.generator(a) for a in range(8)]


def _fd(action, U, s, mu, a, t):
    def cd(h):
        Up, Um = U.copy(), U.copy()
        Up[s, mu] = scipy_expm(h * TAU[a]) @ U[s, mu]
        Um[s, mu] = scipy_expm(-h * TAU[a]) @ U[s, mu]
        return (action(Up) - action(Um)) / (2 * h)
    return (4 * cd(t) - cd(2 * t)) / 3


def test_T1_smeared_force_is_derivative_of_smeared_action():
    dims, kappa = DIMS, 0.11
    U = synth.warm_links(dims, 0.25, 2001)
    eta = synth.gaussian_spinor(dims, 2002)
    V = U.shape[0]
    for n, sites in ((1, [(0, 0), (V - 1, 3), (77, 1), (130, 2)]), (2, [(5, 2), (V - 3, 3)])):
        Un = stout.smear_levels(dims, RHO, n, U)[0][-1]
        phi = oracle.dslash(dims, kappa, BC, Un, eta, dagger=True)
        F, it, ok = stout.fermion_force(dims, kappa, BC, U, phi, n, RHO, 1e-14, 5000)
        assert ok
        act = lambda W: stout.fermion_action(dims, kappa, BC, W, phi, n, RHO, 1e-14, 5000)[0]
        worst = 0.0
        for s, mu in sites:
            for a in range(8):
                fd = _fd(act, U, s, mu, a, 2e-3)
                an = (-2 * np.trace(TAU[a] @ F[s, mu])).real
                worst = max(worst, abs(fd - an))
        assert worst < 2e-8 * np.abs(F).max(), (n, worst)
        # the result is an su(3) field and differs from the unsmeared force
        assert np.abs(F + dagger(F)).max() < 1e-13 and np.abs(np.trace(F, axis1=-2, axis2=-1)).max() < 1e-13


def test_T2_phi_minus_against_block_exponential():
    rng = np.random.default_rng(5)
    for scale in (1e-3, 0.3, 1.5):
        A = scale * synth.gaussian_momenta((2, 2, 2, 2), 9).reshape(-1, 3, 3)[:12]
        F = synth.gaussian_momenta((2, 2, 2, 2), 10).reshape(-1, 3, 3)[:12]
        G = stout.phi_minus(A, F)
        for i in range(12):
            # exp([[X, E], [0, X]]) = [[e^X, dexp_X(E)], [0, e^X]], dexp_X(E) e^-X = Phi_X(E); here X = -A
            blk = np.zeros((6, 6), complex)
            blk[:3, :3] = blk[3:, 3:] = -A[i]
            blk[:3, 3:] = F[i]
            ex = scipy_expm(blk)
            ref = ex[:3, 3:] @ scipy_expm(A[i])
            assert np.abs(G[i] - ref).max() < 1e-13 * max(1.0, np.abs(ref).max())
        # adjointness used in the derivation: tr[Phi_A(X) F] = tr[X Phi_{-A}(F)]
        X = synth.gaussian_momenta((2, 2, 2, 2), 11).reshape(-1, 3, 3)[:12]
        lhs = np.trace(stout.phi_minus(-A, X) @ F, axis1=-2, axis2=-1)
        rhs = np.trace(X @ G, axis1=-2, axis2=-1)
        assert np.abs(lhs - rhs).max() < 1e-12


def test_T3_smearing_properties():
    dims = (4, 2, 6, 4)
    U = synth.warm_links(dims, 0.3, 31)
    U1, A = stout.smear(dims, RHO, U)
    # SU(3), exponent in su(3)
    assert np.abs(U1 @ dagger(U1) - np.eye(3)).max() < 1e-13 and np.abs(np.linalg.det(U1) - 1).max() < 1e-13
    assert np.abs(A + dagger(A)).max() < 1e-14
    # covariance
    g = random_su3(U.shape[0], np.random.default_rng(3))
    U1g, _ = stout.smear(dims, RHO, gauge_transform_links(U, g, dims))
    assert np.abs(U1g - gauge_transform_links(U1, g, dims)).max() < 1e-13
    # rho = 0, unit field
    assert np.array_equal(stout.smear(dims, 0.0, U)[0], U) or np.abs(stout.smear(dims, 0.0, U)[0] - U).max() < 1e-15
    one = synth.unit_links(dims)
    assert np.abs(stout.smear(dims, RHO, one)[0] - one).max() < 1e-15
    # smoothing (rho = 0.1 is inside the perturbatively safe range; 0.3 on this rough field still raises it)
    p0 = oracle.gauge_action(dims, 1.0, U)[1]
    assert oracle.gauge_action(dims, 1.0, stout.smear(dims, 0.1, U)[0])[1] > p0
    assert oracle.gauge_action(dims, 1.0, stout.smear_levels(dims, 0.1, 3, U)[0][-1])[1] > p0 + 0.05


def test_T4_w_force_is_the_hessian_of_the_plaquette_sum():
    dims = DIMS
    U = synth.warm_links(dims, 0.3, 41)
    G = synth.gaussian_momenta(dims, 42)
    FW = stout.w_force(dims, RHO, U, G)
    assert np.abs(FW + dagger(FW)).max() < 1e-13
    assert np.abs(stout.w_force(dims, RHO, U, 0 * G)).max() == 0.0
    assert np.abs(stout.w_force(dims, RHO, U, 2.5 * G) - 2.5 * FW).max() < 1e-12
    # W[U] = 2 rho sum Re tr[U V G] = 2 rho sum tr[P_su(3)(U V) G] = (12 rho / beta) sum tr[F^g G]; its derivative along
    # tau^a at one link by central differences of the pinned gauge force
    W = lambda X: 2.0 * RHO * np.sum(np.trace(oracle.gauge_force(dims, 6.0, X) @ G, axis1=-2, axis2=-1)).real
    V = U.shape[0]
    worst = 0.0
    for s, mu in [(0, 0), (V - 1, 3), (100, 2)]:
        for a in range(8):
            fd = _fd(W, U, s, mu, a, 2e-3)
            worst = max(worst, abs(fd - (-2 * np.trace(TAU[a] @ FW[s, mu])).real))
    assert worst < 2e-9 * np.abs(FW).max(), worst


def test_T5_reference_form_of_the_smearing():
    dims = (4, 3, 2, 6)
    U = synth.warm_links(dims, 0.3, 55)
    U1, _ = stout.smear(dims, RHO, U)
    for mu in range(4):
        C = np.zeros_like(U[:, mu])
        for nu in range(4):
            if nu == mu:
                continue
            Un, Um = U[:, nu], U[:, mu]
            C += Un @ shift(Um, dims, nu) @ dagger(shift(Un, dims, mu))
            C += dagger(shift(Un, dims, nu, -1)) @ shift(Um, dims, nu, -1) @ shift(shift(Un, dims, nu, -1), dims, mu)
        Om = RHO * C @ dagger(U[:, mu])
        Q = 0.5j * (dagger(Om) - Om)
        Q -= (np.trace(Q, axis1=-2, axis2=-1) / 3.0)[:, None, None] * np.eye(3)
        ref = np.array([scipy_expm(1j * q) for q in Q]) @ U[:, mu]
        assert np.abs(U1[:, mu] - ref).max() < 1e-13
