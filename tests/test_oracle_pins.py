"""Pins for the CPU oracle (no GPU): what the paper and the physics fix, not the oracle itself.

P1  unit gauge: plaquette 1, S_g 0, zero gauge force (also on a pure-gauge field)
P2  free-field spectrum of D and D^dag D on plane waves; CG converges in one step
P3  gamma5-hermiticity and <a, D b> = <D^dag a, b>
P4  gauge covariance / invariance of D, S_g, S_F and both forces
P5  force = central finite difference of the action along U -> exp(t tau^a) U
P6  phi = D^dag eta  =>  S_F = |eta|^2 and Y = D X = eta
P7  leapfrog |dH| ~ dt^2 and exact reversibility
P8  matrix exponential: library routine, closed form, unitarity
P9  the paper's own route: G from real-component differences, F = -1/2 TA(U G^dag)
P10 su(3) projector properties
P11 half-spinor outer-product identity that licenses the fused force kernel
plus: Clifford algebra of the gamma table, generator normalisation, dense solve vs CG,
a second (np.roll) statement of D, and the input generators' group properties.
"""
import numpy as np
import pytest
from scipy.linalg import expm as scipy_expm

import oracle
from paper_2602_20516_b200 import synth
from lattice_util import (coord, dagger, gauge_transform_links, gauge_transform_spinor,
                          link_rel_err, numpy_dslash, random_su3, shift)

DIMS = (4, 4, 4, 4)
ODD = (4, 3, 5, 6)
BC = (1, 1, 1, -1)
GAM = [oracle.gamma(m) for m in range(5)]
TAU = [oracle.generator(a) for a in range(8)]


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ---------------------------------------------------------------- tables
def test_gamma_table_is_chiral_clifford():
    for m in range(4):
        assert np.array_equal(GAM[m], dagger(GAM[m]))
        for n in range(4):
            assert np.array_equal(GAM[m] @ GAM[n] + GAM[n] @ GAM[m], 2.0 * (m == n) * np.eye(4))
        # chiral basis: gamma_mu is block off-diagonal
        assert not GAM[m][:2, :2].any() and not GAM[m][2:, 2:].any()
    assert np.array_equal(GAM[4], np.diag([1, 1, -1, -1]).astype(complex))
    assert np.array_equal(GAM[3][:2, 2:], np.eye(2))  # sigma_t = 1


def test_generators_normalised():
    lam = synth.gell_mann()
    for a in range(8):
        assert np.allclose(TAU[a], 0.5j * lam[a])
        assert abs(np.trace(TAU[a])) == 0
        assert np.allclose(TAU[a], -dagger(TAU[a]))
        for b in range(8):
            assert np.isclose(np.trace(TAU[a] @ TAU[b]), -0.5 * (a == b))


# ---------------------------------------------------------------- P10
def test_P10_projector():
    rng = np.random.default_rng(5)
    for _ in range(10):
        M = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
        A = oracle.ta(M)
        assert np.allclose(A, -dagger(A), atol=1e-16)
        assert abs(np.trace(A)) < 1e-15
        assert np.allclose(oracle.ta(A), A, atol=1e-16)  # idempotent
        assert np.allclose(oracle.ta(dagger(M)), -A, atol=1e-16)  # S2.24
        # components: A = sum_a tau^a (-2 tr(tau^a M_antiherm)) ; Re tr(tau M) = tr(tau TA(M))
        for a in range(8):
            assert np.isclose(np.trace(TAU[a] @ M).real, np.trace(TAU[a] @ A).real, atol=1e-14)
            assert abs(np.trace(TAU[a] @ A).imag) < 1e-15
    H = rng.standard_normal((3, 3))
    H = H + H.T  # Hermitian part is annihilated
    assert np.allclose(oracle.ta(H.astype(complex)), 0)
    assert np.allclose(oracle.ta(np.eye(3) * (2 + 3j)), 0)


# ---------------------------------------------------------------- P8
def test_P8_expm():
    rng = np.random.default_rng(6)
    for scale in [1e-8, 1e-3, 0.1, 1.0, 5.0, 30.0]:
        for _ in range(5):
            A = sum(rng.standard_normal() * t for t in TAU) * scale
            E = oracle.expm(A)
            assert np.allclose(E, scipy_expm(A), atol=2e-14 * max(1.0, scale))
            assert np.allclose(E @ dagger(E), np.eye(3), atol=1e-13 * max(1.0, scale))
            assert np.isclose(np.linalg.det(E), 1.0, atol=1e-13 * max(1.0, scale))
            assert np.allclose(E @ oracle.expm(-A), np.eye(3), atol=1e-13 * max(1.0, scale))
    d = np.array([0.3, -1.1, 0.8])
    assert np.allclose(oracle.expm(np.diag(1j * d)), np.diag(np.exp(1j * d)), atol=1e-15)
    # general (non anti-Hermitian) matrix against the library routine
    M = rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3))
    assert np.allclose(oracle.expm(M), scipy_expm(M), atol=1e-13)
    assert np.array_equal(oracle.expm(np.zeros((3, 3))), np.eye(3))


# ---------------------------------------------------------------- generators
def test_generators_make_group_elements():
    for U in (synth.warm_links(ODD, 0.3, 11), synth.haar_links(ODD, 12)):
        assert np.allclose(U @ dagger(U), np.eye(3), atol=1e-14)
        assert np.allclose(np.linalg.det(U), 1.0, atol=1e-14)
    P = synth.gaussian_momenta(DIMS, 13)
    assert np.allclose(P, -dagger(P)) and np.allclose(np.trace(P, axis1=-2, axis2=-1), 0)
    K = oracle.kinetic(DIMS, P)
    assert abs(K / (P.shape[0] * 4 * 8) - 0.5) < 0.02  # K = 1/2 sum (pi^a)^2
    pi = -2 * np.einsum("aij,sji->sa", np.array(TAU), P[:, 0])
    assert np.isclose(0.5 * np.sum(pi.real ** 2), np.sum(np.abs(P[:, 0]) ** 2))
    eta = synth.gaussian_spinor(DIMS, 14)
    assert abs(np.mean(np.abs(eta) ** 2) - 1.0) < 0.03
    _, plaq = oracle.gauge_action(DIMS, 1.0, synth.warm_links(DIMS, 0.2, 1001))
    assert 0.75 < plaq < 0.87  # SURVEY A-17: about 0.81 at eps = 0.2
    _, plaq = oracle.gauge_action(DIMS, 1.0, synth.haar_links(DIMS, 3))
    assert abs(plaq) < 0.05  # Haar measure: <tr U_P> = 0


# ---------------------------------------------------------------- P1
def test_P1_unit_and_pure_gauge():
    U = synth.unit_links(ODD)
    S, plaq = oracle.gauge_action(ODD, 5.5, U)
    assert S == 0.0 and plaq == 1.0
    assert not oracle.gauge_force(ODD, 5.5, U).any()
    g = random_su3(U.shape[0], np.random.default_rng(1))
    Ug = gauge_transform_links(U, g, ODD)
    S, plaq = oracle.gauge_action(ODD, 5.5, Ug)
    assert abs(S) < 1e-10 and abs(plaq - 1) < 1e-14
    assert np.abs(oracle.gauge_force(ODD, 5.5, Ug)).max() < 1e-13


# ---------------------------------------------------------------- P2
@pytest.mark.parametrize("n", [(0, 0, 0, 0), (1, 0, 0, 0), (0, 1, 0, 0), (0, 0, 2, 0), (0, 0, 0, 1), (1, 2, 3, 2)])
def test_P2_free_field_spectrum(n):
    dims, kappa = ODD, 0.11
    U = synth.unit_links(dims)
    p = [2 * np.pi * (n[m] + (0.5 if BC[m] < 0 else 0.0)) / dims[m] for m in range(4)]
    phase = np.exp(1j * sum(p[m] * coord(dims, m) for m in range(4)))
    rng = np.random.default_rng(2)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi = phase[:, None, None] * u[None]
    a = 1 - 2 * kappa * sum(np.cos(p))
    Mp = a * np.eye(4) + 2j * kappa * sum(np.sin(p[m]) * GAM[m] for m in range(4))
    lam = a ** 2 + 4 * kappa ** 2 * sum(np.sin(p) ** 2)
    D = oracle.dslash(dims, kappa, BC, U, psi)
    assert np.allclose(D, phase[:, None, None] * (Mp @ u)[None], atol=1e-14)
    Dd = oracle.dslash(dims, kappa, BC, U, psi, dagger=True)
    assert np.allclose(Dd, phase[:, None, None] * (dagger(Mp) @ u)[None], atol=1e-14)
    DdD = oracle.dslash(dims, kappa, BC, U, D, dagger=True)
    assert np.allclose(DdD, lam * psi, atol=1e-13)
    x, iters, rel, ok = oracle.cg(dims, kappa, BC, U, psi, 1e-12, 100)
    assert ok and iters == 1 and np.allclose(x, psi / lam, atol=1e-13)


# ---------------------------------------------------------------- P3, second statement of D
def test_P3_gamma5_hermiticity_and_adjoint():
    dims, kappa = ODD, 0.12
    U = synth.warm_links(dims, 0.3, 21)
    a = synth.gaussian_spinor(dims, 22)
    b = synth.gaussian_spinor(dims, 23)
    g5 = np.array([1, 1, -1, -1.0])[None, :, None]
    Db = oracle.dslash(dims, kappa, BC, U, b)
    Dda = oracle.dslash(dims, kappa, BC, U, a, dagger=True)
    assert abs(vdot(a, Db) - vdot(Dda, b)) < 1e-12 * abs(vdot(a, Db))
    assert np.array_equal(g5 * oracle.dslash(dims, kappa, BC, U, g5 * a), Dda)  # g5 D g5 = D^dag


@pytest.mark.parametrize("dag", [False, True])
def test_oracle_D_matches_numpy_roll_statement(dag):
    dims, kappa = ODD, 0.12
    U = synth.warm_links(dims, 0.3, 31)
    psi = synth.gaussian_spinor(dims, 32)
    bc = (1, -1, 1, -1)
    ref = numpy_dslash(U, psi, dims, kappa, bc, GAM, dag)
    assert np.allclose(oracle.dslash(dims, kappa, bc, U, psi, dagger=dag), ref, atol=1e-14)
    sites = np.array([0, 7, 100, 359])
    assert np.array_equal(oracle.dslash_sites(dims, kappa, bc, U, psi, sites, dagger=dag),
                          oracle.dslash(dims, kappa, bc, U, psi, dagger=dag)[sites])


# ---------------------------------------------------------------- P4
def test_P4_gauge_covariance():
    dims, kappa, beta = ODD, 0.12, 5.6
    U = synth.warm_links(dims, 0.3, 41)
    eta = synth.gaussian_spinor(dims, 42)
    psi = synth.gaussian_spinor(dims, 43)
    g = random_su3(U.shape[0], np.random.default_rng(44))  # periodic g respects the fermion bc
    Ug = gauge_transform_links(U, g, dims)
    # D[U^g] g psi = g D[U] psi
    lhs = oracle.dslash(dims, kappa, BC, Ug, gauge_transform_spinor(psi, g))
    rhs = gauge_transform_spinor(oracle.dslash(dims, kappa, BC, U, psi), g)
    assert np.allclose(lhs, rhs, atol=1e-13)
    # S_g invariant, F^g covariant
    assert np.isclose(oracle.gauge_action(dims, beta, Ug)[0], oracle.gauge_action(dims, beta, U)[0], rtol=1e-13)
    Fg, Fg_g = oracle.gauge_force(dims, beta, U), oracle.gauge_force(dims, beta, Ug)
    assert np.allclose(Fg_g, g[:, None] @ Fg @ dagger(g)[:, None], atol=1e-12)
    # S_F invariant, F^f covariant
    phi = oracle.dslash(dims, kappa, BC, U, eta, dagger=True)
    S, X, it, ok = oracle.fermion_action(dims, kappa, BC, U, phi, 1e-13, 2000)
    Sg_, Xg, itg, okg = oracle.fermion_action(dims, kappa, BC, Ug, gauge_transform_spinor(phi, g), 1e-13, 2000)
    assert ok and okg and np.isclose(S, Sg_, rtol=1e-12)
    Y = oracle.dslash(dims, kappa, BC, U, X)
    Yg = oracle.dslash(dims, kappa, BC, Ug, Xg)
    Ff, Ff_g = oracle.fermion_force(dims, kappa, BC, U, X, Y), oracle.fermion_force(dims, kappa, BC, Ug, Xg, Yg)
    assert np.allclose(Ff_g, g[:, None] @ Ff @ dagger(g)[:, None], atol=1e-11 * np.abs(Ff).max())


# ---------------------------------------------------------------- P5
def _fd(action, U, s, mu, a, t):
    """Richardson-extrapolated central difference of action along U_mu(s) -> exp(t tau^a) U_mu(s)."""
    def cd(h):
        Up, Um = U.copy(), U.copy()
        Up[s, mu] = scipy_expm(h * TAU[a]) @ U[s, mu]
        Um[s, mu] = scipy_expm(-h * TAU[a]) @ U[s, mu]
        return (action(Up) - action(Um)) / (2 * h)
    return (4 * cd(t) - cd(2 * t)) / 3


def test_P5_gauge_force_is_derivative_of_action():
    dims, beta = ODD, 5.5
    U = synth.warm_links(dims, 0.3, 51)
    F = oracle.gauge_force(dims, beta, U)
    V = U.shape[0]
    worst = 0.0
    for s, mu in [(0, 0), (3, 1), (V - 1, 3), (17, 2), (V // 2, 3), (V - 1, 0)]:
        assert np.array_equal(oracle.gauge_force_link(dims, beta, U, s, mu), F[s, mu])
        for a in range(8):
            fd = _fd(lambda W: oracle.gauge_action(dims, beta, W)[0], U, s, mu, a, 2e-3)
            an = (-2 * np.trace(TAU[a] @ F[s, mu])).real
            worst = max(worst, abs(fd - an))
    assert worst < 2e-9 * np.abs(F).max(), worst


def test_P5_fermion_force_is_derivative_of_action():
    dims, kappa = DIMS, 0.10
    U = synth.warm_links(dims, 0.2, 1001)
    eta = synth.gaussian_spinor(dims, 1002)
    phi = oracle.dslash(dims, kappa, BC, U, eta, dagger=True)
    S, X, it, ok = oracle.fermion_action(dims, kappa, BC, U, phi, 1e-14, 5000)
    assert ok
    Y = oracle.dslash(dims, kappa, BC, U, X)
    F = oracle.fermion_force(dims, kappa, BC, U, X, Y)
    V = U.shape[0]
    act = lambda W: oracle.fermion_action(dims, kappa, BC, W, phi, 1e-14, 5000)[0]
    worst = 0.0
    # (V-1, 3) and (V-64.., 3) cross the antiperiodic time boundary; (3, 0) crosses a periodic one
    for s, mu in [(0, 0), (3, 0), (V - 1, 3), (V - 20, 3), (77, 1), (130, 2)]:
        assert np.array_equal(oracle.fermion_force_link(dims, kappa, BC, U, X, Y, s, mu), F[s, mu])
        for a in range(8):
            fd = _fd(act, U, s, mu, a, 2e-3)
            an = (-2 * np.trace(TAU[a] @ F[s, mu])).real
            worst = max(worst, abs(fd - an))
    assert worst < 1e-8 * np.abs(F).max(), worst


# ---------------------------------------------------------------- P6 and the solver
def test_P6_phi_from_eta_closed_form():
    c = synth.CONFIGS[0]
    dims, kappa = c["dims"], c["kappa"]
    U = synth.config_links(0)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, c["bc"], U, eta, dagger=True)
    S, X, iters, ok = oracle.fermion_action(dims, kappa, c["bc"], U, phi, c["cg_tol"], 10 * 256)
    assert ok and 40 < iters < 200
    n2 = np.sum(np.abs(eta) ** 2)
    assert abs(S - n2) < 1e-12 * n2
    Y = oracle.dslash(dims, kappa, c["bc"], U, X)
    assert np.abs(Y - eta).max() < 1e-12


def test_cg_matches_dense_solve():
    dims, kappa = (2, 3, 2, 4), 0.12
    V = int(np.prod(dims))
    U = synth.warm_links(dims, 0.4, 61)
    n = V * 12
    Dm = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1
        Dm[:, j] = oracle.dslash(dims, kappa, BC, U, e.reshape(V, 4, 3)).ravel()
    Ddm = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1
        Ddm[:, j] = oracle.dslash(dims, kappa, BC, U, e.reshape(V, 4, 3), dagger=True).ravel()
    assert np.allclose(Ddm, dagger(Dm), atol=1e-15)
    b = synth.gaussian_spinor(dims, 62)
    x, iters, rel, ok = oracle.cg(dims, kappa, BC, U, b, 1e-13, 5000)
    xd = np.linalg.solve(dagger(Dm) @ Dm, b.ravel())
    assert ok and rel <= 1e-13
    assert np.abs(x.ravel() - xd).max() < 1e-11 * np.abs(xd).max()
    # cap: returns not-converged with iters == max_iter
    x2, it2, rel2, ok2 = oracle.cg(dims, kappa, BC, U, b, 1e-13, 3)
    assert (not ok2) and it2 == 3 and rel2 > 1e-13
    # zero right-hand side
    x0, it0, rel0, ok0 = oracle.cg(dims, kappa, BC, U, np.zeros_like(b), 1e-13, 10)
    assert ok0 and it0 == 0 and not x0.any()


# ---------------------------------------------------------------- P7
def test_P7_leapfrog_gauge_only():
    dims, beta = (4, 4, 4, 4), 6.0
    U0 = synth.haar_links(dims, 71)
    P0 = synth.gaussian_momenta(dims, 72)
    H0 = oracle.hamiltonian(dims, beta, 0.0, BC, U0, None, P0)[0]
    dH = []
    for nsteps, dt in [(10, 0.04), (20, 0.02), (40, 0.01)]:
        U1, P1, _, ok = oracle.trajectory(dims, beta, 0.0, BC, U0, None, P0, nsteps, dt)
        dH.append(oracle.hamiltonian(dims, beta, 0.0, BC, U1, None, P1)[0] - H0)
    assert 3.6 < dH[0] / dH[1] < 4.4 and 3.8 < dH[1] / dH[2] < 4.2, dH
    # reversibility: forward, flip momenta, forward again
    U1, P1, _, _ = oracle.trajectory(dims, beta, 0.0, BC, U0, None, P0, 20, 0.02)
    U2, P2, _, _ = oracle.trajectory(dims, beta, 0.0, BC, U1, None, -P1, 20, 0.02)
    assert np.abs(U2 - U0).max() < 1e-12 and np.abs(P2 + P0).max() < 1e-11
    # links stay in SU(3) without reunitarisation
    assert np.allclose(U1 @ dagger(U1), np.eye(3), atol=1e-13)


def test_P7_leapfrog_with_fermions():
    c = synth.CONFIGS[0]
    dims, beta, kappa, bc = c["dims"], c["beta"], c["kappa"], c["bc"]
    U0 = synth.config_links(0)
    P0 = synth.gaussian_momenta(dims, 73)
    phi = oracle.dslash(dims, kappa, bc, U0, synth.gaussian_spinor(dims, c["seed_eta"]), dagger=True)
    H0 = oracle.hamiltonian(dims, beta, kappa, bc, U0, phi, P0, tol=1e-13)[0]
    dH = []
    for nsteps, dt in [(4, 0.05), (8, 0.025)]:
        U1, P1, its, ok = oracle.trajectory(dims, beta, kappa, bc, U0, phi, P0, nsteps, dt, tol=1e-13)
        assert ok and its > 0
        dH.append(oracle.hamiltonian(dims, beta, kappa, bc, U1, phi, P1, tol=1e-13)[0] - H0)
    assert 3.5 < dH[0] / dH[1] < 4.5, dH
    U1, P1, _, _ = oracle.trajectory(dims, beta, kappa, bc, U0, phi, P0, 4, 0.05, tol=1e-13)
    U2, P2, _, _ = oracle.trajectory(dims, beta, kappa, bc, U1, phi, -P1, 4, 0.05, tol=1e-13)
    assert np.abs(U2 - U0).max() < 1e-10 and np.abs(P2 + P0).max() < 1e-9


# ---------------------------------------------------------------- P9
def test_P9_paper_route_G_matrix():
    """S2.12: G_ij = dS/dRe U_ij + i dS/dIm U_ij by brute-force differences of S_g in the real
    components; S4 / S2.23 (with U G^dag and S2.24's sign): F = -1/2 TA(U G^dag)."""
    dims, beta = (4, 3, 3, 4), 5.5
    U = synth.warm_links(dims, 0.3, 91)
    F = oracle.gauge_force(dims, beta, U)
    h = 1e-5
    for s, mu in [(5, 0), (100, 3), (143, 2)]:
        G = np.zeros((3, 3), complex)
        for i in range(3):
            for j in range(3):
                for part, unit in ((0, 1.0), (1, 1j)):
                    Up, Um = U.copy(), U.copy()
                    Up[s, mu, i, j] += h * unit
                    Um[s, mu, i, j] -= h * unit
                    d = (oracle.gauge_action(dims, beta, Up)[0] - oracle.gauge_action(dims, beta, Um)[0]) / (2 * h)
                    G[i, j] += d * (1.0 if part == 0 else 1j)
        Fpaper = -0.5 * oracle.ta(U[s, mu] @ dagger(G))
        assert np.abs(Fpaper - F[s, mu]).max() < 1e-7 * np.abs(F[s, mu]).max()


# ---------------------------------------------------------------- P11
def test_P11_half_spinor_outer_product_identity():
    """sum_alpha [(1 +- g_mu) a]_alpha (x) conj(b_alpha) = sum_{t=0,1} h[a]_t (x) conj(h[b]_t),
    h^{+-}_mu[psi] = psi_upper +- sigma_mu psi_lower, sigma_mu = upper-right block of gamma_mu."""
    rng = np.random.default_rng(111)
    a = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    b = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    for mu in range(4):
        sig = GAM[mu][:2, 2:]
        for sg in (+1, -1):
            full = np.einsum("ia,ib->ab", (np.eye(4) + sg * GAM[mu]) @ a, b.conj())
            ha = a[:2] + sg * sig @ a[2:]
            hb = b[:2] + sg * sig @ b[2:]
            assert np.allclose(full, np.einsum("ta,tb->ab", ha, hb.conj()), atol=1e-14)
            # reconstruction: (1 +- gamma) psi = (h, +- sigma^dag h)
            assert np.allclose((np.eye(4) + sg * GAM[mu]) @ a, np.concatenate([ha, sg * dagger(sig) @ ha]), atol=1e-14)


def test_link_rel_err_metric():
    F = synth.gaussian_momenta(DIMS, 5)
    assert link_rel_err(F, F) == (0.0, 0.0)
    G = F.copy()
    G[3, 1] *= 1 + 1e-6
    e, p = link_rel_err(G, F)
    assert abs(e - 1e-6) < 1e-9 and abs(p - 1e-6) < 1e-9
