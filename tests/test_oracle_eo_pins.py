"""Pins for the even/odd oracle (oracle/evenodd.py), no GPU.  What fixes it is linear algebra, not the oracle:

E1  M equals the Schur complement D_ee - D_eo D_oo^-1 D_oe of the dense matrix of D, D_oo = 1, det D = det M,
    and M^dag is the conjugate transpose (2^4 lattice, antiperiodic time);
E2  CG on M^dag M against a dense solve; caps and the zero right-hand side;
E3  phi_e = M^dag eta_e  =>  S_F^eo = |eta_e|^2 and Y_e = M X_e = eta_e (closed form);
E4  the force of S_F^eo equals the Richardson central difference of S_F^eo along U -> exp(t tau^a) U on links that
    start on even and on odd sites and that cross the antiperiodic boundary (this pins the reconstruction
    X_o = kappa H_oe X_e, Y_o = kappa H_oe^dag Y_e and every sign in it);
E5  S_F^eo is gauge invariant and odd extents are refused.
"""
import numpy as np
import pytest
from scipy.linalg import expm as scipy_expm

import oracle
from oracle import evenodd as eo
from paper_2602_20516_b200 import synth
from lattice_util import dagger, gauge_transform_links, gauge_transform_spinor, random_su3

BC = (1, 1, 1, -1)
TAU = [oracle.generator(a) for a in range(8)]


def dense(op, V):
    n = V * 12
    M = np.empty((n, n), complex)
    for j in range(n):
        e = np.zeros(n, complex)
        e[j] = 1
        M[:, j] = op(e.reshape(V, 4, 3)).ravel()
    return M


def test_E1_mhat_is_the_schur_complement_and_preserves_the_determinant():
    dims, kappa = (2, 2, 2, 2), 0.13
    V = 16
    U = synth.warm_links(dims, 0.5, 301)
    par = eo.parity(dims)
    assert par.sum() == V // 2 and par[0] == 0 and par[1] == 1 and par[2] == 1 and par[3] == 0
    D = dense(lambda v: oracle.dslash(dims, kappa, BC, U, v), V)
    M = dense(lambda v: eo.mhat(dims, kappa, BC, U, v), V)
    Md = dense(lambda v: eo.mhat(dims, kappa, BC, U, v, dagger=True), V)
    ev = np.repeat(par == 0, 12)
    od = ~ev
    Dee, Deo, Doe, Doo = D[np.ix_(ev, ev)], D[np.ix_(ev, od)], D[np.ix_(od, ev)], D[np.ix_(od, od)]
    assert np.allclose(Doo, np.eye(Doo.shape[0]), atol=1e-15) and np.allclose(Dee, np.eye(Dee.shape[0]), atol=1e-15)
    schur = Dee - Deo @ np.linalg.solve(Doo, Doe)
    assert np.abs(M[np.ix_(ev, ev)] - schur).max() < 1e-14
    assert not M[np.ix_(od, ev)].any() and not M[np.ix_(ev, od)].any() and not M[np.ix_(od, od)].any()
    assert np.abs(Md - dagger(M)).max() < 1e-14
    dD, dM = np.linalg.det(D), np.linalg.det(schur)
    assert abs(dD - dM) < 1e-11 * abs(dD)


def test_E2_cg_matches_dense_solve():
    dims, kappa = (2, 4, 2, 2), 0.12
    V = int(np.prod(dims))
    U = synth.warm_links(dims, 0.4, 311)
    M = dense(lambda v: eo.mhat(dims, kappa, BC, U, v), V)
    ev = np.repeat(eo.parity(dims) == 0, 12)
    Me = M[np.ix_(ev, ev)]
    b = synth.gaussian_spinor(dims, 312)
    x, it, rel, ok = eo.cg(dims, kappa, BC, U, b, 1e-13, 2000)
    assert ok and rel <= 1e-13 and it > 3
    xd = np.linalg.solve(dagger(Me) @ Me, b.ravel()[ev])
    assert np.abs(x.ravel()[ev] - xd).max() < 1e-11 * np.abs(xd).max()
    assert not x.ravel()[~ev].any()
    x2, it2, rel2, ok2 = eo.cg(dims, kappa, BC, U, b, 1e-13, 2)
    assert (not ok2) and it2 == 2 and rel2 > 1e-13
    x0, it0, _, ok0 = eo.cg(dims, kappa, BC, U, np.zeros_like(b), 1e-13, 10)
    assert ok0 and it0 == 0 and not x0.any()


def test_E3_phi_from_eta_closed_form():
    dims, kappa = (4, 4, 4, 4), 0.12
    U = synth.warm_links(dims, 0.3, 321)
    eta = eo.keep(synth.gaussian_spinor(dims, 322), dims, 0)
    phi = eo.mhat(dims, kappa, BC, U, eta, dagger=True)
    S, Xe, it, ok = eo.action(dims, kappa, BC, U, phi, 1e-14, 2000)
    n2 = np.sum(np.abs(eta) ** 2)
    assert ok and abs(S - n2) < 1e-12 * n2
    X, Y, _, _ = eo.solve_xy(dims, kappa, BC, U, phi, 1e-14, 2000)
    assert np.abs(eo.keep(Y, dims, 0) - eta).max() < 1e-12
    # fewer iterations than the unpreconditioned solve of the same determinant
    _, it_full, _, _ = oracle.cg(dims, kappa, BC, U, oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 322), dagger=True),
                                 1e-14, 5000)
    assert it < it_full


def test_E4_force_is_derivative_of_the_even_odd_action():
    dims, kappa = (4, 4, 2, 4), 0.11
    V = int(np.prod(dims))
    U = synth.warm_links(dims, 0.25, 331)
    phi = synth.gaussian_spinor(dims, 332)
    F, it, ok = eo.fermion_force(dims, kappa, BC, U, phi, 1e-14, 3000)
    assert ok
    act = lambda W: eo.action(dims, kappa, BC, W, phi, 1e-14, 3000)[0]
    par = eo.parity(dims)

    def fd(s, mu, a, t):
        def cd(h):
            Up, Um = U.copy(), U.copy()
            Up[s, mu] = scipy_expm(h * TAU[a]) @ U[s, mu]
            Um[s, mu] = scipy_expm(-h * TAU[a]) @ U[s, mu]
            return (act(Up) - act(Um)) / (2 * h)
        return (4 * cd(t) - cd(2 * t)) / 3

    worst = 0.0
    links = [(0, 0), (1, 1), (V - 1, 3), (V - 2, 3), (21, 2), (38, 0)]
    assert {int(par[s]) for s, _ in links} == {0, 1}
    for s, mu in links:
        for a in (0, 1, 2, 4, 7):
            an = (-2 * np.trace(TAU[a] @ F[s, mu])).real
            worst = max(worst, abs(fd(s, mu, a, 2e-3) - an))
    assert worst < 1e-8 * np.abs(F).max(), worst
    # a wrong reconstruction (odd parts dropped) is far from the derivative: the pin has teeth
    Xe, _, _, _ = eo.cg(dims, kappa, BC, U, phi, 1e-14, 3000)
    Fbad = oracle.fermion_force(dims, kappa, BC, U, Xe, eo.mhat(dims, kappa, BC, U, Xe))
    assert np.abs(Fbad - F).max() > 0.1 * np.abs(F).max()


def test_E5_gauge_invariance_and_odd_extents():
    dims, kappa = (4, 2, 4, 2), 0.12
    V = int(np.prod(dims))
    U = synth.warm_links(dims, 0.3, 341)
    phi = synth.gaussian_spinor(dims, 342)
    g = random_su3(V, np.random.default_rng(343))
    S, _, _, ok = eo.action(dims, kappa, BC, U, phi, 1e-13, 2000)
    Sg, _, _, okg = eo.action(dims, kappa, BC, gauge_transform_links(U, g, dims), gauge_transform_spinor(phi, g), 1e-13, 2000)
    assert ok and okg and abs(S - Sg) < 1e-10 * abs(S)
    with pytest.raises(ValueError):
        eo.parity((4, 3, 4, 4))
