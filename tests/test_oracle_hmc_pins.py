"""Pins for the HMC-layer oracle (oracle/hmc.py), no GPU.

H1  Philox4x32-10 against the generator's three published known-answer vectors
H2  heat-bath fields: momenta traceless anti-Hermitian with pi^a recovered by -2 tr(tau^a Pi), unit variance,
    K / (8 links) = 1/2; eta with E|eta|^2 = 1; streams, trajectories and seeds are independent
H3  Omelyan with lambda = 1/4 is two leapfrog steps of dt/2 (exact identity of the kick/drift sequences)
H4  Sexton-Weingarten on a gauge-only action is leapfrog with m n steps of dt/m; with fermions and m = 1 it is leapfrog
H5  reversibility and |dH| ~ dt^2 for Omelyan and Sexton-Weingarten; Omelyan beats leapfrog at the same dt
H6  Metropolis: dH = H1 - H0 with S_F(0) = |eta|^2, accept iff u < exp(-dH), links restored on rejection
"""
import numpy as np

import oracle
from oracle import hmc
from paper_2602_20516_b200 import synth

DIMS = (4, 4, 4, 4)
BC = (1, 1, 1, -1)


def test_H1_philox_known_answers():
    kat = [((0, 0, 0, 0), (0, 0), (0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8)),
           ((0xFFFFFFFF,) * 4, (0xFFFFFFFF,) * 2, (0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD)),
           ((0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344), (0xA4093822, 0x299F31D0),
            (0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1))]
    for ctr, key, want in kat:
        got = hmc.philox4x32_10(*ctr, *key)
        assert tuple(int(v[0]) for v in got) == want
    # vectorised call = scalar calls
    c0 = np.arange(5)
    many = hmc.philox4x32_10(c0, 7, 1, 3, 11, 13)
    for i in range(5):
        one = hmc.philox4x32_10(i, 7, 1, 3, 11, 13)
        assert all(int(many[w][i]) == int(one[w][0]) for w in range(4))


def test_H2_heatbath_fields():
    dims = (8, 8, 8, 8)
    V = synth.volume(dims)
    P, pi = hmc.momentum_heatbath(dims, seed=12345, trajectory=0)
    assert np.abs(P + P.conj().swapaxes(-1, -2)).max() < 1e-15
    assert np.abs(np.trace(P, axis1=-2, axis2=-1)).max() < 1e-15
    tau = np.array([oracle.generator(a) for a in range(8)])
    back = -2.0 * np.einsum("aij,nji->na", tau, P.reshape(-1, 3, 3)).real
    assert np.abs(back - pi).max() < 1e-14
    n = pi.size
    assert abs(pi.mean()) < 5 / np.sqrt(n)
    assert abs(pi.var() - 1.0) < 5 * np.sqrt(2.0 / n)
    assert abs(np.mean(pi ** 4) - 3.0) < 5 * np.sqrt(96.0 / n)
    K = oracle.kinetic(dims, P)
    assert abs(K / (4 * V * 8) - 0.5) < 5 * np.sqrt(0.5 / n)
    # components are uncorrelated
    cov = np.cov(pi.T)
    assert np.abs(cov - np.eye(8)).max() < 6 / np.sqrt(4 * V)
    eta = hmc.pseudofermion_noise(dims, seed=12345, trajectory=0)
    m = eta.size
    assert abs(np.mean(np.abs(eta) ** 2) - 1.0) < 5 / np.sqrt(m)
    assert abs(eta.real.var() - 0.5) < 5 * np.sqrt(0.5 / m) and abs(eta.imag.var() - 0.5) < 5 * np.sqrt(0.5 / m)
    assert abs(np.mean(eta.real * eta.imag)) < 5 * 0.5 / np.sqrt(m)
    # different trajectory / seed / stream: different numbers, same call: same numbers
    P1, pi1 = hmc.momentum_heatbath(dims, 12345, 1)
    P2, pi2 = hmc.momentum_heatbath(dims, 12346, 0)
    assert abs(np.mean(pi * pi1)) < 5 / np.sqrt(n) and abs(np.mean(pi * pi2)) < 5 / np.sqrt(n)
    assert abs(np.mean(pi.reshape(V, 32)[:, :12] * eta.real.reshape(V, 12))) < 5 / np.sqrt(12 * V)
    assert np.array_equal(hmc.momentum_heatbath(dims, 12345, 0)[1], pi)
    u = [hmc.metropolis_uniform(99, t) for t in range(2000)]
    assert 0.0 < min(u) and max(u) < 1.0 and abs(np.mean(u) - 0.5) < 5 / np.sqrt(12 * 2000)


def _start(kappa=0.10, beta=5.5, seed=3):
    U = synth.warm_links(DIMS, 0.2, 1001)
    P = synth.gaussian_momenta(DIMS, seed)
    phi = None
    if kappa:
        eta = synth.gaussian_spinor(DIMS, seed + 1)
        phi = oracle.dslash(DIMS, kappa, BC, U, eta, dagger=True)
    return U, P, phi


def test_H3_omelyan_quarter_lambda_is_two_half_leapfrog_steps():
    beta, kappa = 5.5, 0.10
    U, P, phi = _start(kappa, beta)
    Ua, Pa, _ = hmc.integrate(DIMS, beta, kappa, BC, U, phi, P, 3, 0.04, hmc.OMELYAN, lam=0.25)
    Ub, Pb, _ = hmc.integrate(DIMS, beta, kappa, BC, U, phi, P, 6, 0.02, hmc.LEAPFROG)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-12
    # and the library leapfrog of the pinned oracle is the same sequence
    Uc, Pc, _, ok = oracle.trajectory(DIMS, beta, kappa, BC, U, phi, P, 6, 0.02)
    assert ok and np.abs(Uc - Ub).max() < 1e-13 and np.abs(Pc - Pb).max() < 1e-12


def test_H4_sexton_weingarten_special_cases():
    beta = 5.5
    U, P, _ = _start(0.0, beta)
    Ua, Pa, _ = hmc.integrate(DIMS, beta, 0.0, BC, U, None, P, 2, 0.06, hmc.SEXTON_WEINGARTEN, n_inner=3)
    Ub, Pb, _ = hmc.integrate(DIMS, beta, 0.0, BC, U, None, P, 6, 0.02, hmc.LEAPFROG)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-12
    kappa = 0.10
    U, P, phi = _start(kappa, beta)
    Ua, Pa, _ = hmc.integrate(DIMS, beta, kappa, BC, U, phi, P, 3, 0.02, hmc.SEXTON_WEINGARTEN, n_inner=1)
    Ub, Pb, _ = hmc.integrate(DIMS, beta, kappa, BC, U, phi, P, 3, 0.02, hmc.LEAPFROG)
    assert np.abs(Ua - Ub).max() < 1e-13 and np.abs(Pa - Pb).max() < 1e-12


def test_H5_reversibility_and_dt2_scaling():
    beta, kappa = 5.5, 0.10
    U, P, phi = _start(kappa, beta)
    H0 = oracle.hamiltonian(DIMS, beta, kappa, BC, U, phi, P)[0]
    dH = {}
    for integ, m in ((hmc.LEAPFROG, 1), (hmc.OMELYAN, 1), (hmc.SEXTON_WEINGARTEN, 4)):
        for n, dt in ((4, 0.05), (8, 0.025)):
            U1, P1, _ = hmc.integrate(DIMS, beta, kappa, BC, U, phi, P, n, dt, integ, n_inner=m)
            dH[(integ, n)] = oracle.hamiltonian(DIMS, beta, kappa, BC, U1, phi, P1)[0] - H0
            if n == 4:  # flip the momenta and integrate back
                U2, P2, _ = hmc.integrate(DIMS, beta, kappa, BC, U1, phi, -P1, n, dt, integ, n_inner=m)
                assert np.abs(U2 - U).max() < 1e-12 and np.abs(P2 + P).max() < 1e-11
        ratio = dH[(integ, 4)] / dH[(integ, 8)]
        assert 3.3 < ratio < 4.8, (integ, ratio, dH)
    assert abs(dH[(hmc.OMELYAN, 4)]) < 0.5 * abs(dH[(hmc.LEAPFROG, 4)])


def test_H6_metropolis():
    beta, kappa = 5.5, 0.10
    U = synth.warm_links(DIMS, 0.2, 1001)
    out = hmc.hmc_trajectory(DIMS, beta, kappa, BC, U, seed=7, trajectory=0, nsteps=4, dt=0.02)
    # H0 with S_F from the solve equals H0 with S_F = |eta|^2 (pin P6 of the base oracle)
    H0 = oracle.hamiltonian(DIMS, beta, kappa, BC, U, out["phi"], out["P0"], 1e-14)[0]
    assert abs(H0 - out["H0"]) < 1e-9 * abs(H0)
    assert abs(out["dH"]) < 0.5 and out["accepted"] == (out["u"] < np.exp(-out["dH"]))
    # a coarse step is rejected for some trajectory number and then the links come back untouched
    seen = set()
    for traj in range(6):
        o = hmc.hmc_trajectory(DIMS, beta, 0.0, BC, U, seed=7, trajectory=traj, nsteps=1, dt=0.1)
        seen.add(o["accepted"])
        if o["accepted"]:
            assert np.array_equal(o["U"], o["U_proposed"])
        else:
            assert np.array_equal(o["U"], U) and o["dH"] > 0
    assert seen == {True, False}
