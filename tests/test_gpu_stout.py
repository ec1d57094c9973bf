"""GPU parity for stout-smeared fermions through the C ABI against oracle/stout.py: smeared links,
Dirac operator and solve on them, the pulled-back fermion force per link (1e-11), MD with the smeared action.
"""
import numpy as np
import pytest

import oracle
from oracle import stout as ost
from paper_2602_20516_b200 import synth
from lattice_util import link_rel_err

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
RHO = 0.3
TOL64 = 1e-11


@pytest.fixture(scope="module")
def lgt():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the product path has no CPU fallback")
    from paper_2602_20516_b200 import lgt as m

    m.lib()
    return m


def smeared_links(lgt, lat, V):
    U = lat.empty(V, 4, 3, 3)
    lgt.lgt_get_smeared_links(lat.ctx, U)
    return U.cpu().numpy()


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 4), 1), ((4, 3, 5, 6), 2), ((8, 8, 8, 8), 1), ((6, 2, 1, 10), 3)])
def test_smeared_links_and_dslash(lgt, dims, n):
    kappa = 0.11
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 401)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lgt.lgt_set_smearing(lat.ctx, n, RHO)
    Un = ost.smear_levels(dims, RHO, n, U)[0][-1]
    assert np.abs(smeared_links(lgt, lat, V) - Un).max() < 1e-13
    assert np.abs(lat.get_links() - U).max() == 0.0  # the thin links are untouched
    psi = synth.gaussian_spinor(dims, 402)
    for dag in (False, True):
        ref = oracle.dslash(dims, kappa, BC, Un, psi, dagger=dag)
        assert np.abs(lat.dslash(psi, dagger=dag) - ref).max() < 1e-12
    # the gauge action stays on the thin links
    S_g, _, _, _ = lgt.lgt_action(lat.ctx)
    assert abs(S_g - oracle.gauge_action(dims, 5.5, U)[0]) < 1e-11 * abs(S_g)
    # switching off restores the thin operator; new links invalidate the smeared ones
    lgt.lgt_set_smearing(lat.ctx, 0)
    assert np.abs(lat.dslash(psi) - oracle.dslash(dims, kappa, BC, U, psi)).max() < 1e-12
    lgt.lgt_set_smearing(lat.ctx, n, RHO)
    U2 = synth.warm_links(dims, 0.2, 403)
    lat.set_links(U2)
    assert np.abs(smeared_links(lgt, lat, V) - ost.smear_levels(dims, RHO, n, U2)[0][-1]).max() < 1e-13
    lat.close()


@pytest.mark.parametrize("dims,n,rho,eps", [((4, 4, 4, 4), 1, 0.3, 0.25), ((4, 4, 4, 4), 2, 0.3, 0.25),
                                            ((4, 3, 5, 6), 1, 0.3, 0.3), ((4, 6, 2, 4), 3, 0.1, 0.3),
                                            ((4, 4, 4, 4), 1, 0.3, 0.01), ((4, 4, 4, 4), 1, 1e-3, 0.2)])
def test_smeared_fermion_force(lgt, dims, n, rho, eps):
    """Per-link force with respect to the thin links; eps = 0.01 and rho = 1e-3 put every |Q| into the series branch of
    stout_local_kernel, the others into the closed Cayley-Hamilton branch."""
    kappa = 0.11
    U = synth.warm_links(dims, eps, 411)
    eta = synth.gaussian_spinor(dims, 412)
    Un = ost.smear_levels(dims, rho, n, U)[0][-1]
    phi = oracle.dslash(dims, kappa, BC, Un, eta, dagger=True)
    F_ref, it_ref, ok = ost.fermion_force(dims, kappa, BC, U, phi, n, rho, 1e-13, 5000)
    assert ok
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    lgt.lgt_set_smearing(lat.ctx, n, rho)
    F, it = lat.fermion_force(tol=1e-13, max_iter=5000)
    assert it == it_ref
    err, plain = link_rel_err(F, F_ref)
    assert err < TOL64, (err, plain)
    _, S_F, _, _ = lgt.lgt_action(lat.ctx, 1e-13, 5000)
    S_ref = ost.fermion_action(dims, kappa, BC, U, phi, n, rho, 1e-13, 5000)[0]
    assert abs(S_F - S_ref) < 1e-11 * abs(S_ref)
    lat.close()


def test_smeared_force_pieces_one_level(lgt):
    """X, Y given: the pull-back alone (no solve on the GPU side), against oracle.pull_back and its direct part."""
    dims, kappa = (4, 4, 4, 4), 0.12
    U = synth.warm_links(dims, 0.3, 421)
    U1, A = ost.smear(dims, RHO, U)
    X = synth.gaussian_spinor(dims, 422)
    Y = synth.gaussian_spinor(dims, 423)
    Fp = oracle.fermion_force(dims, kappa, BC, U1, X, Y)
    F_ref, F_dir, G = ost.pull_back(dims, RHO, U, A, Fp)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lgt.lgt_set_smearing(lat.ctx, 1, RHO)
    F, _ = lat.fermion_force(X, Y)
    err, plain = link_rel_err(F, F_ref)
    assert err < TOL64, (err, plain)
    # rho = 0: the smeared force is the thin force on the same links
    lgt.lgt_set_smearing(lat.ctx, 2, 0.0)
    F0, _ = lat.fermion_force(X, Y)
    assert link_rel_err(F0, oracle.fermion_force(dims, kappa, BC, U, X, Y))[0] < TOL64
    lat.close()


def test_smeared_md_conserves_energy_and_reverses(lgt):
    """Wilson fermions on stout links (rho = 0.3), Sexton-Weingarten; |dH| ~ dt^2 and reversibility
    with the GPU force, and one step against the oracle's kick assembled from ost.fermion_force."""
    dims, beta, kappa = (4, 4, 4, 4), 5.6, 0.11
    U0 = synth.warm_links(dims, 0.25, 431)
    P0 = synth.gaussian_momenta(dims, 432)
    Un = ost.smear_levels(dims, RHO, 1, U0)[0][-1]
    phi = oracle.dslash(dims, kappa, BC, Un, synth.gaussian_spinor(dims, 433), dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_smearing(lat.ctx, 1, RHO)
    lat.set_links(U0)
    lat.set_momenta(P0)
    lat.set_pseudofermion(phi)
    # one kick against the oracle
    lgt.lgt_md_kick(lat.ctx, 0.05, 1e-13, 5000)
    Ff, _, _ = ost.fermion_force(dims, kappa, BC, U0, phi, 1, RHO, 1e-13, 5000)
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + Ff)
    assert link_rel_err(lat.get_momenta(), P_ref)[0] < TOL64
    # dt^2 scaling and reversibility with the Sexton-Weingarten integrator
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 4)
    dH = []
    for nsteps, dt in ((4, 0.04), (8, 0.02)):
        lat.set_links(U0)
        lat.set_momenta(P0)
        H0, H1, _ = lgt.lgt_md_trajectory(lat.ctx, nsteps, dt, tol=1e-13, max_iter=5000)
        dH.append(H1 - H0)
        if nsteps == 4:
            lat.set_momenta(-lat.get_momenta())
            lgt.lgt_md_trajectory(lat.ctx, nsteps, dt, tol=1e-13, max_iter=5000, measure=False)
            assert np.abs(lat.get_links() - U0).max() < 1e-11
            assert np.abs(lat.get_momenta() + P0).max() < 1e-10
    assert 3.0 < dH[0] / dH[1] < 5.0, dH
    lat.close()


def test_smearing_with_solver_variants_and_fp32(lgt):
    """Even/odd action and mixed-precision solver run on the smeared links too; fp32 force at 2e-5; bad arguments."""
    dims, kappa = (4, 4, 4, 8), 0.11
    U = synth.warm_links(dims, 0.25, 441)
    Un = ost.smear_levels(dims, RHO, 1, U)[0][-1]
    phi = oracle.dslash(dims, kappa, BC, Un, synth.gaussian_spinor(dims, 442), dagger=True)
    F_ref, _, _ = ost.fermion_force(dims, kappa, BC, U, phi, 1, RHO, 1e-13, 5000)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    lgt.lgt_set_smearing(lat.ctx, 1, RHO)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    F, _ = lat.fermion_force(tol=1e-13, max_iter=5000)
    assert link_rel_err(F, F_ref)[0] < 1e-10
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_CG)
    from oracle import evenodd as oeo
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    Xe, Ye, _, _ = oeo.solve_xy(dims, kappa, BC, Un, phi, 1e-13, 5000)
    Fp = oracle.fermion_force(dims, kappa, BC, Un, Xe, Ye)
    Feo_ref = ost.pull_back(dims, RHO, U, ost.smear(dims, RHO, U)[1], Fp)[0]
    Feo, _ = lat.fermion_force(tol=1e-13, max_iter=5000)
    assert link_rel_err(Feo, Feo_ref)[0] < TOL64
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_smearing(lat.ctx, 9, 0.1)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_smearing(lat.ctx, 1, -0.1)
    lat.close()
    lat32 = lgt.Lattice(dims, 5.5, kappa, BC, lgt.LGT_F32)
    lat32.set_links(U.astype(np.complex64))
    lgt.lgt_set_smearing(lat32.ctx, 1, RHO)
    X, _, _, _ = oracle.cg(dims, kappa, BC, Un, phi, 1e-13, 5000)
    Y = oracle.dslash(dims, kappa, BC, Un, X)
    F32, _ = lat32.fermion_force(X.astype(np.complex64), Y.astype(np.complex64))
    assert link_rel_err(F32.astype(np.complex128), F_ref)[0] < 2e-4  # fp32 inputs and a deeper chain than the thin force
    lat32.close()


def test_paper_second_hmc_setup(lgt):
    """6^4, Wilson fermions on stout links (rho = 0.3), Sexton-Weingarten with 10 inner gauge steps.
    A few HMC trajectories from a warm start: |dH| small and shrinking like dt^2 between two step sizes on the same
    (seed, trajectory), trajectories accepted, links stay SU(3)."""
    dims, beta, kappa = (6, 6, 6, 6), 5.6, 0.11
    U0 = synth.warm_links(dims, 0.25, 451)
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_smearing(lat.ctx, 1, RHO)
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 10)
    dH = {}
    for nsteps, dt in ((5, 0.04), (10, 0.02)):
        lat.set_links(U0)
        d, acc, its, H0, ok = lgt.lgt_hmc_trajectory(lat.ctx, nsteps, dt, 451, 0, tol=1e-11, max_iter=5000)
        assert ok and its > 0
        dH[nsteps] = d
    assert abs(dH[5]) < 1.0 and 2.5 < dH[5] / dH[10] < 6.0, dH
    lat.set_links(U0)
    accs = []
    for traj in range(4):
        d, acc, _, _, ok = lgt.lgt_hmc_trajectory(lat.ctx, 10, 0.02, 452, traj, tol=1e-11, max_iter=5000)
        assert ok and abs(d) < 0.5
        accs.append(acc)
    assert sum(accs) >= 3
    U = lat.get_links()
    assert np.abs(U @ U.conj().swapaxes(-1, -2) - np.eye(3)).max() < 1e-12
    lat.close()


def test_smeared_force_16x16x16x16(lgt):
    """configs[2]'s lattice (several hundred blocks per kernel, ragged nothing): one stout level, X and Y given, so that
    the pull-back kernels alone are compared per link with the oracle at a size well beyond one tile."""
    c = synth.CONFIGS[2]
    dims, kappa, bc = c["dims"], c["kappa"], c["bc"]
    U = synth.config_links(2)
    U1, A = ost.smear(dims, RHO, U)
    X = synth.gaussian_spinor(dims, 461)
    Y = synth.gaussian_spinor(dims, 462)
    Fp = oracle.fermion_force(dims, kappa, bc, U1, X, Y)
    F_ref = ost.pull_back(dims, RHO, U, A, Fp)[0]
    lat = lgt.Lattice(dims, 5.6, kappa, bc)
    lat.set_links(U)
    lgt.lgt_set_smearing(lat.ctx, 1, RHO)
    assert np.abs(smeared_links(lgt, lat, synth.volume(dims)) - U1).max() < 1e-13
    F, _ = lat.fermion_force(X, Y)
    err, plain = link_rel_err(F, F_ref)
    assert err < TOL64, (err, plain)
    lat.close()
