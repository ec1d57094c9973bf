"""GPU parity for the HMC layer: heat baths, integrators, Metropolis through the C ABI against
oracle/hmc.py on the same (seed, trajectory).  Gaussians agree to libm rounding (both sides run the same
counter-based generator in double), integrator end states to the base tolerance 1e-11.
"""
import numpy as np
import pytest

import oracle
from oracle import evenodd as oeo
from oracle import hmc as ohmc
from paper_2602_20516_b200 import synth
from lattice_util import link_rel_err

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL64 = 1e-11


@pytest.fixture(scope="module")
def lgt():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the product path has no CPU fallback")
    from paper_2602_20516_b200 import lgt as m

    m.lib()
    return m


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 3, 5, 6), (8, 8, 8, 8)])
def test_heatbaths_match_oracle(lgt, dims):
    kappa, seed, traj = 0.11, 0x1234567890ABCDEF, 5
    U = synth.warm_links(dims, 0.25, 77)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lgt.lgt_momentum_heatbath(lat.ctx, seed, traj)
    P_ref, _ = ohmc.momentum_heatbath(dims, seed, traj)
    P = lat.get_momenta()
    assert np.abs(P - P_ref).max() < 2e-15 * max(1.0, np.abs(P_ref).max())
    n2 = lgt.lgt_pseudofermion_heatbath(lat.ctx, seed, traj)
    eta = ohmc.pseudofermion_noise(dims, seed, traj)
    assert abs(n2 - np.sum(np.abs(eta) ** 2)) < 1e-13 * n2
    phi = lat.empty(synth.volume(dims), 4, 3)
    lgt.lgt_get_pseudofermion(lat.ctx, phi)
    phi_ref = oracle.dslash(dims, kappa, BC, U, eta, dagger=True)
    assert np.abs(phi.cpu().numpy() - phi_ref).max() < 1e-13
    # other trajectory number: other field
    lgt.lgt_momentum_heatbath(lat.ctx, seed, traj + 1)
    assert np.abs(lat.get_momenta() - P_ref).max() > 0.1
    lat.close()


def test_heatbath_even_odd_and_fp32(lgt):
    dims, kappa, seed, traj = (4, 4, 6, 8), 0.12, 99, 2
    U = synth.warm_links(dims, 0.25, 78)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    n2 = lgt.lgt_pseudofermion_heatbath(lat.ctx, seed, traj)
    eta = ohmc.pseudofermion_noise(dims, seed, traj)
    eta_e = oeo.keep(eta, dims, 0)
    assert abs(n2 - np.sum(np.abs(eta_e) ** 2)) < 1e-13 * n2
    phi = lat.empty(synth.volume(dims), 4, 3)
    lgt.lgt_get_pseudofermion(lat.ctx, phi)
    assert np.abs(phi.cpu().numpy() - oeo.mhat(dims, kappa, BC, U, eta_e, dagger=True)).max() < 1e-13
    # S_F of the even/odd action at the start equals |eta_e|^2
    _, S_F, _, _ = lgt.lgt_action(lat.ctx, 1e-13, 5000)
    assert abs(S_F - n2) < 1e-10 * n2
    lat.close()
    lat32 = lgt.Lattice(dims, 5.5, kappa, BC, lgt.LGT_F32)
    lgt.lgt_momentum_heatbath(lat32.ctx, seed, traj)
    P_ref, _ = ohmc.momentum_heatbath(dims, seed, traj)
    assert np.abs(lat32.get_momenta() - P_ref).max() < 1e-6
    lat32.close()


@pytest.mark.parametrize("integ,m", [("omelyan", 1), ("sw", 3), ("sw", 1)])
def test_integrators_match_oracle(lgt, integ, m):
    dims, beta, kappa = (4, 4, 4, 4), 5.5, 0.10
    U0 = synth.warm_links(dims, 0.2, 1001)
    P0 = synth.gaussian_momenta(dims, 5)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 6), dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lat.set_links(U0)
    lat.set_momenta(P0)
    lat.set_pseudofermion(phi)
    code = lgt.LGT_INT_OMELYAN if integ == "omelyan" else lgt.LGT_INT_SEXTON_WEINGARTEN
    ocode = ohmc.OMELYAN if integ == "omelyan" else ohmc.SEXTON_WEINGARTEN
    lgt.lgt_set_integrator(lat.ctx, code, m)
    H0, H1, its = lgt.lgt_md_trajectory(lat.ctx, 3, 0.04, tol=1e-13, max_iter=5000)
    U_ref, P_ref, its_ref = ohmc.integrate(dims, beta, kappa, BC, U0, phi, P0, 3, 0.04, ocode, n_inner=m, tol=1e-13, max_iter=5000)
    assert its == its_ref
    assert np.abs(lat.get_links() - U_ref).max() < 1e-12
    assert link_rel_err(lat.get_momenta(), P_ref)[0] < TOL64
    dH_ref = (oracle.hamiltonian(dims, beta, kappa, BC, U_ref, phi, P_ref, 1e-13, 5000)[0]
              - oracle.hamiltonian(dims, beta, kappa, BC, U0, phi, P0, 1e-13, 5000)[0])
    assert abs((H1 - H0) - dH_ref) < 1e-9 * abs(H0)
    # back to leapfrog: lgt_md_trajectory is the pinned oracle trajectory again
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_LEAPFROG)
    lat.set_links(U0)
    lat.set_momenta(P0)
    lgt.lgt_md_trajectory(lat.ctx, 2, 0.04, tol=1e-13, max_iter=5000, measure=False)
    U_lf, P_lf, _, _ = oracle.trajectory(dims, beta, kappa, BC, U0, phi, P0, 2, 0.04, tol=1e-13, max_iter=5000)
    assert np.abs(lat.get_links() - U_lf).max() < 1e-12 and link_rel_err(lat.get_momenta(), P_lf)[0] < TOL64
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_integrator(lat.ctx, 7)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 0)
    lat.close()


def test_hmc_trajectories_match_oracle(lgt):
    """Three consecutive trajectories with fermions, and coarse gauge-only ones that get rejected: dH, the decision
    (away from the threshold) and the links after the test agree with the oracle."""
    dims, beta, kappa, seed = (4, 4, 4, 4), 5.5, 0.10, 20260220516
    U = synth.warm_links(dims, 0.2, 1001)
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lat.set_links(U)
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_OMELYAN)
    for traj in range(3):
        dH, acc, its, H0, ok = lgt.lgt_hmc_trajectory(lat.ctx, 4, 0.03, seed, traj, tol=1e-13, max_iter=5000)
        ref = ohmc.hmc_trajectory(dims, beta, kappa, BC, U, seed, traj, 4, 0.03, ohmc.OMELYAN, tol=1e-13, max_iter=5000)
        assert ok and abs(H0 - ref["H0"]) < 1e-12 * abs(ref["H0"])
        assert abs(dH - ref["dH"]) < 1e-9 * abs(ref["H0"])
        if abs(ref["u"] - np.exp(-ref["dH"])) > 1e-6:
            assert acc == ref["accepted"]
            assert np.abs(lat.get_links() - ref["U"]).max() < 1e-11
        U = lat.get_links()
    lat.close()
    lat = lgt.Lattice(dims, beta, 0.0, BC)
    U = synth.warm_links(dims, 0.2, 1001)
    lat.set_links(U)
    seen = set()
    for traj in range(6):
        dH, acc, _, _, _ = lgt.lgt_hmc_trajectory(lat.ctx, 1, 0.1, 7, traj)
        ref = ohmc.hmc_trajectory(dims, beta, 0.0, BC, U, 7, traj, 1, 0.1)
        assert abs(dH - ref["dH"]) < 1e-9 * abs(ref["H0"]) and acc == ref["accepted"]
        assert np.abs(lat.get_links() - ref["U"]).max() < 1e-11
        if not acc:
            assert np.array_equal(lat.get_links(), U)  # restored bit for bit
        seen.add(acc)
        U = lat.get_links()
    assert seen == {True, False}
    with pytest.raises(lgt.LgtError):
        lgt.lgt_pseudofermion_heatbath(lat.ctx, 1, 0)  # kappa == 0
    lat.close()


def test_hmc_even_odd_mixed_acceptance(lgt):
    """8^4 with the even/odd action and the Sexton-Weingarten integrator: dH small, exp(-dH) averages to about 1 over a
    few trajectories (Creutz identity, loose), plaquette stays a plaquette."""
    dims, beta, kappa = (8, 8, 8, 8), 5.6, 0.12
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lat.set_links(synth.warm_links(dims, 0.3, 11))
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 4)
    dHs, accs = [], []
    for traj in range(6):
        dH, acc, its, H0, ok = lgt.lgt_hmc_trajectory(lat.ctx, 10, 0.02, 31337, traj, tol=1e-10, max_iter=5000)
        assert ok and its > 0
        dHs.append(dH)
        accs.append(acc)
    assert max(abs(d) for d in dHs) < 1.0 and sum(accs) >= 3
    assert 0.3 < np.mean(np.exp(-np.array(dHs))) < 3.0
    assert 0.3 < lgt.lgt_plaquette(lat.ctx) < 1.0
    lat.close()


def test_pure_gauge_hmc_reproduces_the_known_plaquette(lgt):
    """End-to-end physics check of heat bath + integrator + Metropolis on the GPU: SU(3) Wilson gauge action at
    beta = 6.0 thermalises to the textbook mean plaquette 0.5937 (8^4 is within 1e-3 of the infinite-volume value)."""
    dims, beta = (8, 8, 8, 8), 6.0
    lat = lgt.Lattice(dims, beta, 0.0, (1, 1, 1, 1))
    lat.set_links(synth.warm_links(dims, 0.3, 601))
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_OMELYAN)
    plaq, accs, dHs = [], [], []
    for traj in range(140):  # the white-noise warm start is far from equilibrium: fine steps (trajectory length 1)
        dH, acc, _, _, _ = lgt.lgt_hmc_trajectory(lat.ctx, 25, 0.04, 4242, traj)
        accs.append(acc)
        dHs.append(dH)
        plaq.append(lgt.lgt_plaquette(lat.ctx))
    tail = np.array(plaq[60:])
    assert np.mean(accs[60:]) > 0.7, np.mean(accs)
    assert abs(np.mean(np.exp(-np.array(dHs[60:]))) - 1.0) < 0.15  # <exp(-dH)> = 1
    assert abs(tail.mean() - 0.5937) < 0.004, (tail.mean(), tail.std())
    lat.close()


def test_dynamical_hmc_creutz_identity_with_every_option(lgt):
    """Exactness of the whole chain with fermions: even/odd action + mixed-precision solver + one stout level +
    Sexton-Weingarten.  If any force (the smeared pull-back included) disagreed with the action that Metropolis
    evaluates, or the solver tolerance leaked into dH, <exp(-dH)> would drift from 1 (Creutz) and acceptance would
    collapse; reversibility errors show the same way."""
    dims, beta, kappa = (8, 8, 8, 8), 5.6, 0.12
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lat.set_links(synth.warm_links(dims, 0.3, 9))
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    lgt.lgt_set_smearing(lat.ctx, 1, 0.3)
    lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 10)
    dHs, accs = [], []
    for traj in range(160):
        dH, acc, its, _, ok = lgt.lgt_hmc_trajectory(lat.ctx, 10, 0.1, 90210, traj, tol=1e-10, max_iter=5000)
        assert ok and np.isfinite(dH)
        dHs.append(dH)
        accs.append(acc)
    e = np.exp(-np.array(dHs[60:]))
    sigma = e.std() / np.sqrt(len(e))
    assert np.mean(accs[60:]) > 0.6, np.mean(accs[60:])
    assert abs(e.mean() - 1.0) < max(4 * sigma, 0.05), (e.mean(), sigma)
    U = lat.get_links()
    assert np.abs(U @ U.conj().swapaxes(-1, -2) - np.eye(3)).max() < 1e-12
    lat.close()


@pytest.mark.parametrize("setup", ["8^4 leapfrog", "6^4 stout rho=0.3 Sexton-Weingarten 10"])
def test_fig3_step_size_scaling(lgt, setup):
    """The paper's dynamical validation (Fig. 3): Wilson-fermion HMC at 8^4 without smearing and at 6^4
    with one stout level (rho = 0.3) under Sexton-Weingarten with 10 inner steps; dH must fall like dt^2 at fixed
    trajectory length.  After a short thermalisation every measured configuration is evolved from the same links with
    the same (seed, trajectory) heat bath at dt, dt/2, dt/4, so the ratio is taken configuration by configuration."""
    if setup.startswith("8"):
        dims, smear, integ, m, n0 = (8, 8, 8, 8), 0, lgt.LGT_INT_LEAPFROG, 1, 32
    else:  # the gauge force sits on the inner level, so the outer step can be four times coarser
        dims, smear, integ, m, n0 = (6, 6, 6, 6), 1, lgt.LGT_INT_SEXTON_WEINGARTEN, 10, 8
    lat = lgt.Lattice(dims, 5.6, 0.12, BC)
    lat.set_links(synth.warm_links(dims, 0.3, 33))
    if smear:
        lgt.lgt_set_smearing(lat.ctx, smear, 0.3)
    lgt.lgt_set_integrator(lat.ctx, integ, m)
    seed = 20516
    for traj in range(30):
        _, _, _, _, ok = lgt.lgt_hmc_trajectory(lat.ctx, 10, 0.05, seed, traj, tol=1e-10, max_iter=5000)
        assert ok
    steps = tuple((n0 * k, 1.0 / (n0 * k)) for k in (1, 2, 4))
    dH = {n: [] for n, _ in steps}
    accs = []
    for traj in range(30, 42):
        U = lat.get_links()
        for n, dt in steps:
            lat.set_links(U)
            d, acc, _, _, ok = lgt.lgt_hmc_trajectory(lat.ctx, n, dt, seed, traj, tol=1e-12, max_iter=5000)
            assert ok
            dH[n].append(d)
        accs.append(acc)  # the chain goes on from the finest step's outcome
    a = {n: np.mean(np.abs(dH[n])) for n in dH}
    a0, a1, a2 = (a[n0 * k] for k in (1, 2, 4))
    print("%s: <|dH|> at dt = 1/%d, 1/%d, 1/%d: %.3e %.3e %.3e, ratios %.2f %.2f, acceptance at the finest %.2f"
          % (setup, n0, 2 * n0, 4 * n0, a0, a1, a2, a0 / a1, a1 / a2, np.mean(accs)))
    assert a0 < 1.0
    assert 3.0 < a0 / a1 < 5.5 and 3.3 < a1 / a2 < 4.7, a
    assert np.mean(accs) >= 0.75
    lat.close()


def test_heatbaths_full_size_sampled(lgt):
    """configs[3]'s 32^4 lattice: the heat-bath kernels in their production launch shape, sampled links and sites against
    the oracle's generator evaluated at exactly those elements; K / dof and |eta|^2 / dof as global checks."""
    c = synth.CONFIGS[3]
    dims, seed, traj = c["dims"], 0xABCDEF0123, 17
    V = synth.volume(dims)
    lat = lgt.Lattice(dims, c["beta"], c["kappa"], c["bc"])
    lgt.lgt_momentum_heatbath(lat.ctx, seed, traj)
    P = lat.get_momenta().reshape(4 * V, 3, 3)
    links = np.array([0, 1, 127, 128, 4 * 31 + 3, 4 * (V // 2) + 2, 4 * V - 1, 4 * (V - 33)], dtype=np.uint64)
    g0, g1 = ohmc.gaussian_pairs(seed, traj, ohmc.STREAM_MOMENTA, links[:, None], np.arange(4, dtype=np.uint64)[None, :])
    pi = np.empty((len(links), 8))
    pi[:, 0::2], pi[:, 1::2] = g0, g1
    tau = np.array([oracle.generator(a) for a in range(8)])
    ref = np.einsum("na,aij->nij", pi, tau)
    assert np.abs(P[links.astype(np.int64)] - ref).max() < 1e-14
    _, _, K, _ = lgt.lgt_action(lat.ctx)
    assert abs(K / (4 * V * 8) - 0.5) < 5 * np.sqrt(0.5 / (32 * V))
    n2 = lgt.lgt_pseudofermion_heatbath(lat.ctx, seed, traj)
    assert abs(n2 / (12 * V) - 1.0) < 5 / np.sqrt(12 * V)
    lat.close()


def test_sexton_weingarten_inner_loop_graph_is_bitwise_the_plain_launches(lgt):
    """The 2 m + 1 launches of the inner gauge loop of a Sexton-Weingarten step are replayed as one CUDA graph; with
    per-kernel timing on they are plain launches.  Same kernels in the same order: links, momenta, CG counts and launch
    counts must be identical, with fermions on the even/odd action (whose link copies the replay must invalidate) and
    without, and a second trajectory must reuse the graph."""
    dims = (8, 8, 8, 4)
    U = synth.warm_links(dims, 0.3, 91)
    P = synth.gaussian_momenta(dims, 92)
    for kappa in (0.0, 0.12):
        runs = []
        for timing in (False, True):
            lat = lgt.Lattice(dims, 5.6, kappa, BC)
            lat.set_links(U)
            lat.set_momenta(P)
            if kappa:
                lat.set_pseudofermion(oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 93), dagger=True))
                lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
            lgt.lgt_set_integrator(lat.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 5)
            lgt.lgt_timing_enable(lat.ctx, timing)
            n0 = lgt.lgt_launch_count(lat.ctx)
            its = [lgt.lgt_md_trajectory(lat.ctx, 3, 0.05, 1e-11, 5000, measure=False)[2] for _ in range(2)]
            runs.append((lat.get_links(), lat.get_momenta(), its, lgt.lgt_launch_count(lat.ctx) - n0))
            lat.close()
        assert runs[0][2] == runs[1][2] and runs[0][3] == runs[1][3]
        assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1])
