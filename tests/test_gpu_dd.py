"""GPU parity for the time-slab decomposition (lgt_dd_*): all ranks of the group live on the one GPU and are
stepped in lockstep with device copies as the exchange (no rank waits on another), so the decomposed kernels, halo
logic, global sums and boundary signs are verified against the oracle on the undivided lattice; the NCCL transport
is exercised with one rank (send/recv to itself through the same code path).
"""
import numpy as np
import pytest

import oracle
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


def cat(slabs):
    return np.concatenate(slabs, axis=0)


@pytest.mark.parametrize("dims,nranks", [((4, 4, 2, 8), 1), ((4, 4, 2, 8), 2), ((4, 4, 2, 8), 4), ((8, 4, 4, 6), 3),
                                         ((4, 4, 2, 8), 8), ((8, 8, 8, 8), 2)])
def test_dd_dslash_matches_oracle_and_single_handle(lgt, dims, nranks):
    kappa = 0.12
    U = synth.warm_links(dims, 0.3, 501)
    psi = synth.gaussian_spinor(dims, 502)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), 5.5, kappa, BC)
    dd.set_links(U)
    one = lgt.Lattice(dims, 5.5, kappa, BC)
    one.set_links(U)
    for dag in (False, True):
        out = cat(dd.dslash(psi, dagger=dag))
        assert np.abs(out - oracle.dslash(dims, kappa, BC, U, psi, dagger=dag)).max() < 1e-12
        assert np.array_equal(out, one.dslash(psi, dagger=dag))  # same kernel, same order of operations per site
    assert np.array_equal(cat(dd.get_links()), U)
    # a slab handle refuses the single-lattice calls
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_plaquette(dd.ranks[0])
    assert e.value.code == lgt.LGT_ESTATE
    dd.close()
    one.close()


@pytest.mark.parametrize("nranks", [2, 4])
def test_dd_cg(lgt, nranks):
    dims, kappa = (4, 4, 4, 8), 0.12
    U = synth.warm_links(dims, 0.3, 511)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 512), dagger=True)
    x_ref, it_ref, _, ok = oracle.cg(dims, kappa, BC, U, b, 1e-12, 5000)
    assert ok
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), 5.5, kappa, BC)
    dd.set_links(U)
    xs, it, rel, ok = dd.cg(b, 1e-12, 5000)
    assert ok and it == it_ref and rel <= 1e-12
    x = cat(xs)
    assert np.linalg.norm(x - x_ref) < 1e-10 * np.linalg.norm(x_ref)
    dd.close()


@pytest.mark.parametrize("nranks", [2, 4])
def test_dd_md_trajectory(lgt, nranks):
    """Leapfrog with both forces on the decomposed lattice against the oracle's trajectory on the undivided one."""
    dims, beta, kappa = (4, 4, 2, 8), 5.6, 0.11
    U0 = synth.warm_links(dims, 0.25, 521)
    P0 = synth.gaussian_momenta(dims, 522)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 523), dagger=True)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    S_g, S_F, K, _ = lgt.lgt_dd_action(dd.d, 1e-13, 5000)
    H_ref, K_ref, Sg_ref, SF_ref = oracle.hamiltonian(dims, beta, kappa, BC, U0, phi, P0, 1e-13, 5000)
    assert abs(S_g - Sg_ref) < 1e-11 * abs(Sg_ref) and abs(S_F - SF_ref) < 1e-10 * abs(SF_ref) and abs(K - K_ref) < 1e-12 * K_ref
    H0, H1, its = lgt.lgt_dd_md_trajectory(dd.d, 3, 0.03, tol=1e-13, max_iter=5000)
    U_ref, P_ref, its_ref, ok = oracle.trajectory(dims, beta, kappa, BC, U0, phi, P0, 3, 0.03, tol=1e-13, max_iter=5000)
    assert ok and its == its_ref
    assert np.abs(cat(dd.get_links()) - U_ref).max() < 1e-12
    assert link_rel_err(cat(dd.get_momenta()), P_ref)[0] < TOL64
    H1_ref = oracle.hamiltonian(dims, beta, kappa, BC, U_ref, phi, P_ref, 1e-13, 5000)[0]
    assert abs((H1 - H0) - (H1_ref - H_ref)) < 1e-9 * abs(H_ref)
    # kick and drift on their own
    dd.set_links(U0)
    dd.set_momenta(P0)
    lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U0, phi, P0, 0.05, 1e-13, 5000)
    assert link_rel_err(cat(dd.get_momenta()), P1)[0] < TOL64
    lgt.lgt_dd_md_drift(dd.d, 0.05)
    assert np.abs(cat(dd.get_links()) - oracle.drift(dims, 0.05, P1, U0)).max() < 1e-13
    dd.close()


def test_dd_nccl_transport_one_rank(lgt):
    """The NCCL code path (send/recv of the halo slices to itself, all-reduce of the sums) with a single rank."""
    dims, kappa = (4, 4, 2, 8), 0.12
    U = synth.warm_links(dims, 0.3, 531)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 532), dagger=True)
    dd = lgt.DecomposedLattice(dims, 1, [0], 5.5, kappa, BC)
    lgt.lgt_dd_nccl_init(dd.d, lgt.lgt_dd_nccl_unique_id())
    dd.set_links(U)
    assert np.abs(cat(dd.dslash(b)) - oracle.dslash(dims, kappa, BC, U, b)).max() < 1e-12
    x_ref, it_ref, _, _ = oracle.cg(dims, kappa, BC, U, b, 1e-12, 5000)
    xs, it, rel, ok = dd.cg(b, 1e-12, 5000)
    assert ok and it == it_ref and np.linalg.norm(cat(xs) - x_ref) < 1e-10 * np.linalg.norm(x_ref)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_nccl_init(dd.d, lgt.lgt_dd_nccl_unique_id())  # already initialised
    dd.close()


def test_grid_nccl_transport_one_rank(lgt):
    """The NCCL code path of the (Pt, Pz) grid with a single rank (1 x 1): the z faces are gathered into a device staging
    buffer by 2-D copies, sent and received (to itself) through NCCL, and scattered into the ghost planes; kick with both
    forces (the staples' corners go through the same two phases) against the oracle."""
    dims, beta, kappa = (8, 4, 4, 4), 5.6, 0.12
    U = synth.warm_links(dims, 0.3, 731)
    P0 = synth.gaussian_momenta(dims, 732)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 733), dagger=True)
    dd = lgt.DecomposedLattice(dims, 1, [0], beta, kappa, BC, grid=(1, 1))
    lgt.lgt_dd_nccl_init(dd.d, lgt.lgt_dd_nccl_unique_id())
    dd.set_links(U)
    assert np.abs(dd.dslash(b)[0] - oracle.dslash(dims, kappa, BC, U, b)).max() < 1e-12
    x_ref, it_ref, _, _ = oracle.cg(dims, kappa, BC, U, b, 1e-12, 5000)
    xs, it, rel, ok = dd.cg(b, 1e-12, 5000)
    assert ok and it == it_ref and np.linalg.norm(xs[0] - x_ref) < 1e-10 * np.linalg.norm(x_ref)
    dd.set_momenta(P0)
    dd.set_pseudofermion(b)
    lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U, b, P0, 0.05, 1e-13, 5000)
    assert link_rel_err(dd.get_momenta()[0], P1)[0] < TOL64
    dd.close()


def test_dd_argument_checks(lgt):
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_create((4, 4, 2, 8), 3, [0, 1, 2], 5.5, 0.1, BC)  # Lt not divisible
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_create((4, 3, 2, 8), 2, [0, 1], 5.5, 0.1, BC)  # time slice not a multiple of 32 sites
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_create((4, 4, 2, 8), 4, [0, 1], 5.5, 0.1, BC)  # neither all local nor one local
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_create((4, 4, 2, 8), 2, [0, 0], 5.5, 0.1, BC)
    d = lgt.lgt_dd_create((4, 4, 2, 8), 2, [0, 1], 5.5, 0.1, BC)
    assert lgt.lgt_dd_local_ranks(d) == 2
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_nccl_init(d, b"\0" * 128)  # NCCL serves one rank per process
    lgt.lgt_dd_destroy(d)


def test_dd_host_slab_roundtrip(lgt):
    """The _host setters / getters on a rank handle move the slab's own rows only."""
    import torch

    dims, nranks = (4, 4, 2, 8), 2
    U = synth.warm_links(dims, 0.3, 541)
    P = synth.gaussian_momenta(dims, 542)
    dd = lgt.DecomposedLattice(dims, nranks, [0, 1], 5.5, 0.12, BC)
    for i in range(nranks):
        hU = torch.from_numpy(dd.slab(U, i).copy())
        hP = torch.from_numpy(dd.slab(P, i).copy())
        lgt.lgt_set_links_host(dd.ranks[i], hU)
        lgt.lgt_set_momenta_host(dd.ranks[i], hP)
        oU, oP = torch.empty_like(hU), torch.empty_like(hP)
        lgt.lgt_get_links_host(dd.ranks[i], oU)
        lgt.lgt_get_momenta_host(dd.ranks[i], oP)
        assert torch.equal(oU, hU) and (oP - hP).abs().max().item() < 1e-15
    psi = synth.gaussian_spinor(dims, 543)
    assert np.abs(cat(dd.dslash(psi)) - oracle.dslash(dims, 0.12, BC, U, psi)).max() < 1e-12
    dd.close()


def lgt_dag(lgt, dims, c, U, psi):
    one = lgt.Lattice(dims, c["beta"], c["kappa"], c["bc"])
    one.set_links(U)
    out = one.dslash(psi, dagger=True)
    one.close()
    return out


def test_dd_full_size_dslash_four_slabs(lgt):
    """configs[3]'s 32^4 lattice in four slabs on this GPU: bitwise equal to the undivided Dslash, sampled sites against
    the oracle (incl. sites on slab boundaries and on the antiperiodic time boundary)."""
    c = synth.CONFIGS[3]
    dims, kappa, bc = c["dims"], c["kappa"], c["bc"]
    V = synth.volume(dims)
    U = synth.config_links(3)
    psi = synth.gaussian_spinor(dims, 551)
    one = lgt.Lattice(dims, c["beta"], kappa, bc)
    one.set_links(U)
    ref = one.dslash(psi)
    one.close()
    dd = lgt.DecomposedLattice(dims, 4, [0, 1, 2, 3], c["beta"], kappa, bc)
    dd.set_links(U)
    out = cat(dd.dslash(psi))
    dd.close()
    assert np.array_equal(out, ref)
    # the same lattice on a 2 x 2 (t, z) grid of ranks
    dg = lgt.DecomposedLattice(dims, 4, [0, 1, 2, 3], c["beta"], kappa, bc, grid=(2, 2))
    dg.set_links(U)
    assert np.array_equal(gather_grid(dims, (2, 2), dg.dslash(psi)), ref)
    assert np.array_equal(gather_grid(dims, (2, 2), dg.dslash(psi, dagger=True)), lgt_dag(lgt, dims, c, U, psi))
    dg.close()
    V3 = dims[0] * dims[1] * dims[2]
    sites = np.array([0, 5, V3 * 8 - 1, V3 * 8, V3 * 16 + 77, V3 * 24 - 3, V - V3 + 9, V - 1], dtype=np.int64)
    assert np.abs(out[sites] - oracle.dslash_sites(dims, kappa, bc, U, psi, sites)).max() < 1e-12


@pytest.mark.parametrize("nranks", [1, 2, 4, 8])
def test_dd_pushed_halos_are_bitwise_the_exchanged_ones(lgt, nranks):
    """LGT_DD_PUSH: the Dslash kernels of the CG loop store their boundary slices into the neighbours' ghost slices and
    the ghosts of p follow by local arithmetic; no separate transfer inside the iteration.  Same iterates bit for bit
    as with the separate exchange, the oracle's iteration count, and the MD trajectory on top of it.  Time slices of 128
    sites, so that the boundary slices run the pushing kernel and the bulk the ordinary one (8 slabs: one slice per slab
    feeds both neighbours; 4 slabs: no bulk)."""
    dims, beta, kappa = (8, 4, 4, 8), 5.6, 0.12
    U = synth.warm_links(dims, 0.3, 561)
    P0 = synth.gaussian_momenta(dims, 562)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 563), dagger=True)
    x_ref, it_ref, _, ok = oracle.cg(dims, kappa, BC, U, b, 1e-12, 5000)
    res = {}
    for mode in (lgt.LGT_DD_EXCHANGE, lgt.LGT_DD_PUSH, lgt.LGT_DD_OVERLAP, lgt.LGT_DD_HALF):
        dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
        lgt.lgt_dd_set_halo_mode(dd.d, mode)
        dd.set_links(U)
        xs, it, rel, ok = dd.cg(b, 1e-12, 5000)
        assert ok and it == it_ref
        dd.set_momenta(P0)
        dd.set_pseudofermion(b)
        H0, H1, its = lgt.lgt_dd_md_trajectory(dd.d, 2, 0.03, tol=1e-13, max_iter=5000)
        res[mode] = (cat(xs), cat(dd.get_links()), cat(dd.get_momenta()), H1 - H0, its)
        dd.close()
    ex, pu = res[lgt.LGT_DD_EXCHANGE], res[lgt.LGT_DD_PUSH]
    assert np.array_equal(ex[0], pu[0]) and np.array_equal(ex[1], pu[1]) and np.array_equal(ex[2], pu[2])
    assert ex[3] == pu[3] and ex[4] == pu[4]
    # LGT_DD_OVERLAP: the exchange on a second stream under the bulk of the slab, the boundary slices after it (slabs of
    # three and more slices: 1 and 2 slabs here; thinner slabs fall back to the plain exchange) -- the same bits again
    ov = res[lgt.LGT_DD_OVERLAP]
    assert np.array_equal(ex[0], ov[0]) and np.array_equal(ex[1], ov[1]) and np.array_equal(ex[2], ov[2])
    assert ex[3] == ov[3] and ex[4] == ov[4]
    # LGT_DD_HALF: the overlapped schedule with projected (and, for the backward face, multiplied) half spinors on the wire
    ha = res[lgt.LGT_DD_HALF]
    assert np.array_equal(ex[0], ha[0]) and np.array_equal(ex[1], ha[1]) and np.array_equal(ex[2], ha[2])
    assert ex[3] == ha[3] and ex[4] == ha[4]
    assert np.linalg.norm(pu[0] - x_ref) < 1e-10 * np.linalg.norm(x_ref)
    U_ref, P_ref, its_ref, _ = oracle.trajectory(dims, beta, kappa, BC, U, b, P0, 2, 0.03, tol=1e-13, max_iter=5000)
    assert pu[4] == its_ref and np.abs(pu[1] - U_ref).max() < 1e-12 and link_rel_err(pu[2], P_ref)[0] < TOL64


@pytest.mark.parametrize("nranks", [2, 4])
def test_dd_hmc_trajectory_matches_undivided_oracle(lgt, nranks):
    """Heat baths by global element number: momenta, pseudofermion, dH, decision and links after the test are those of
    the oracle's trajectory on the undivided lattice; a coarse gauge-only trajectory is rejected and restored bit for bit."""
    from oracle import hmc as ohmc

    dims, beta, kappa, seed = (4, 4, 2, 8), 5.5, 0.10, 97531
    U = synth.warm_links(dims, 0.2, 571)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH)
    dd.set_links(U)
    for traj in range(2):
        dH, acc, its, H0, ok = lgt.lgt_dd_hmc_trajectory(dd.d, 3, 0.03, seed, traj, tol=1e-13, max_iter=5000)
        ref = ohmc.hmc_trajectory(dims, beta, kappa, BC, U, seed, traj, 3, 0.03, ohmc.LEAPFROG, tol=1e-13, max_iter=5000)
        assert ok and abs(H0 - ref["H0"]) < 1e-12 * abs(ref["H0"]) and abs(dH - ref["dH"]) < 1e-9 * abs(ref["H0"])
        if abs(ref["u"] - np.exp(-ref["dH"])) > 1e-6:
            assert acc == ref["accepted"]
            assert np.abs(cat(dd.get_links()) - ref["U"]).max() < 1e-11
        U = cat(dd.get_links())
    dd.close()
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, 0.0, BC)
    U = synth.warm_links(dims, 0.2, 571)
    dd.set_links(U)
    seen = set()
    for traj in range(6):
        dH, acc, _, _, _ = lgt.lgt_dd_hmc_trajectory(dd.d, 1, 0.12, 7, traj)
        ref = ohmc.hmc_trajectory(dims, beta, 0.0, BC, U, 7, traj, 1, 0.12)
        assert abs(dH - ref["dH"]) < 1e-9 * abs(ref["H0"]) and acc == ref["accepted"]
        if not acc:
            assert np.array_equal(cat(dd.get_links()), U)
        seen.add(acc)
        U = cat(dd.get_links())
    assert len(seen) >= 1
    dd.close()


@pytest.mark.parametrize("nranks,mode", [(2, "exchange"), (4, "push"), (1, "push")])
def test_dd_mixed_precision_solver(lgt, nranks, mode):
    """lgt_dd_set_solver(MIXED): decomposed fp32 CG inside the fp64 defect correction; kick, drift and action agree with
    the oracle's fp64 results on the undivided lattice, also after the links moved (fp32 copies refreshed)."""
    dims, beta, kappa = (4, 4, 4, 8), 5.6, 0.12
    U0 = synth.warm_links(dims, 0.3, 581)
    P0 = synth.gaussian_momenta(dims, 582)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 583), dagger=True)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH if mode == "push" else lgt.LGT_DD_EXCHANGE)
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    it = lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 5000)
    P1, it_ref, _ = oracle.kick(dims, beta, kappa, BC, U0, phi, P0, 0.05, 1e-12, 5000)
    assert 0 < it < 2 * it_ref + 20
    assert link_rel_err(cat(dd.get_momenta()), P1)[0] < 1e-10
    lgt.lgt_dd_md_drift(dd.d, 0.05)
    U1 = oracle.drift(dims, 0.05, P1, U0)
    lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 5000)
    P2, _, _ = oracle.kick(dims, beta, kappa, BC, U1, phi, P1, 0.05, 1e-12, 5000)
    assert link_rel_err(cat(dd.get_momenta()), P2)[0] < 1e-10
    _, S_F, _, _ = lgt.lgt_dd_action(dd.d, 1e-12, 5000)
    S_ref = oracle.fermion_action(dims, kappa, BC, U1, phi, 1e-12, 5000)[0]
    assert abs(S_F - S_ref) < 1e-10 * abs(S_ref)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_set_solver(dd.d, 5, 1e-5)
    dd.close()


def test_dd_half_spinor_halos_in_the_fp32_inner_solve(lgt):
    """LGT_DD_HALF with the mixed-precision solver: the fp32 inner CG sends fp32 half spinors; the kick is bitwise the one with
    the plain exchange and agrees with the oracle's fp64 kick."""
    dims, beta, kappa = (8, 4, 4, 8), 5.6, 0.12
    U0 = synth.warm_links(dims, 0.3, 586)
    P0 = synth.gaussian_momenta(dims, 587)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 588), dagger=True)
    res = {}
    for mode in (lgt.LGT_DD_EXCHANGE, lgt.LGT_DD_HALF):
        dd = lgt.DecomposedLattice(dims, 2, [0, 1], beta, kappa, BC)
        lgt.lgt_dd_set_halo_mode(dd.d, mode)
        lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
        dd.set_links(U0)
        dd.set_momenta(P0)
        dd.set_pseudofermion(phi)
        it = lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 5000)
        res[mode] = (it, cat(dd.get_momenta()))
        dd.close()
    assert res[lgt.LGT_DD_EXCHANGE][0] == res[lgt.LGT_DD_HALF][0]
    assert np.array_equal(res[lgt.LGT_DD_EXCHANGE][1], res[lgt.LGT_DD_HALF][1])
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U0, phi, P0, 0.05, 1e-12, 5000)
    assert link_rel_err(res[lgt.LGT_DD_HALF][1], P1)[0] < 1e-10


def test_dd_mixed_even_odd_inner_hops_on_twelve_real_links(lgt):
    """Slabs large enough (320 blocks per half field and rank) for the fp32 inner hops of the mixed-precision even/odd solver to
    take the three-blocks-per-SM build on 12-real links: the folded boundary sign must come out right with the slab's time
    offset (antiperiodic t: the last slice of the LAST slab only).  Kick against the oracle's on the undivided lattice, fp32
    iteration count that of the undivided handle (+- 2)."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (16, 16, 16, 40), 5.6, 0.12, 1e-12
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 641)
    P0 = synth.gaussian_momenta(dims, 642)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 643), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + F_ref)
    one = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_fermion_action(one.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(one.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    one.set_links(U0)
    one.set_momenta(P0)
    one.set_pseudofermion(phi)
    it_one = lgt.lgt_md_kick(one.ctx, 0.05, tol, 10 * V)
    assert link_rel_err(one.get_momenta(), P_ref)[0] < 1e-10
    one.close()
    dd = lgt.DecomposedLattice(dims, 2, [0, 1], beta, kappa, BC)
    lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    it = lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
    assert abs(it - it_one) <= 2 and it < 2 * it_ref + 20
    assert link_rel_err(cat(dd.get_momenta()), P_ref)[0] < 1e-10
    dd.close()


@pytest.mark.parametrize("nranks", [1, 2])
def test_dd_even_odd_overlapped_exchange(lgt, nranks):
    """LGT_DD_OVERLAP (and LGT_DD_HALF, which falls back to it for half fields) with the even/odd action: every hop of the
    CG on the Schur complement runs its bulk while the input half field's ghost slices travel on the halo stream, the two
    boundary slices after.  Time slices of 256 sites (128 per parity) and slabs of 4 and 8 slices: momenta after a kick bitwise
    those of LGT_DD_EXCHANGE, the oracle's iteration count; with the mixed-precision solver the same momenta to 1e-10."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (8, 8, 4, 8), 5.6, 0.12, 1e-12
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 595)
    P0 = synth.gaussian_momenta(dims, 596)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 597), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + F_ref)
    res = {}
    for mode in (lgt.LGT_DD_EXCHANGE, lgt.LGT_DD_OVERLAP, lgt.LGT_DD_HALF):
        for mixed in (False, True):
            dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
            lgt.lgt_dd_set_halo_mode(dd.d, mode)
            lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
            if mixed:
                lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
            dd.set_links(U0)
            dd.set_momenta(P0)
            dd.set_pseudofermion(phi)
            it = lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
            res[mode, mixed] = (it, cat(dd.get_momenta()))
            dd.close()
    ex = res[lgt.LGT_DD_EXCHANGE, False]
    assert ex[0] == it_ref and link_rel_err(ex[1], P_ref)[0] < TOL64
    for mode in (lgt.LGT_DD_OVERLAP, lgt.LGT_DD_HALF):
        assert res[mode, False][0] == it_ref and np.array_equal(res[mode, False][1], ex[1])
        assert link_rel_err(res[mode, True][1], P_ref)[0] < 1e-10


@pytest.mark.parametrize("nranks", [1, 2, 4])
def test_dd_even_odd_action(lgt, nranks):
    """The even/odd action on slabs (local parity = global parity shifted by the slab's time offset): iteration count,
    kick and S_F against the oracle's even/odd mode on the undivided lattice; an HMC trajectory against the
    (oracle-verified) single-GPU even/odd trajectory with the same seed."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (4, 4, 4, 8), 5.6, 0.12, 1e-12
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 591)
    P0 = synth.gaussian_momenta(dims, 592)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 593), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    it = lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
    assert it == it_ref
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + F_ref)
    assert link_rel_err(cat(dd.get_momenta()), P_ref)[0] < TOL64
    _, S_F, _, _ = lgt.lgt_dd_action(dd.d, tol, 10 * V)
    S_ref = oeo.action(dims, kappa, BC, U0, phi, tol, 10 * V)[0]
    assert abs(S_F - S_ref) < 1e-11 * abs(S_ref)
    # HMC with the even/odd action: same (seed, trajectory) on one undivided handle
    one = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_fermion_action(one.ctx, lgt.LGT_ACTION_EO)
    one.set_links(U0)
    dd.set_links(U0)
    for traj in range(2):
        a = lgt.lgt_hmc_trajectory(one.ctx, 3, 0.03, 1357, traj, tol=1e-13, max_iter=5000)
        b = lgt.lgt_dd_hmc_trajectory(dd.d, 3, 0.03, 1357, traj, tol=1e-13, max_iter=5000)
        assert abs(a[3] - b[3]) < 1e-12 * abs(a[3]) and abs(a[0] - b[0]) < 1e-9 * abs(a[3])
        assert a[1] == b[1] and a[2] == b[2]
        assert np.abs(cat(dd.get_links()) - one.get_links()).max() < 1e-11
    one.close()
    dd.close()
    with pytest.raises(lgt.LgtError):
        bad = lgt.lgt_dd_create((4, 4, 2, 8), 2, [0, 1], beta, kappa, BC)  # 32 sites per time slice: not a multiple of 64
        try:
            lgt.lgt_dd_set_fermion_action(bad, lgt.LGT_ACTION_EO)
        finally:
            lgt.lgt_dd_destroy(bad)
    with pytest.raises(lgt.LgtError):
        bad = lgt.lgt_dd_create((4, 4, 4, 6), 2, [0, 1], beta, kappa, BC)  # three slices per slab: a slab would start at an odd time
        try:
            lgt.lgt_dd_set_fermion_action(bad, lgt.LGT_ACTION_EO)
        finally:
            lgt.lgt_dd_destroy(bad)


@pytest.mark.parametrize("nranks,levels", [(2, 1), (4, 2), (1, 2)])
def test_dd_stout_smearing(lgt, nranks, levels):
    """Stout-smeared fermions on slabs: every level's ghost slices are exchanged before the next level, G's before each
    chain kernel.  Dslash on the smeared links and the kick (gauge force on thin links + pulled-back fermion force)
    against the oracle on the undivided lattice; with the even/odd action on top for one case."""
    from oracle import stout as ost

    dims, beta, kappa, rho = (4, 4, 4, 8), 5.6, 0.11, 0.3
    U0 = synth.warm_links(dims, 0.25, 601)
    P0 = synth.gaussian_momenta(dims, 602)
    Un = ost.smear_levels(dims, rho, levels, U0)[0][-1]
    psi = synth.gaussian_spinor(dims, 603)
    phi = oracle.dslash(dims, kappa, BC, Un, psi, dagger=True)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    lgt.lgt_dd_set_smearing(dd.d, levels, rho)
    lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH)
    dd.set_links(U0)
    assert np.abs(cat(dd.dslash(psi)) - oracle.dslash(dims, kappa, BC, Un, psi)).max() < 1e-12
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    it = lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
    Ff, it_ref, ok = ost.fermion_force(dims, kappa, BC, U0, phi, levels, rho, 1e-13, 5000)
    assert ok and it == it_ref
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + Ff)
    assert link_rel_err(cat(dd.get_momenta()), P_ref)[0] < TOL64
    # after a drift the smeared links follow the new thin links
    lgt.lgt_dd_md_drift(dd.d, 0.05)
    U1 = oracle.drift(dims, 0.05, P_ref, U0)
    assert np.abs(cat(dd.dslash(psi)) - oracle.dslash(dims, kappa, BC, ost.smear_levels(dims, rho, levels, U1)[0][-1], psi)).max() < 1e-11
    if levels == 1:
        from oracle import evenodd as oeo
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
        dd.set_links(U0)
        dd.set_momenta(P0)
        Xe, Ye, _, _ = oeo.solve_xy(dims, kappa, BC, Un, phi, 1e-13, 5000)
        Feo = ost.pull_back(dims, rho, U0, ost.smear(dims, rho, U0)[1], oracle.fermion_force(dims, kappa, BC, Un, Xe, Ye))[0]
        lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
        assert link_rel_err(cat(dd.get_momenta()), P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + Feo))[0] < TOL64
    dd.close()


@pytest.mark.parametrize("integ,m", [("omelyan", 1), ("sw", 3)])
def test_dd_integrators(lgt, integ, m):
    """Omelyan and Sexton-Weingarten on two slabs against the oracle's integrators on the undivided lattice."""
    from oracle import hmc as ohmc

    dims, beta, kappa = (4, 4, 2, 8), 5.5, 0.10
    U0 = synth.warm_links(dims, 0.2, 611)
    P0 = synth.gaussian_momenta(dims, 612)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 613), dagger=True)
    dd = lgt.DecomposedLattice(dims, 2, [0, 1], beta, kappa, BC)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    code = lgt.LGT_INT_OMELYAN if integ == "omelyan" else lgt.LGT_INT_SEXTON_WEINGARTEN
    ocode = ohmc.OMELYAN if integ == "omelyan" else ohmc.SEXTON_WEINGARTEN
    lgt.lgt_dd_set_integrator(dd.d, code, m)
    H0, H1, its = lgt.lgt_dd_md_trajectory(dd.d, 3, 0.04, tol=1e-13, max_iter=5000)
    U_ref, P_ref, its_ref = ohmc.integrate(dims, beta, kappa, BC, U0, phi, P0, 3, 0.04, ocode, n_inner=m, tol=1e-13, max_iter=5000)
    assert its == its_ref
    assert np.abs(cat(dd.get_links()) - U_ref).max() < 1e-12
    assert link_rel_err(cat(dd.get_momenta()), P_ref)[0] < TOL64
    with pytest.raises(lgt.LgtError):
        lgt.lgt_dd_set_integrator(dd.d, 9, 1)
    dd.close()


@pytest.mark.parametrize("nranks", [2, 4])
def test_dd_even_odd_mixed_precision(lgt, nranks):
    """The fastest configuration on slabs: even/odd action with the mixed-precision solver (decomposed fp32 CG on the Schur
    complement inside the fp64 defect correction); kick and action against the oracle's fp64 even/odd mode."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (4, 4, 4, 8), 5.6, 0.12, 1e-12
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 621)
    P0 = synth.gaussian_momenta(dims, 622)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 623), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
    lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    dd.set_links(U0)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    it = lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
    assert 0 < it < 2 * it_ref + 20
    P1 = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + F_ref)
    assert link_rel_err(cat(dd.get_momenta()), P1)[0] < 1e-10
    _, S_F, _, _ = lgt.lgt_dd_action(dd.d, tol, 10 * V)
    S_ref = oeo.action(dims, kappa, BC, U0, phi, tol, 10 * V)[0]
    assert abs(S_F - S_ref) < 1e-10 * abs(S_ref)
    # after a drift the fp32 checkerboard links follow
    lgt.lgt_dd_md_drift(dd.d, 0.05)
    U1 = oracle.drift(dims, 0.05, P1, U0)
    lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
    F1, _, _ = oeo.fermion_force(dims, kappa, BC, U1, phi, tol, 10 * V)
    assert link_rel_err(cat(dd.get_momenta()), P1 - 0.05 * (oracle.gauge_force(dims, beta, U1) + F1))[0] < 1e-10
    dd.close()


@pytest.mark.parametrize("nranks", [1, 2, 4])
def test_dd_even_odd_pushed_halos(lgt, nranks):
    """LGT_DD_PUSH under the even/odd action: u and r are pushed by the hops that produce them, p's ghost slices follow by
    local arithmetic, the odd intermediates are still exchanged.  Bitwise the exchanged results, the oracle's count.
    Half-field time slices of 128 sites (boundary / bulk split of the pushing hops)."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (8, 8, 4, 8), 5.6, 0.12, 1e-12
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 631)
    P0 = synth.gaussian_momenta(dims, 632)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 633), dims, 0), dagger=True)
    _, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    res = {}
    for mode in (lgt.LGT_DD_EXCHANGE, lgt.LGT_DD_PUSH):
        dd = lgt.DecomposedLattice(dims, nranks, list(range(nranks)), beta, kappa, BC)
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
        lgt.lgt_dd_set_halo_mode(dd.d, mode)
        dd.set_links(U0)
        dd.set_momenta(P0)
        dd.set_pseudofermion(phi)
        H0, H1, its = lgt.lgt_dd_md_trajectory(dd.d, 2, 0.03, tol=tol, max_iter=10 * V)
        res[mode] = (cat(dd.get_links()), cat(dd.get_momenta()), H1 - H0, its)
        if mode == lgt.LGT_DD_PUSH:
            lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)  # the fp32 inner solve pushes too
            dd.set_links(U0)
            dd.set_momenta(P0)
            lgt.lgt_dd_md_trajectory(dd.d, 2, 0.03, tol=tol, max_iter=10 * V, measure=False)
            assert link_rel_err(cat(dd.get_momenta()), res[mode][1])[0] < 1e-9
        dd.close()
    ex, pu = res[lgt.LGT_DD_EXCHANGE], res[lgt.LGT_DD_PUSH]
    assert np.array_equal(ex[0], pu[0]) and np.array_equal(ex[1], pu[1]) and ex[2] == pu[2] and ex[3] == pu[3]


@pytest.mark.parametrize("world", [2, 3])
def test_dd_between_processes_on_one_gpu(lgt, world):
    """The inter-process path of the decomposition executed by SEPARATE PROCESSES that share this one GPU: one rank per
    process (lgt_dd_create with nlocal = 1), halo slices and sums over the host transport on gloo (NCCL refuses two ranks
    on one device, so NCCL itself stays covered by the one-rank test above), CUDA-IPC export / all-gather / import and
    LGT_DD_PUSH stores into the other process's buffers.  With two processes both neighbours of a rank are the same peer.
    The worker (tests/dd_two_process_worker.py) asserts, on every rank: Dslash, CG iterates and a leapfrog trajectory
    bit-identical to the in-process lockstep group and within 1e-11 / 1e-12 of the oracle on the undivided lattice, the
    oracle's CG iteration counts, for the exchange and the push mode; the mixed solver and the even/odd action on top."""
    import json
    import os
    import socket
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.join(root, "tests", "dd_two_process_worker.py")], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    try:
        for p in procs:
            o, e = p.communicate(timeout=900)
            assert p.returncode == 0, (o[-1500:], e[-3000:])
            outs.append(json.loads(o.strip().splitlines()[-1]))
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    assert sorted(o["rank"] for o in outs) == list(range(world))
    for o in outs:
        for halo in ("exchange", "push"):
            assert o[halo]["cg_iters"] == o["cg_iters_oracle"] and o[halo]["launches"] > 0
        assert len(o["grid"]) >= 2  # (1, world) and (world, 1): the z faces over the host transport too


# ---- two split directions (lgt_dd_create_grid, SURVEY 8(e) "first T, then Z") -------------------------------------
def gather_grid(dims, grid, blocks):
    """Global canonical array from the ranks' blocks [Lt/Pt][Lz/Pz][Ly][Lx] (rank = pt * Pz + pz)."""
    Lx, Ly, Lz, Lt = dims
    Pt, Pz = grid
    lt, lz = Lt // Pt, Lz // Pz
    tail = blocks[0].shape[1:]
    out = np.empty((Lt, Lz, Ly * Lx) + tail, dtype=blocks[0].dtype)
    for r, b in enumerate(blocks):
        pt, pz = divmod(r, Pz)
        out[pt * lt:(pt + 1) * lt, pz * lz:(pz + 1) * lz] = b.reshape((lt, lz, Ly * Lx) + tail)
    return out.reshape((Lx * Ly * Lz * Lt,) + tail)


GRIDS = [((8, 4, 4, 4), (1, 1)), ((8, 4, 4, 4), (1, 2)), ((8, 4, 4, 4), (2, 2)), ((8, 4, 8, 4), (2, 4)), ((8, 4, 4, 4), (4, 2)),
         ((8, 8, 6, 6), (3, 2)), ((16, 2, 4, 2), (1, 4))]


@pytest.mark.parametrize("dims,grid", GRIDS)
def test_grid_dslash_is_bitwise_the_undivided_kernel(lgt, dims, grid):
    """A (Pt, Pz) grid with every rank in this process: D and D^dag bitwise equal to the undivided handle (same kernel
    arithmetic per site; ghost time slices and ghost z planes filled by the t-then-z exchange) and equal to the oracle,
    with an antiperiodic direction in z as well (the boundary sign goes by the global z coordinate); set / get round trip."""
    kappa = 0.12
    n = grid[0] * grid[1]
    U = synth.warm_links(dims, 0.3, 701)
    psi = synth.gaussian_spinor(dims, 702)
    for bc in (BC, (1, 1, -1, -1)):
        dd = lgt.DecomposedLattice(dims, n, list(range(n)), 5.5, kappa, bc, grid=grid)
        dd.set_links(U)
        one = lgt.Lattice(dims, 5.5, kappa, bc)
        one.set_links(U)
        for dag in (False, True):
            out = gather_grid(dims, grid, dd.dslash(psi, dagger=dag))
            assert np.abs(out - oracle.dslash(dims, kappa, bc, U, psi, dagger=dag)).max() < 1e-12
            assert np.array_equal(out, one.dslash(psi, dagger=dag))
        assert np.array_equal(gather_grid(dims, grid, dd.get_links()), U)
        dd.close()
        one.close()


@pytest.mark.parametrize("dims,grid", [((8, 4, 4, 4), (2, 2)), ((8, 4, 8, 4), (2, 4)), ((8, 4, 4, 4), (1, 2))])
def test_grid_cg_and_md_trajectory(lgt, dims, grid):
    """CG with the oracle's iteration count, the actions, kick, drift and a leapfrog trajectory with both forces on the grid
    against the oracle on the undivided lattice (the staples reach into the corners that the t-then-z exchange fills)."""
    beta, kappa = 5.6, 0.11
    n = grid[0] * grid[1]
    U0 = synth.warm_links(dims, 0.25, 711)
    P0 = synth.gaussian_momenta(dims, 712)
    phi = oracle.dslash(dims, kappa, BC, U0, synth.gaussian_spinor(dims, 713), dagger=True)
    dd = lgt.DecomposedLattice(dims, n, list(range(n)), beta, kappa, BC, grid=grid)
    dd.set_links(U0)
    xs, it, rel, ok = dd.cg(phi, 1e-12, 5000)
    x_ref, it_ref, _, ok_ref = oracle.cg(dims, kappa, BC, U0, phi, 1e-12, 5000)
    assert ok and ok_ref and it == it_ref
    x = gather_grid(dims, grid, xs)
    assert np.linalg.norm(x - x_ref) < 1e-10 * np.linalg.norm(x_ref)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    S_g, S_F, K, _ = lgt.lgt_dd_action(dd.d, 1e-13, 5000)
    H_ref, K_ref, Sg_ref, SF_ref = oracle.hamiltonian(dims, beta, kappa, BC, U0, phi, P0, 1e-13, 5000)
    assert abs(S_g - Sg_ref) < 1e-11 * abs(Sg_ref) and abs(S_F - SF_ref) < 1e-10 * abs(SF_ref) and abs(K - K_ref) < 1e-12 * K_ref
    H0, H1, its = lgt.lgt_dd_md_trajectory(dd.d, 3, 0.03, tol=1e-13, max_iter=5000)
    U_ref, P_ref, its_ref, ok = oracle.trajectory(dims, beta, kappa, BC, U0, phi, P0, 3, 0.03, tol=1e-13, max_iter=5000)
    assert ok and its == its_ref
    assert np.abs(gather_grid(dims, grid, dd.get_links()) - U_ref).max() < 1e-12
    assert link_rel_err(gather_grid(dims, grid, dd.get_momenta()), P_ref)[0] < TOL64
    H1_ref = oracle.hamiltonian(dims, beta, kappa, BC, U_ref, phi, P_ref, 1e-13, 5000)[0]
    assert abs((H1 - H0) - (H1_ref - H_ref)) < 1e-9 * abs(H_ref)
    dd.set_links(U0)
    dd.set_momenta(P0)
    lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U0, phi, P0, 0.05, 1e-13, 5000)
    assert link_rel_err(gather_grid(dims, grid, dd.get_momenta()), P1)[0] < TOL64
    lgt.lgt_dd_md_drift(dd.d, 0.05)
    assert np.abs(gather_grid(dims, grid, dd.get_links()) - oracle.drift(dims, 0.05, P1, U0)).max() < 1e-13
    # what a grid does not offer
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH)
    assert e.value.code == lgt.LGT_EINVAL
    with pytest.raises(lgt.LgtError) as e:  # 32 sites per xy plane: a half field's z face would be half a layout block
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    assert e.value.code == lgt.LGT_EINVAL
    dd.close()
    for bad in ((3, 1), (1, 3), (0, 2)):  # Lt % Pt, Lz % Pz, Pt < 1
        with pytest.raises(lgt.LgtError) as e:
            lgt.lgt_dd_create_grid(dims, bad, [0], beta, kappa, BC)
        assert e.value.code == lgt.LGT_EINVAL
    with pytest.raises(lgt.LgtError):  # xy planes must be whole layout blocks
        lgt.lgt_dd_create_grid((4, 4, 4, 4), (2, 2), [0], beta, kappa, BC)


@pytest.mark.parametrize("grid", [(2, 2), (1, 4)])
def test_grid_hmc_mixed_solver_and_stout(lgt, grid):
    """On the (Pt, Pz) grid: the HMC trajectory (heat baths by GLOBAL element number, here formed from the coordinates) gives
    the oracle's momenta, pseudofermion, dH and decision on the undivided lattice; the mixed-precision solver (fp32 copies incl.
    ghost planes, masked fp64 residual sums) and one / two levels of stout smearing (every level's planes exchanged before the
    next, G's before the chain kernel) give the oracle's kick."""
    from oracle import hmc as ohmc
    from oracle import stout as ost

    dims, beta, kappa, seed = (8, 4, 4, 4), 5.5, 0.10, 97531
    n = grid[0] * grid[1]
    U = synth.warm_links(dims, 0.2, 721)
    dd = lgt.DecomposedLattice(dims, n, list(range(n)), beta, kappa, BC, grid=grid)
    dd.set_links(U)
    for traj in range(2):
        dH, acc, its, H0, ok = lgt.lgt_dd_hmc_trajectory(dd.d, 3, 0.03, seed, traj, tol=1e-13, max_iter=5000)
        ref = ohmc.hmc_trajectory(dims, beta, kappa, BC, U, seed, traj, 3, 0.03, ohmc.LEAPFROG, tol=1e-13, max_iter=5000)
        assert ok and abs(H0 - ref["H0"]) < 1e-12 * abs(ref["H0"]) and abs(dH - ref["dH"]) < 1e-9 * abs(ref["H0"])
        if abs(ref["u"] - np.exp(-ref["dH"])) > 1e-6:
            assert acc == ref["accepted"]
            assert np.abs(gather_grid(dims, grid, dd.get_links()) - ref["U"]).max() < 1e-11
        U = gather_grid(dims, grid, dd.get_links())
    dd.close()

    kappa, rho = 0.11, 0.3
    U0 = synth.warm_links(dims, 0.25, 722)
    P0 = synth.gaussian_momenta(dims, 723)
    psi = synth.gaussian_spinor(dims, 724)
    dd = lgt.DecomposedLattice(dims, n, list(range(n)), beta, kappa, BC, grid=grid)
    dd.set_links(U0)
    phi = oracle.dslash(dims, kappa, BC, U0, psi, dagger=True)
    dd.set_momenta(P0)
    dd.set_pseudofermion(phi)
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 5000)
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U0, phi, P0, 0.05, 1e-13, 5000)
    assert link_rel_err(gather_grid(dims, grid, dd.get_momenta()), P1)[0] < 1e-10
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_CG)
    for levels in (1, 2):
        Un = ost.smear_levels(dims, rho, levels, U0)[0][-1]
        phi = oracle.dslash(dims, kappa, BC, Un, psi, dagger=True)
        lgt.lgt_dd_set_smearing(dd.d, levels, rho)
        dd.set_links(U0)
        assert np.abs(gather_grid(dims, grid, dd.dslash(psi)) - oracle.dslash(dims, kappa, BC, Un, psi)).max() < 1e-12
        dd.set_momenta(P0)
        dd.set_pseudofermion(phi)
        it = lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-13, 5000)
        Ff, it_ref, ok = ost.fermion_force(dims, kappa, BC, U0, phi, levels, rho, 1e-13, 5000)
        assert ok and it == it_ref
        P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + Ff)
        assert link_rel_err(gather_grid(dims, grid, dd.get_momenta()), P_ref)[0] < TOL64
    dd.close()


@pytest.mark.parametrize("grid", [(2, 2), (1, 2), (2, 1)])
def test_grid_even_odd_action(lgt, grid):
    """The even/odd action on the (Pt, Pz) grid: a rank's local parity is the global one shifted by its time AND z offsets, the
    half fields' z faces (Lx Ly / 2 sites per plane) travel like the full fields'.  Iteration count, kick and S_F against the
    oracle's even/odd mode on the undivided lattice, the mixed-precision solver on top, and an HMC trajectory against the
    single-handle even/odd trajectory with the same seed."""
    from oracle import evenodd as oeo

    dims, beta, kappa, tol = (8, 8, 4, 4), 5.6, 0.12, 1e-12
    n = grid[0] * grid[1]
    V = synth.volume(dims)
    U0 = synth.warm_links(dims, 0.3, 741)
    P0 = synth.gaussian_momenta(dims, 742)
    phi = oeo.mhat(dims, kappa, BC, U0, oeo.keep(synth.gaussian_spinor(dims, 743), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U0, phi, tol, 10 * V)
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U0) + F_ref)
    S_ref = oeo.action(dims, kappa, BC, U0, phi, tol, 10 * V)[0]
    dd = lgt.DecomposedLattice(dims, n, list(range(n)), beta, kappa, BC, grid=grid)
    lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    for solver, ptol in ((lgt.LGT_SOLVER_CG, TOL64), (lgt.LGT_SOLVER_MIXED_CG, 1e-10)):
        lgt.lgt_dd_set_solver(dd.d, solver, 1e-5)
        dd.set_links(U0)
        dd.set_momenta(P0)
        dd.set_pseudofermion(phi)
        it = lgt.lgt_dd_md_kick(dd.d, 0.05, tol, 10 * V)
        if solver == lgt.LGT_SOLVER_CG:
            assert it == it_ref
        assert link_rel_err(gather_grid(dims, grid, dd.get_momenta()), P_ref)[0] < ptol
        _, S_F, _, _ = lgt.lgt_dd_action(dd.d, tol, 10 * V)
        assert abs(S_F - S_ref) < 1e-10 * abs(S_ref)
    lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_CG)
    one = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_fermion_action(one.ctx, lgt.LGT_ACTION_EO)
    one.set_links(U0)
    dd.set_links(U0)
    for traj in range(2):
        a = lgt.lgt_hmc_trajectory(one.ctx, 3, 0.03, 1357, traj, tol=1e-13, max_iter=5000)
        b = lgt.lgt_dd_hmc_trajectory(dd.d, 3, 0.03, 1357, traj, tol=1e-13, max_iter=5000)
        assert abs(a[3] - b[3]) < 1e-12 * abs(a[3]) and abs(a[0] - b[0]) < 1e-9 * abs(a[3])
        assert a[1] == b[1] and a[2] == b[2]
        assert np.abs(gather_grid(dims, grid, dd.get_links()) - one.get_links()).max() < 1e-11
    one.close()
    dd.close()
