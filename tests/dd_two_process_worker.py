"""Worker of tests/test_gpu_dd.py::test_dd_between_processes_on_one_gpu (not a test module itself).

One rank of a time-slab group per PROCESS, all processes on cuda:0, launched with RANK / WORLD_SIZE / MASTER_* in the
environment.  NCCL refuses two ranks on one device, so the transport is the library's host transport over gloo
(lgt_dd_set_host_transport); everything else is the production inter-process path: lgt_dd_create(nlocal = 1), the halo
plan between distinct peers (with two processes both neighbours are the same peer), lgt_dd_ipc_export -> all-gather ->
lgt_dd_ipc_import, LGT_DD_PUSH stores into the other process's memory.  No kernel ever waits on another process: the
ranks meet only in host-side gloo calls after a stream synchronisation.
Every rank checks its slab against the oracle on the undivided lattice and, bit for bit, against the in-process
lockstep group of the same shape; prints one JSON line.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import oracle  # noqa: E402
from lattice_util import link_rel_err  # noqa: E402
from paper_2602_20516_b200 import dist, lgt, synth  # noqa: E402

BC = (1, 1, 1, -1)


def main():
    import torch

    rank, world = dist.init("gloo")
    torch.cuda.set_device(0)
    lgt.lib()
    dims, beta, kappa = (8, 4, 4, 2 * world), 5.6, 0.12  # 128 sites per time slice: the pushing kernels run
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 601)
    P0 = synth.gaussian_momenta(dims, 602)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 603), dagger=True)
    x_ref, it_ref, _, ok = oracle.cg(dims, kappa, BC, U, b, 1e-12, 5000)
    assert ok
    lo, hi = dist.slab_rows(dims, world, rank)
    out = {"rank": rank, "world": world, "cg_iters_oracle": it_ref}

    # a one-of-several-ranks group without a transport must refuse, not read through a wild pointer
    bare = lgt.DecomposedLattice(dims, world, [rank], beta, kappa, BC)
    for call in (lambda: lgt.lgt_dd_md_drift(bare.d, 0.01), lambda: lgt.lgt_dd_action(bare.d), lambda: bare.dslash(b)):
        try:
            call()
            raise AssertionError("no transport, but the call went through")
        except lgt.LgtError as e:
            assert e.code == lgt.LGT_ESTATE, e
    bare.close()

    # the same group shape with every rank in this process: the bitwise reference for this rank's slab
    ref = lgt.DecomposedLattice(dims, world, list(range(world)), beta, kappa, BC)
    ref.set_links(U)
    ref_ds = ref.dslash(b)[rank]
    ref_x, ref_it, _, _ = ref.cg(b, 1e-12, 5000)
    ref.set_momenta(P0)
    ref.set_pseudofermion(b)
    ref_traj = lgt.lgt_dd_md_trajectory(ref.d, 2, 0.03, tol=1e-13, max_iter=5000)
    ref_U, ref_P = ref.get_links()[rank], ref.get_momenta()[rank]
    ref.close()
    U_ref, P_ref, its_ref, _ = oracle.trajectory(dims, beta, kappa, BC, U, b, P0, 2, 0.03, tol=1e-13, max_iter=5000)

    for halo in ("exchange", "push"):
        dd = dist.decomposed_lattice(dims, beta, kappa, BC, lgt.LGT_F64, 0, None, halo=halo, transport="host")
        assert lgt.lgt_dd_local_ranks(dd.d) == 1 and dd.local_ranks == [rank]
        dd.set_links(U)
        ds = dd.dslash(b)[0]
        assert np.abs(ds - oracle.dslash(dims, kappa, BC, U, b)[lo:hi]).max() < 1e-12
        assert np.array_equal(ds, ref_ds)
        xs, it, rel, ok = dd.cg(b, 1e-12, 5000)
        assert ok and it == it_ref == ref_it, (it, it_ref, ref_it)
        assert np.array_equal(xs[0], ref_x[rank])  # same iterates bit for bit as the lockstep group, in both halo modes
        assert np.linalg.norm(xs[0] - x_ref[lo:hi]) < 1e-10 * np.linalg.norm(x_ref[lo:hi])
        dd.set_momenta(P0)
        dd.set_pseudofermion(b)
        traj = lgt.lgt_dd_md_trajectory(dd.d, 2, 0.03, tol=1e-13, max_iter=5000)
        assert traj == ref_traj and traj[2] == its_ref
        Uo, Po = dd.get_links()[0], dd.get_momenta()[0]
        assert np.array_equal(Uo, ref_U) and np.array_equal(Po, ref_P)
        assert np.abs(Uo - U_ref[lo:hi]).max() < 1e-12 and link_rel_err(Po, P_ref[lo:hi])[0] < 1e-11
        # mixed-precision solver and the even/odd action over the same transport (their fp32 / half fields are not
        # IPC-mapped: in push mode they fall back to the exchange, the fp64 full-field CG keeps pushing)
        dd.set_links(U)
        dd.set_momenta(P0)
        lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
        lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 5000)
        P1, _, _ = oracle.kick(dims, beta, kappa, BC, U, b, P0, 0.05, 1e-12, 5000)
        assert link_rel_err(dd.get_momenta()[0], P1[lo:hi])[0] < 1e-10
        lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_CG)
        from oracle import evenodd as oeo

        phi_e = oeo.mhat(dims, kappa, BC, U, oeo.keep(synth.gaussian_spinor(dims, 604), dims, 0), dagger=True)
        F_eo, it_eo, _ = oeo.fermion_force(dims, kappa, BC, U, phi_e, 1e-12, 10 * V)
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
        dd.set_momenta(P0)
        dd.set_pseudofermion(phi_e)
        assert lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 10 * V) == it_eo
        P_eo = P0 - 0.05 * (oracle.gauge_force(dims, beta, U) + F_eo)
        assert link_rel_err(dd.get_momenta()[0], P_eo[lo:hi])[0] < 1e-11
        out[halo] = {"cg_iters": it, "md_cg_iters": traj[2], "eo_cg_iters": it_eo, "launches": lgt.lgt_launch_count(dd.ranks[0])}
        dd.close()
        dist.barrier()
    # LGT_DD_OVERLAP between processes: slabs of four slices, the exchange (host transport, on the group's halo stream) under
    # the bulk kernel, boundary slices after it; bitwise the plain exchange
    odims = (8, 4, 4, 4 * world)
    oU = synth.warm_links(odims, 0.3, 621)
    ob = oracle.dslash(odims, kappa, BC, oU, synth.gaussian_spinor(odims, 622), dagger=True)
    _, oit_ref, _, ook = oracle.cg(odims, kappa, BC, oU, ob, 1e-12, 5000)
    ores = {}
    for halo in ("exchange", "overlap", "half"):
        dd = dist.decomposed_lattice(odims, beta, kappa, BC, lgt.LGT_F64, 0, None, halo=halo, transport="host")
        dd.set_links(oU)
        xs, it, rel, ok = dd.cg(ob, 1e-12, 5000)
        assert ook and ok and it == oit_ref
        ores[halo] = xs[0]
        dd.close()
        dist.barrier()
    assert np.array_equal(ores["exchange"], ores["overlap"])
    assert np.array_equal(ores["exchange"], ores["half"])  # half spinors on the wire
    # the even/odd action between processes with the overlapped exchange of the half fields (time slices of 256 sites)
    from oracle import evenodd as oeo2

    edims = (8, 8, 4, 4 * world)
    eV = synth.volume(edims)
    eU = synth.warm_links(edims, 0.3, 631)
    eP = synth.gaussian_momenta(edims, 632)
    ephi = oeo2.mhat(edims, kappa, BC, eU, oeo2.keep(synth.gaussian_spinor(edims, 633), edims, 0), dagger=True)
    _, eit_ref, _ = oeo2.fermion_force(edims, kappa, BC, eU, ephi, 1e-12, 10 * eV)
    eres = {}
    for halo in ("exchange", "overlap", "half"):
        dd = dist.decomposed_lattice(edims, beta, kappa, BC, lgt.LGT_F64, 0, None, halo=halo, transport="host")
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
        dd.set_links(eU)
        dd.set_momenta(eP)
        dd.set_pseudofermion(ephi)
        assert lgt.lgt_dd_md_kick(dd.d, 0.05, 1e-12, 10 * eV) == eit_ref
        eres[halo] = dd.get_momenta()[0]
        dd.close()
        dist.barrier()
    assert np.array_equal(eres["exchange"], eres["overlap"])
    assert np.array_equal(eres["exchange"], eres["half"])  # half-spinor faces of the half fields
    out["eo_overlap_cg_iters"] = eit_ref
    out["overlap_cg_iters"] = oit_ref

    # two split directions over the same transport: the z faces are strided (one run per local time slice) and are staged
    # through pinned memory by 2-D copies; a direction that is not split makes the rank its own neighbour
    gdims = (8, 4, 2 * world, 2 * world)
    gU = synth.warm_links(gdims, 0.3, 611)
    gP = synth.gaussian_momenta(gdims, 612)
    gb = oracle.dslash(gdims, kappa, BC, gU, synth.gaussian_spinor(gdims, 613), dagger=True)
    _, git_ref, _, gok = oracle.cg(gdims, kappa, BC, gU, gb, 1e-12, 5000)
    assert gok
    grids = [(1, world), (world, 1)] + ([(2, world // 2)] if world >= 4 else [])
    out["grid"] = {}
    for grid in grids:
        ref = lgt.DecomposedLattice(gdims, world, list(range(world)), beta, kappa, BC, grid=grid)
        ref.set_links(gU)
        ref_ds = ref.dslash(gb)[rank]
        ref_x, ref_it, _, _ = ref.cg(gb, 1e-12, 5000)
        ref.set_momenta(gP)
        ref.set_pseudofermion(gb)
        ref_traj = lgt.lgt_dd_md_trajectory(ref.d, 2, 0.03, tol=1e-13, max_iter=5000)
        ref_U, ref_P = ref.get_links()[rank], ref.get_momenta()[rank]
        ref.close()
        dd = dist.decomposed_lattice(gdims, beta, kappa, BC, lgt.LGT_F64, 0, None, transport="host", grid=grid)
        dd.set_links(gU)
        assert np.array_equal(dd.dslash(gb)[0], ref_ds)
        assert np.abs(dd.dslash(gb)[0] - dd.slab(oracle.dslash(gdims, kappa, BC, gU, gb), rank)).max() < 1e-12
        xs, it, rel, ok = dd.cg(gb, 1e-12, 5000)
        assert ok and it == git_ref == ref_it and np.array_equal(xs[0], ref_x[rank])
        dd.set_momenta(gP)
        dd.set_pseudofermion(gb)
        traj = lgt.lgt_dd_md_trajectory(dd.d, 2, 0.03, tol=1e-13, max_iter=5000)
        assert traj == ref_traj
        assert np.array_equal(dd.get_links()[0], ref_U) and np.array_equal(dd.get_momenta()[0], ref_P)
        out["grid"]["%dx%d" % grid] = {"cg_iters": it, "md_cg_iters": traj[2]}
        dd.close()
        dist.barrier()
    print(json.dumps(out), flush=True)
    dist.shutdown()


if __name__ == "__main__":
    main()
