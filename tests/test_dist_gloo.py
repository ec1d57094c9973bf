"""World-size-2 gloo test (CPU) of the multi-process aggregation bench.py uses for N > 1:
max over ranks of the time, sum over ranks of the work, replica seeds distinct per rank."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, sys
    sys.path.insert(0, %r)
    from paper_2602_20516_b200 import dist, synth
    rank, world = dist.init("gloo")
    assert world == 2
    dist.barrier()
    # rank r "measures" (r+1)*10 ms and 100*(r+1) units
    times, sums = dist.aggregate([10.0 * (rank + 1), 1.0], [100.0 * (rank + 1), 7.0])
    cfg = dict(synth.CONFIGS[0]); cfg["seed_links"] += 100 * rank
    U = synth.config_links(cfg)
    # decomposed mode: the id travels from rank 0, the slabs tile the lattice
    ident = dist.broadcast_bytes(bytes(range(128)) if rank == 0 else None, 128, src=0)
    lo, hi = dist.slab_rows((4, 4, 2, 8), world, rank)
    gathered = dist.allgather_bytes(bytes([rank + 1] * 16), 16)
    assert gathered == [bytes([1] * 16), bytes([2] * 16)]
    print(json.dumps({"rank": rank, "times": times, "sums": sums, "u00": [U[0,0,0,0].real, U[0,0,0,0].imag],
                      "value": dist.throughput(sums[0], times[0] * 1e-3), "id": list(ident), "rows": [lo, hi]}))
    dist.shutdown()
""") % ROOT


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_rank_aggregation_gloo(tmp_path):
    import json

    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["times"] == [20.0, 1.0]  # MAX over ranks
        assert o["sums"] == [300.0, 14.0]  # SUM over ranks
        assert abs(o["value"] - 300.0 / 20e-3) < 1e-9
    assert outs[0]["u00"] != outs[1]["u00"]  # replicas are independent lattices
    assert outs[0]["id"] == outs[1]["id"] == list(range(128))
    assert sorted(o["rows"] for o in outs) == [[0, 128], [128, 256]]


def test_single_process_identity():
    sys.path.insert(0, ROOT)
    from paper_2602_20516_b200 import dist

    t, s = dist.aggregate([3.0], [5.0])
    assert t == [3.0] and s == [5.0]
    assert dist.env_rank_world()[1] >= 1
    assert dist.broadcast_bytes(b"abc", 3) == b"abc"
    assert dist.allgather_bytes(b"xy", 2) == [b"xy"]
    rows = [dist.slab_rows((4, 4, 4, 12), 3, r) for r in range(3)]
    assert rows == [(0, 256), (256, 512), (512, 768)]
    import pytest
    with pytest.raises(ValueError):
        dist.slab_rows((4, 4, 4, 10), 3, 0)


# ---- the halo plan and the host transport of the decomposed lattice (lgt_dd_halo_plan, lgt_dd_set_host_transport)
def test_halo_plan_with_in_order_matching():
    """The plan every transport follows, run through a model of what NCCL, MPI and gloo guarantee -- messages between one
    pair of ranks are matched in the order they were posted -- for 1, 2 (both neighbours are the same peer), 3, 4 and 8
    ranks: every ghost slice must receive exactly the slice SURVEY 8(e) says it mirrors."""
    from collections import defaultdict, deque

    from paper_2602_20516_b200 import lgt

    lgt.lib()
    for nranks in (1, 2, 3, 4, 8):
        for lt in (1, 2, 5):
            plans = [lgt.lgt_dd_halo_plan(nranks, r, lt) for r in range(nranks)]
            # field[r][slice] = (owner rank, owner's local slice) of the data held there; ghosts start empty
            field = [[None] + [(r, t) for t in range(1, lt + 1)] + [None] for r in range(nranks)]
            wires = defaultdict(deque)  # (src, dst) -> messages in posting order
            for r, (sp, ss, rp, rs) in enumerate(plans):
                for k in range(2):
                    assert 1 <= ss[k] <= lt and rs[k] in (0, lt + 1)  # interior slices go out, ghost slices come in
                    wires[(r, sp[k])].append(field[r][ss[k]])
            for r, (sp, ss, rp, rs) in enumerate(plans):
                for k in range(2):
                    field[r][rs[k]] = wires[(rp[k], r)].popleft()
            assert all(not q for q in wires.values())
            for r in range(nranks):
                assert field[r][0] == ((r - 1) % nranks, lt)      # lower ghost = last interior slice of rank r - 1
                assert field[r][lt + 1] == ((r + 1) % nranks, 1)  # upper ghost = first interior slice of rank r + 1
    with __import__("pytest").raises(lgt.LgtError):
        lgt.lgt_dd_halo_plan(2, 2, 4)


HOST_TRANSPORT_WORKER = textwrap.dedent("""
    import json, sys
    import numpy as np
    sys.path.insert(0, %r)
    from paper_2602_20516_b200 import dist, lgt
    rank, world = dist.init("gloo")
    lgt.lib()
    lt, nbytes = 3, 4096
    sp, ss, rp, rs = lgt.lgt_dd_halo_plan(world, rank, lt)
    # a slab of lt + 2 slices; slice t of rank r is filled with the byte 16 * r + t
    slab = np.zeros((lt + 2, nbytes), dtype=np.uint8)
    for t in range(1, lt + 1):
        slab[t] = 16 * rank + t
    for rep in range(3):  # repeated exchanges must not cross-match
        recv = [np.zeros(nbytes, dtype=np.uint8) for _ in range(2)]
        dist.host_sendrecv([slab[ss[0]].copy(), slab[ss[1]].copy()], sp, recv, rp)
        slab[rs[0]], slab[rs[1]] = recv[0], recv[1]
        assert (slab[0] == 16 * ((rank - 1) %% world) + lt).all() and (slab[lt + 1] == 16 * ((rank + 1) %% world) + 1).all()
    buf = np.array([0.1 * (rank + 1), 1e-17 * (rank + 1), 3.0], dtype=np.float64)
    dist.host_allreduce(buf)
    print(json.dumps({"rank": rank, "sum": [x.hex() for x in buf.tolist()]}))
    dist.shutdown()
""") % ROOT


def test_host_transport_gloo_world_sizes(tmp_path):
    """dist.host_sendrecv / host_allreduce (the callbacks behind lgt_dd_set_host_transport) between 2 and 3 gloo ranks:
    with two ranks both neighbours are the one other rank, and each ghost must still get the right slice; the sums
    are bit-identical on every rank and equal the rank-ordered sum."""
    import json

    script = tmp_path / "ht_worker.py"
    script.write_text(HOST_TRANSPORT_WORKER)
    for world in (2, 3):
        port = free_port()
        procs = []
        for r in range(world):
            env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                       MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
            procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                          stderr=subprocess.PIPE, text=True))
        sums = []
        for p in procs:
            o, e = p.communicate(timeout=300)
            assert p.returncode == 0, e[-2000:]
            sums.append(json.loads(o.strip().splitlines()[-1])["sum"])
        expect = [0.0, 0.0, 0.0]
        for r in range(world):
            expect = [a + b for a, b in zip(expect, [0.1 * (r + 1), 1e-17 * (r + 1), 3.0])]
        assert all(s == [x.hex() for x in expect] for s in sums)


def test_host_transport_single_rank_is_a_copy():
    import numpy as np

    from paper_2602_20516_b200 import dist

    a, b = np.arange(8, dtype=np.uint8), np.arange(8, 16, dtype=np.uint8)
    ra, rb = np.zeros(8, dtype=np.uint8), np.zeros(8, dtype=np.uint8)
    dist.host_sendrecv([a, b], [0, 0], [ra, rb], [0, 0])
    assert (ra == a).all() and (rb == b).all()
    buf = np.array([1.5, 2.5])
    dist.host_allreduce(buf)
    assert buf.tolist() == [1.5, 2.5]


def test_grid_blocks_and_neighbours():
    import pytest

    """Host logic of the (Pt, Pz) decomposition: the ranks' blocks tile the lattice exactly once in lexicographic order, and
    the neighbour table is the periodic grid's (a direction that is not split makes a rank its own neighbour)."""
    import numpy as np

    from paper_2602_20516_b200 import dist

    dims = (4, 2, 6, 4)
    V = 4 * 2 * 6 * 4
    a = np.arange(V * 3).reshape(V, 3)
    for grid in ((1, 1), (2, 3), (4, 2), (1, 6)):
        n = grid[0] * grid[1]
        seen = np.zeros(V, dtype=int)
        for r in range(n):
            b = dist.grid_block(a, dims, grid, r)
            assert b.shape == (V // n, 3)
            sites = b[:, 0] // 3
            assert np.all(np.diff(sites) > 0)  # lexicographic inside the block
            t, z = sites // (4 * 2 * 6), (sites // 8) % 6
            pt, pz = divmod(r, grid[1])
            assert np.all(t // (4 // grid[0]) == pt) and np.all(z // (6 // grid[1]) == pz)
            seen[sites] += 1
            dn_t, up_t, dn_z, up_z = dist.grid_neighbours(grid, r)
            assert dist.grid_neighbours(grid, dn_t)[1] == r and dist.grid_neighbours(grid, up_t)[0] == r
            assert dist.grid_neighbours(grid, dn_z)[3] == r and dist.grid_neighbours(grid, up_z)[2] == r
            if grid[0] == 1:
                assert dn_t == up_t == r
            if grid[1] == 1:
                assert dn_z == up_z == r
        assert np.all(seen == 1)
    with pytest.raises(ValueError):
        dist.grid_block(a, dims, (3, 1), 0)
    with pytest.raises(ValueError):
        dist.grid_block(a, dims, (2, 2), 4)
