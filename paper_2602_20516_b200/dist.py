"""Multi-GPU plumbing: one process per GPU.

Two ways to use N GPUs:
  replicas   N independent lattices, no data-path collective (bench.py's default for N > 1, weak scaling);
  decomposed ONE lattice cut into N time slabs (lgt_dd_*): halo slices and the CG / action sums travel over the
             library's own NCCL communicator; this module only carries the 128-byte NCCL id from rank 0 to the
             others and says which rows of a canonical array belong to which rank.
torch.distributed is used for that broadcast, for the barrier around the timed region and for two tiny reductions:
the MAX over ranks of the device time and the SUM over ranks of the work done.
"""
import os


def env_rank_world():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend, device=None):
    """Initialises the default process group from the torchrun environment (no-op for world size 1)."""
    import torch.distributed as dist

    rank, world, _ = env_rank_world()
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if device is not None else {}
        dist.init_process_group(backend, **kw)
    return rank, world


def barrier():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(times, sums, device="cpu"):
    """times: per-rank durations -> elementwise MAX over ranks; sums: per-rank work counts -> SUM over ranks.
    Returns (times_max, sums_total) as python lists; identity for a single process."""
    import torch
    import torch.distributed as dist

    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    s = torch.tensor(list(sums), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return t.tolist(), s.tolist()


def slab_rows(dims, nranks, rank):
    """Row range [lo, hi) of a canonical field [V, ...] (site s = x + Lx*(y + Ly*(z + Lz*t)), t slowest) owned by
    `rank` when the lattice is cut into nranks slabs of Lt / nranks time slices."""
    Lx, Ly, Lz, Lt = [int(d) for d in dims]
    if nranks < 1 or Lt % nranks:
        raise ValueError("Lt must be a multiple of the number of ranks")
    if not 0 <= rank < nranks:
        raise ValueError("bad rank")
    per = Lx * Ly * Lz * (Lt // nranks)
    return rank * per, (rank + 1) * per


def grid_block(a, dims, grid, rank):
    """Block of a canonical field a[V, ...] owned by `rank` = pt * Pz + pz of a (Pt, Pz) grid (lgt_dd_create_grid): time
    slices [pt Lt/Pt, (pt+1) Lt/Pt), z planes [pz Lz/Pz, (pz+1) Lz/Pz), flattened in lexicographic order."""
    Lx, Ly, Lz, Lt = [int(d) for d in dims]
    Pt, Pz = int(grid[0]), int(grid[1])
    if Pt < 1 or Pz < 1 or Lt % Pt or Lz % Pz:
        raise ValueError("Lt must be a multiple of Pt and Lz of Pz")
    if not 0 <= rank < Pt * Pz:
        raise ValueError("bad rank")
    pt, pz = divmod(int(rank), Pz)
    lt, lz = Lt // Pt, Lz // Pz
    b = a.reshape((Lt, Lz, Ly * Lx) + tuple(a.shape[1:]))[pt * lt:(pt + 1) * lt, pz * lz:(pz + 1) * lz]
    return b.reshape((lt * lz * Ly * Lx,) + tuple(a.shape[1:]))


def grid_neighbours(grid, rank):
    """(t_down, t_up, z_down, z_up) ranks of `rank` on a periodic (Pt, Pz) grid -- the peers of the two exchange phases."""
    Pt, Pz = int(grid[0]), int(grid[1])
    pt, pz = divmod(int(rank), Pz)
    return (((pt - 1) % Pt) * Pz + pz, ((pt + 1) % Pt) * Pz + pz, pt * Pz + (pz - 1) % Pz, pt * Pz + (pz + 1) % Pz)


def broadcast_bytes(data, nbytes, src=0, device="cpu"):
    """Rank `src` passes `data` (bytes of length nbytes), everybody returns the same bytes.  Identity without a group."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return bytes(data)
    if dist.get_rank() == src:
        t = torch.tensor(list(bytes(data)), dtype=torch.uint8, device=device)
        assert t.numel() == nbytes
    else:
        t = torch.zeros(nbytes, dtype=torch.uint8, device=device)
    dist.broadcast(t, src=src)
    return bytes(t.cpu().tolist())


def allgather_bytes(data, nbytes, device="cpu"):
    """Every rank passes nbytes bytes; returns the list of all ranks' bytes in rank order."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return [bytes(data)]
    mine = torch.tensor(list(bytes(data)), dtype=torch.uint8, device=device)
    assert mine.numel() == nbytes
    out = [torch.zeros(nbytes, dtype=torch.uint8, device=device) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine)
    return [bytes(t.cpu().tolist()) for t in out]


def host_sendrecv(send_bufs, send_peers, recv_bufs, recv_peers, group=None):
    """The `sendrecv` callback of lgt_dd_set_host_transport over a torch.distributed group with CPU tensors (gloo):
    the k-th send of a rank is the k-th receive of its peer (lgt_dd_halo_plan), so message k carries tag k and the
    pairing does not depend on arrival order.  A rank that is its own peer copies."""
    import numpy as np
    import torch
    import torch.distributed as dist

    me = dist.get_rank(group) if dist.is_available() and dist.is_initialized() else 0
    reqs = []
    for k in range(2):
        if send_peers[k] == me:  # this rank is its own neighbour: its k-th send is its own k-th receive
            assert recv_peers[k] == me
            np.copyto(recv_bufs[k], send_bufs[k])
        else:
            reqs.append(dist.isend(torch.from_numpy(send_bufs[k]), send_peers[k], group=group, tag=k))
    for k in range(2):
        if recv_peers[k] != me:
            reqs.append(dist.irecv(torch.from_numpy(recv_bufs[k]), recv_peers[k], group=group, tag=k))
    for r in reqs:
        r.wait()


def host_allreduce(buf, group=None):
    """The `allreduce` callback: all-gather, then the sum in rank order on every rank -- the same bits everywhere, and
    the same bits as the in-process lockstep mode (dd_local_allreduce_kernel adds in rank order too)."""
    import numpy as np
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return
    mine = torch.from_numpy(np.array(buf, dtype=np.float64))
    parts = [torch.zeros_like(mine) for _ in range(dist.get_world_size(group))]
    dist.all_gather(parts, mine, group=group)
    total = np.zeros_like(buf)
    for p in parts:
        total = total + p.numpy()
    buf[:] = total


def decomposed_lattice(dims, beta, kappa, bc, precision=None, local_device=0, stream=None, halo="exchange", transport="nccl",
                       host_group=None, grid=None):
    """This process's slab of ONE lattice shared by all ranks of the default process group: a DecomposedLattice with one
    local rank.  transport = "nccl": the library's own NCCL communicator, initialised from an id that rank 0 creates and
    broadcasts here.  transport = "host": halo slices and sums travel through host memory over `host_group` (a gloo
    group; the default group if None) -- for clusters without NCCL between the ranks and for running the inter-process
    path with several processes on ONE GPU, which NCCL refuses.
    halo = "push": the neighbours' CG buffers are mapped through CUDA IPC (handles all-gathered here) and the halo
    slices travel inside the Dslash kernels (lgt.LGT_DD_PUSH).
    grid = (Pt, Pz) with Pt * Pz = world size: two split directions (lgt_dd_create_grid), rank = pt * Pz + pz; exchange mode only."""
    from . import lgt

    rank, world, _ = env_rank_world()
    if grid is not None and halo == "push":
        raise ValueError("a (Pt, Pz) grid exchanges its halos; LGT_DD_PUSH is for time slabs")
    dd = lgt.DecomposedLattice(dims, world, [rank], beta, kappa, bc, lgt.LGT_F64 if precision is None else precision,
                               local_device, stream, grid=grid)
    on_cpu = transport == "host"
    if transport == "host":
        lgt.lgt_dd_set_host_transport(dd.d, lambda sb, sp, rb, rp: host_sendrecv(sb, sp, rb, rp, host_group),
                                      lambda buf: host_allreduce(buf, host_group))
    elif world > 1:
        ident = lgt.lgt_dd_nccl_unique_id() if rank == 0 else None
        ident = broadcast_bytes(ident, 128, src=0, device="cuda:%d" % local_device)
        lgt.lgt_dd_nccl_init(dd.d, ident)
    if world > 1 and halo == "push":
        handles = allgather_bytes(lgt.lgt_dd_ipc_export(dd.d), 128, device="cpu" if on_cpu else "cuda:%d" % local_device)
        lgt.lgt_dd_ipc_import(dd.d, handles[(rank - 1) % world], handles[(rank + 1) % world])
    if halo == "push":
        lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH)
    elif halo == "overlap":
        lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_OVERLAP)
    elif halo == "half":
        lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_HALF)
    return dd


def throughput(units_total, time_max_s):
    """Whole-job throughput: units all ranks processed / max-over-ranks time."""
    return units_total / time_max_s


def shutdown():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
