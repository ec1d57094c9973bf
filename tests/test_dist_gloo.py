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
