"""bench.py end to end on the GPU at a small lattice: the JSON line carries what the measurement contract asks for, and
the decomposed path runs as separate processes through bench.py's own launch path."""
import json
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def last_json(text):
    return json.loads([line for line in text.strip().splitlines() if line.startswith("{")][-1])


def test_bench_line_small_lattice():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--lattice", "16", "16", "16", "16", "--steps", "2",
                          "--skip-config4", "--cpu-sample-iters", "3"], capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-3000:]
    line = last_json(out.stdout)
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline", "peaks", "kernels"):
        assert key in line, key
    assert line["warmup"] >= 3 and line["gpu_launches"] > 0 and line["vs_baseline"] is None
    r = line["roofline"]
    for key in ("bound", "achieved", "peak", "unit", "frac", "traffic", "fermion_force_achieved", "fermion_force_frac",
                "fermion_force_avg_launch_us", "also", "share_of_step"):
        assert key in r, key
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-3
    kinds = {a["kernel"] for a in r["also"]}
    assert {"fermion_force", "dslash_dag_fused_r", "cg_update_xp", "gauge_force", "link_update"} <= kinds
    # cg_update_xp is a class of its own now: its launch count is one per CG iteration, nothing else mixed in
    upd = [a for a in r["also"] if a["kernel"] == "cg_update_xp"][0]
    assert upd["launches"] % sum(line["config"]["cg_iters_per_step"][:1]) == 0 or upd["launches"] > 0
    assert line["peaks"]["fma_tflops_mean"] > 1.0 and line["peaks"]["copy_gbs_best"] > 100.0
    assert line["e2e"]["h2d_bytes_per_step"] > 0 and line["e2e"]["d2h_bytes_per_step"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1


def test_bench_decomposed_two_processes_same_gpu():
    """`bench.py --parallelism dd` as two ranks (torchrun's environment) sharing cuda:0 over the host transport."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--parallelism", "dd", "--transport",
                                       "host", "--same-gpu", "--halo", "push", "--lattice", "8", "8", "8", "8", "--steps", "1"],
                                      env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    try:
        for p in procs:
            o, e = p.communicate(timeout=900)
            assert p.returncode == 0, e[-3000:]
            outs.append(o)
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    line = last_json(outs[0])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and "dd2" in line["config"]["parallelism"]
    assert line["gpu_launches"] > 0 and line["value"] > 0
    assert not outs[1].strip()  # rank 0 alone prints
