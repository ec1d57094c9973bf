#!/usr/bin/env python
"""bench.py -- one JSON line for the HMC MD-step hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one molecular-dynamics step of BASELINE.json configs[3] in the reading DESIGN.md A-13:
kick(dt) = gauge force + CG on D^dag D to 1e-12 + Y = D X + fused fermion force, then drift(dt) = link update,
on a 32^4 SU(3) lattice in fp64 (beta 5.6, kappa 0.12, antiperiodic time, dt 0.01, seeded warm-start links).

What is timed, in this order:
  1. K steps on the path users get (CUDA graphs for the CG chunks, no per-kernel events): `value`, `ms_per_step`.
     `value` is the algorithmic HBM traffic of all kernels of the step / device time.
  2. a few more steps with a CUDA-event pair around every launch (lgt_timing_*): `roofline` -- the dominant kernel
     (Dslash inside CG) and, because the metric names it too, the fused fermion force; every kernel class of the step.
  3. the same step end to end through the C ABI with HOST buffers in and out every step: `e2e`.
  4. the metric's kernels in isolation, fp64 and fp32 (`kernels`), the measured fp64 FMA / copy peaks (`peaks`),
     configs[4] (48^3 x 96) as a short sweep (`configs4`), the oracle on the host cores (`cpu_baseline`).
  --extras adds the non-headline solver arms, the paper's own lattice sizes and the one-GPU slab runs.
N > 1: N independent replicas (one lattice per GPU, no data-path collective), weak scaling, plus -- guarded by a watchdog --
one pass of the same step on ONE lattice cut into N time slabs (`decomposed`); --parallelism dd makes that the headline.
--impl reference times the CPU oracle on a bounded sample of the same workload (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fermion-force + Dslash HBM GB/s and GFLOP/s (fp64, 32^4) vs B200 roofline"

# Algorithmic bytes and flops per site in units of one REAL number (x8 B in fp64, x4 B in fp32); DESIGN.md.
REALS = dict(
    dslash=2 * (36 + 12 + 12),               # U + in + out                      -> 960 B fp64
    dslash_fused_r=2 * (36 + 12 + 2 * 12),   # U + t + r rw (q = D^dag t stays on chip) -> 1152 B
    cg_update_xp=2 * (5 * 12),               # x rw, p rw, r r                   -> 960 B
    cg_iter=2 * (60 + 72 + 60),              # the three launches above          -> 3072 B
    cg_init=2 * (4 * 12),                    # b r; x, r, p w
    fermion_force=2 * (36 + 12 + 12) + 2 * 32,  # U + X + Y + Pi (8 reals x 4 links) rw -> 1472 B
    gauge_force=2 * 36 + 2 * 32,             # U + Pi rw                         -> 1088 B
    link_update=32 + 2 * 2 * 36,             # Pi r + U rw                       -> 1408 B
    plaquette=2 * 36,                        # U r (six planes per site)         -> 576 B
)
FLOPS = dict(dslash=1368, dslash_fused_r=1368 + 96, cg_update_xp=96, cg_iter=2 * 1368 + 192, fermion_force=2300, gauge_force=10900, link_update=3500,
             plaquette=2600)

# dram__bytes_read.sum + dram__bytes_write.sum per launch at 32^4 fp64 from the ncu --set full captures summarised in
# profiles/ (the file named beside each figure); None = not captured for the current kernel.
NCU_TRAFFIC_BYTES = {
    "dslash": 1022402560,          # profiles/r02b_bench_kernels.md, dslash_kernel<double,0,1>: 0.831 + 0.192 GB
    "dslash_fused_r": 1226198936,  # profiles/r02b_bench_kernels.md, dslash_kernel<double,1,2>: 1.036 + 0.191 GB
    "cg_update_xp": 954585528,     # profiles/r02b_bench_kernels.md, cg_update_xp_kernel<double>: 0.604 + 0.351 GB
    "fermion_force": 1545540064,   # profiles/r02b_bench_kernels.md, fermion_force_kernel<double,1>: 1.290 + 0.256 GB
    "gauge_force": 1237131631,     # profiles/r02b_bench_kernels.md, gauge_force_kernel<double,1,1>: 0.974 + 0.263 GB
    "link_update": 1421068328,     # profiles/r02b_bench_kernels.md, link_update_kernel<double>: 0.872 + 0.549 GB
}

# even/odd action, per site of the FULL lattice: a half-lattice hop reads 8 links + 1 spinor and writes 1 spinor per
# output site, and there are V/2 output sites
REALS_EO = dict(hop=(2 * (72 + 12 + 12)) // 2, hop_fused_r=(2 * (72 + 12 + 2 * 12)) // 2, update_xp=(2 * 5 * 12) // 2)
REALS_EO["cg_iter"] = 3 * REALS_EO["hop"] + REALS_EO["hop_fused_r"] + REALS_EO["update_xp"]   # -> 3408 B fp64

# one stout level, forward (staples -> A, exp(A) U -> U') and backward (local: A, F' rw, G; chain: U, G, Fdir, out rw)
REALS_STOUT_LEVEL = (2 * 36 + 32) + (32 + 2 * 2 * 36) + (32 + 2 * 32 + 32) + (2 * 36 + 32 + 32 + 2 * 32)


# lgt_set_kernel_variant: what each number means (include/lgt.h has the same list)
VARIANT_NAMES = {
    "dslash": ["one 128-site block per chunk (default)",
               "persistent, next chunk's first two hops requested before the current chunk's last",
               "persistent, forward links by bulk copy (TMA) into per-warp shared-memory slots one chunk ahead",
               "256-thread blocks on 2 x 2 x 2 tiles of 32-site layout blocks",
               "variant 0 + L2 prefetch for the block 2 x SMs further on",
               "variant 0 with the z and t neighbours loaded past L1 (no_allocate)",
               "variant 0 with the DRAM-bound hops first (t+, z+, y+, x+, then the backward ones)",
               "12-real links: rows 0, 1 read, row 2 rebuilt in registers (768 B per site)",
               "variant 0 + the L2 prefetch of variant 4 issued at the end of each block (the fp32 default)",
               "persistent, DRAM-bound operands (forward links, t+1 spinor) by per-thread cp.async into shared memory one chunk ahead",
               "variant 1 with the chunks drawn from a global counter instead of a fixed stride",
               "two chunks per block as straight-line code",
               "12-real links in the fp32 default's build (3 blocks per SM, late prefetch of rows 0, 1); fp64 runs variant 7"],
    "gauge_force": ["one 32-site layout block x 4 directions per 128-thread block (default)",
                    "two layout blocks per 256-thread block",
                    "four layout blocks per 512-thread block (128 registers)",
                    "one thread per site: up staples plaquette by plaquette (3 products serve 2 links), 46 instead of 52 products per site"],
}


def step_reals(cg_iters, solver="cg", action="full", smear=0):
    fixed = REALS["gauge_force"] + REALS["fermion_force"] + REALS["link_update"] + smear * REALS_STOUT_LEVEL
    if action == "eo":  # CG on M^dag M, then Y_e = M X_e, X_o, Y_o (3 hops), split of phi and two merges (5 x 24 x 2)
        return fixed + cg_iters * REALS_EO["cg_iter"] + 3 * REALS_EO["hop"] + 5 * 48
    if solver == "mixed":  # fp32 iterations move half the bytes; about 4 fp64 defect-correction cycles of 2 Dslash + 3 BLAS-1
        return fixed + cg_iters * REALS["cg_iter"] // 2 + 4 * (2 * REALS["dslash"] + 3 * 48)
    return fixed + REALS["cg_init"] + cg_iters * REALS["cg_iter"] + REALS["dslash"]


def step_flops(cg_iters):
    return (FLOPS["gauge_force"] + cg_iters * FLOPS["cg_iter"] + FLOPS["dslash"] + FLOPS["fermion_force"]
            + FLOPS["link_update"])


def workload_name(config, dims):
    return ("configs[%d]: %s SU(3) one MD step = kick(dt) [gauge force, CG on D^dag D, Y = D X, fermion force] + drift(dt)"
            % (config, "x".join(map(str, dims))))


def measured_peaks():
    """(HBM GB/s burst, HBM source, sustained bf16 figure unused here)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe): NVML in a
    thread every 20 ms, or the recipe's nvidia-smi line every 100 ms when pynvml is missing."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.index, self.rows, self.proc, self.stop_flag, self.thread, self.source = index, [], None, False, None, None

    def start(self):
        try:
            import pynvml

            pynvml.nvmlInit()
            # NVML enumerates physical devices; map through CUDA_VISIBLE_DEVICES when it lists plain indices
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            ids = [v for v in vis.split(",") if v.strip().isdigit()]
            phys = int(ids[self.index]) if self.index < len(ids) else self.index
            h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            mx = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            bits = [pynvml.nvmlClocksThrottleReasonHwSlowdown, pynvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                    pynvml.nvmlClocksThrottleReasonSwThermalSlowdown, pynvml.nvmlClocksThrottleReasonSwPowerCap]

            def loop():
                while not self.stop_flag:
                    try:
                        sm = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                        pw = pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0
                        r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                        self.rows.append([sm, mx, pw] + [bool(r & b) for b in bits])
                    except Exception:
                        pass
                    time.sleep(0.02)

            self.source = "nvml"
            self.thread = threading.Thread(target=loop, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.source = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi"
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            try:
                self.rows.append([float(r[0]), float(r[1]), float(r[2])] + [x.lower() == "active" for x in r[3:7]])
            except (ValueError, IndexError):
                pass

    def stop(self):
        if self.source is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no NVML and no nvidia-smi"]}
        self.stop_flag = True
        if self.proc is not None:
            self.proc.terminate()
        self.thread.join(timeout=2)
        rows = list(self.rows)
        # "under load": samples drawing more than half of the maximum power seen (drops the idle lead-in and tail)
        pmax = max((r[2] for r in rows), default=0.0)
        load = [r for r in rows if r[2] >= 0.5 * pmax] or rows
        sm = sorted(r[0] for r in load)
        reasons = [n for i, n in enumerate(self.NAMES) if any(r[3 + i] for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max((r[1] for r in rows), default=None),
                "power_w_max": round(pmax, 1) if rows else None, "samples": len(rows), "samples_under_load": len(load),
                "source": self.source, "reasons": reasons}


def make_inputs(cfg):
    """Seeded synthetic fields of the workload (numpy, canonical layout)."""
    from paper_2602_20516_b200 import synth

    dims = cfg["dims"]
    U = synth.config_links(cfg)
    P = synth.gaussian_momenta(dims, cfg.get("seed_mom", cfg["seed_links"] + 1))
    eta = synth.gaussian_spinor(dims, cfg.get("seed_eta", cfg["seed_links"] + 2))
    return U, P, eta


def event_pair():
    import torch

    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def time_calls(fn, n=20, warm=5):
    """Mean device time (s) of one call, CUDA events on torch's current stream (the handles' stream), after warm-up."""
    import torch

    for _ in range(warm):
        fn()
    a, b = event_pair()
    torch.cuda.synchronize()
    a.record()
    for _ in range(n):
        fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b) / n * 1e-3


def isolated_kernels(lgt, handle, real_bytes, V, tag, out, n=20):
    """The path's kernels one at a time on resident native fields (inputs exceed L2 at 32^4 and above)."""
    import torch

    hctx = handle.ctx
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    bufs = []
    for _ in range(3):
        b = handle.native_spinor()
        b.view(torch.float64 if real_bytes == 8 else torch.float32).normal_(generator=g)
        bufs.append(b)
    for name, fn, key in (
            ("dslash", lambda: lgt.lgt_dslash_native(hctx, bufs[0], bufs[1], False), "dslash"),
            ("dslash_dagger", lambda: lgt.lgt_dslash_native(hctx, bufs[0], bufs[1], True), "dslash"),
            ("fermion_force", lambda: lgt.lgt_fermion_force_native(hctx, bufs[0], bufs[2], 1e-3), "fermion_force"),
            ("gauge_force", lambda: lgt.lgt_gauge_force_accumulate(hctx, 1e-3), "gauge_force"),
            ("link_update", lambda: lgt.lgt_md_drift(hctx, 1e-6), "link_update"),
            # S_g: plaquette kernel + fixed-order sum; the call reads its 8-byte result back, so this is call time
            ("plaquette_action_call", lambda: lgt.lgt_plaquette(hctx), "plaquette")):
        t = time_calls(fn, n=n)
        out[name + tag] = {"us": round(t * 1e6, 2), "GB/s": round(REALS[key] * real_bytes * V / t / 1e9, 1),
                           "GFLOP/s": round(FLOPS[key] * V / t / 1e9, 1)}
    del bufs


def configs4_sweep(lgt, synth, local, stream, peak):
    """BASELINE.json configs[4]: 48^3 x 96, kappa 0.12, fp64 and fp32 -- isolated Dslash, CG on D^dag D to 1e-10, fermion
    force, gauge force.  Links: the seeded 24^4 warm field (eps = 0.3, seed 1401) tiled periodically 2 x 2 x 2 x 4 (the recipe
    of the parity test; drawing 42 M matrix exponentials in numpy would take minutes); eta: seeded Gaussian."""
    import numpy as np
    import torch

    c = synth.CONFIGS[4]
    dims, kappa, bc = tuple(c["dims"]), c["kappa"], c["bc"]
    V = synth.volume(dims)
    small = (24, 24, 24, 24)
    Us = torch.from_numpy(synth.warm_links(small, 0.3, c["seed_links"])).cuda().reshape(24, 24, 24, 24, 4, 3, 3)  # [t][z][y][x]
    U = Us.repeat(dims[3] // 24, dims[2] // 24, dims[1] // 24, dims[0] // 24, 1, 1, 1).reshape(V, 4, 3, 3).contiguous()
    del Us
    g = torch.Generator(device="cuda")
    g.manual_seed(c.get("seed_eta", 1402))
    eta = torch.view_as_complex((torch.randn((V, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64) * np.sqrt(0.5)).contiguous())
    res = {"lattice": "x".join(map(str, dims)), "kappa": kappa, "cg_tol": c.get("cg_tol", 1e-10),
           "links": "24^4 warm field (eps 0.3, seed %d) tiled periodically" % c["seed_links"]}
    lat = lgt.Lattice(dims, c.get("beta", 5.6), kappa, bc, lgt.LGT_F64, local, stream)
    lgt.lgt_set_links(lat.ctx, U)
    phi, x = lat.empty(V, 4, 3), lat.empty(V, 4, 3)
    lgt.lgt_dslash(lat.ctx, eta, phi, True)
    del eta
    torch.cuda.synchronize()
    a, b = event_pair()
    lgt.lgt_timing_reset(lat.ctx)
    lgt.lgt_timing_enable(lat.ctx, True)
    a.record()
    it, rel, ok = lgt.lgt_cg(lat.ctx, phi, x, c.get("cg_tol", 1e-10), 10 * V)
    b.record()
    torch.cuda.synchronize()
    lgt.lgt_timing_enable(lat.ctx, False)
    cg_ms = a.elapsed_time(b)
    ds_ms, ds_n = lgt.lgt_timing_read(lat.ctx, lgt.LGT_K_DSLASH)
    lgt.lgt_timing_reset(lat.ctx)
    gbs = REALS["dslash"] * 8 * V / (ds_ms / max(ds_n, 1) * 1e-3) / 1e9
    res["cg_f64"] = {"iters": it, "converged": bool(ok), "rel_resid": rel, "ms": round(cg_ms, 2),
                     "ms_per_iter": round(cg_ms / max(it, 1), 3),
                     "GB/s": round((REALS["cg_init"] + it * REALS["cg_iter"]) * 8 * V / (cg_ms * 1e-3) / 1e9, 1),
                     "dslash_in_cg_us": round(ds_ms / max(ds_n, 1) * 1e3, 1), "dslash_in_cg_GB/s": round(gbs, 1),
                     "dslash_in_cg_frac": round(gbs / peak, 4),
                     "note": "call time incl. the canonical <-> native conversion of b and x"}
    del phi, x
    kern = {}
    isolated_kernels(lgt, lat, 8, V, "_f64", kern, n=10)
    lat.close()
    lat32 = lgt.Lattice(dims, c.get("beta", 5.6), kappa, bc, lgt.LGT_F32, local, stream)
    lgt.lgt_set_links(lat32.ctx, U.to(torch.complex64))
    del U
    isolated_kernels(lgt, lat32, 4, V, "_f32", kern, n=10)
    # fp32 "CG" = time per iteration at a fixed count (reading A-20: 1e-10 is out of reach in pure fp32)
    g.manual_seed(1403)
    b32 = torch.view_as_complex(torch.randn((V, 4, 3, 2), generator=g, device="cuda", dtype=torch.float32).contiguous())
    x32 = torch.empty_like(b32)
    a.record()
    it32, rel32, _ = lgt.lgt_cg(lat32.ctx, b32, x32, 0.0, 40)
    b.record()
    torch.cuda.synchronize()
    res["cg_f32_fixed_40_iters"] = {"iters": it32, "ms_per_iter": round(a.elapsed_time(b) / max(it32, 1), 3), "rel_resid": rel32}
    lat32.close()
    res["kernels"] = kern
    return res


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch

    from paper_2602_20516_b200 import dist, lgt, synth

    rank, world, local = dist.env_rank_world()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist.init("nccl", torch.device("cuda", local))
    lgt.lib()

    cfg = dict(synth.CONFIGS[args.config])
    if args.lattice:
        cfg["dims"] = tuple(args.lattice)
    cfg["seed_links"] += 100 * rank  # replicas: one independent lattice per GPU
    dims, beta, kappa, bc = cfg["dims"], cfg["beta"], cfg["kappa"], cfg["bc"]
    tol, dt = cfg.get("cg_tol", 1e-12), cfg.get("dt", 0.01)
    V = synth.volume(dims)
    max_iter = 10 * V
    U, P, eta = make_inputs(cfg)

    stream = torch.cuda.current_stream().cuda_stream
    lat = lgt.Lattice(dims, beta, kappa, bc, lgt.LGT_F64, local, stream)
    ctx = lat.ctx
    if args.smear:
        lgt.lgt_set_smearing(ctx, args.smear, 0.3)  # rho = 0.3
    hU, hP = torch.from_numpy(U).pin_memory(), torch.from_numpy(P).pin_memory()
    d_eta, d_phi = lat.to_device(eta), lat.empty(V, 4, 3)
    lgt.lgt_set_links_host(ctx, hU)
    lgt.lgt_dslash(ctx, d_eta, d_phi, True)  # phi = D^dag eta, made by the CUDA path itself
    hphi = d_phi.cpu().pin_memory()
    hU_out, hP_out = torch.empty_like(hU).pin_memory(), torch.empty_like(hP).pin_memory()
    del U, P, eta, d_eta

    def reset_state():
        lgt.lgt_set_links_host(ctx, hU)
        lgt.lgt_set_momenta_host(ctx, hP)
        lgt.lgt_set_pseudofermion_host(ctx, hphi)

    def md_step():
        it = lgt.lgt_md_kick(ctx, dt, tol, max_iter)
        lgt.lgt_md_drift(ctx, dt)
        return it

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    if args.solver == "mixed":
        lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    if args.action == "eo":
        lgt.lgt_set_fermion_action(ctx, lgt.LGT_ACTION_EO)
    variant = args.solver != "cg" or args.action != "full" or args.smear > 0
    reset_state()
    for _ in range(args.warmup):
        md_step()

    # ---- 1. the timed region: K steps on the product path (CG chunks replayed as CUDA graphs, no per-kernel events),
    # device time by CUDA events on the handle's stream, max over ranks
    sampler = ClockSampler(local)
    launches0 = lgt.lgt_launch_count(ctx)
    e0, e1 = event_pair()
    sampler.start()
    barrier()
    e0.record()
    iters = [md_step() for _ in range(args.steps)]
    e1.record()
    barrier()
    clocks = sampler.stop()
    elapsed_ms = e0.elapsed_time(e1)
    launches = lgt.lgt_launch_count(ctx) - launches0
    total_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in iters) * V
    total_flops = sum(step_flops(i) for i in iters) * V

    # ---- 2. the same steps once more with a CUDA-event pair around every launch (plain launches): per-kernel times in place
    k_ev = max(1, min(args.steps, 5))
    lgt.lgt_timing_reset(ctx)
    lgt.lgt_timing_enable(ctx, True)
    sampler_ev = ClockSampler(local)
    sampler_ev.start()
    ev0, ev1 = event_pair()
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(k_ev):
        md_step()
    ev1.record()
    torch.cuda.synchronize()
    clocks_ev = sampler_ev.stop()
    lgt.lgt_timing_enable(ctx, False)
    ev_ms = ev0.elapsed_time(ev1)
    per_class = {name: lgt.lgt_timing_read(ctx, k) for k, name in enumerate(lgt.KERNEL_CLASSES)}
    lgt.lgt_timing_reset(ctx)

    # ---- 3. end to end: host buffers in, host buffers out, through the C ABI, every step
    k_e2e = max(1, args.steps)
    barrier()
    t0 = time.perf_counter()
    e2e_iters = []
    for _ in range(k_e2e):
        # every step: inputs from pinned host memory, results back to pinned host memory, through the C ABI.  The links and
        # the pseudofermion are needed at once (blocking calls); the momenta upload overlaps the solve and the downloads
        # of the results overlap the next step (lgt_*_host_async); the region ends when every transfer has completed.
        lgt.lgt_set_links_host(ctx, hU)
        lgt.lgt_set_pseudofermion_host(ctx, hphi)
        lgt.lgt_set_momenta_host_async(ctx, hP)
        e2e_iters.append(md_step())
        lgt.lgt_get_links_host_async(ctx, hU_out)
        lgt.lgt_get_momenta_host_async(ctx, hP_out)
    lgt.lgt_host_transfers_wait(ctx)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in e2e_iters) * V
    h2d = hU.numel() * 16 + hP.numel() * 16 + hphi.numel() * 16
    d2h = hU_out.numel() * 16 + hP_out.numel() * 16

    extras = {}
    if rank == 0 and args.extras and not variant:
        extras = run_extras(args, lgt, synth, lat, cfg, hU, hP, hphi, reset_state, md_step, local, stream)

    # ---- max over ranks, aggregate
    (elapsed_ms, e2e_s), (total_reals, total_flops, e2e_reals, launches_all) = dist.aggregate(
        [elapsed_ms, e2e_s], [total_reals, total_flops, e2e_reals, launches], device="cuda")

    # ---- N > 1: the same step on ONE lattice cut into N time slabs (lgt_dd_*, NCCL), after the headline numbers are safe
    decomposed = None
    if world > 1 and not args.skip_dd_leg and not variant:
        lat.close()
        lat = None
        decomposed = guarded_decomposed_leg(args, rank, world, local)

    # ---- 4. the metric's two kernels in isolation (inputs exceed L2: links 604 MB, spinors 201 MB each), fp64 and fp32
    kernels, peaks, cfg4 = {}, None, None
    if rank == 0:
        if lat is None:
            lat = lgt.Lattice(dims, beta, kappa, bc, lgt.LGT_F64, local, stream)
            lgt.lgt_set_links_host(lat.ctx, hU)
        ctx = lat.ctx
        isolated_kernels(lgt, lat, 8, V, "_f64", kernels)
        peaks = lgt.lgt_measure_peaks(ctx, 20)
        lat32 = lgt.Lattice(dims, beta, kappa, bc, lgt.LGT_F32, local, stream)
        lgt.lgt_get_links(ctx, d_U := lat.empty(V, 4, 3, 3))
        lgt.lgt_set_links(lat32.ctx, d_U.to(torch.complex64))
        del d_U
        isolated_kernels(lgt, lat32, 4, V, "_f32", kernels)
        peaks["fma_f32_tflops_mean"] = lgt.lgt_measure_peaks(lat32.ctx, 20, copy=False)["fma_tflops_mean"]
        lat32.close()
    if lat is not None:
        lat.close()
    if rank == 0 and not args.skip_config4 and not variant and args.config == 3 and not args.lattice:
        try:
            cfg4 = configs4_sweep(lgt, synth, local, stream, measured_peaks()[0])
        except Exception as e:  # the sweep must never cost the headline line
            cfg4 = {"error": "%s: %s" % (type(e).__name__, e)}

    dd_hung = isinstance(decomposed, dict) and "timed out" in str(decomposed.get("error", ""))
    if rank != 0:
        if dd_hung:
            os._exit(0)  # a collective of the guarded leg never returned: do not wait for it in the teardown either
        dist.shutdown()
        return

    peak, peak_src = measured_peaks()
    fma_peak = peaks["fma_tflops_mean"] if peaks else None
    full = tuple(dims) == (32, 32, 32, 32) and not variant

    def in_place(name, key, bound="hbm"):
        ms, n = per_class[name]
        if not n:
            return None
        avg_s = ms / n * 1e-3
        real_bytes = 4 if args.solver == "mixed" and name.startswith(("dslash", "cg_")) else 8
        nbytes = (REALS_EO["hop"] if args.action == "eo" and name == "dslash" else REALS[key]) * real_bytes * V
        gbs = nbytes / avg_s / 1e9
        d = {"kernel": name, "where": "inside the MD step (event pair per launch)", "launches": n, "avg_launch_us": round(avg_s * 1e6, 2),
             "bound": bound, "achieved": round(gbs, 1), "peak": peak, "unit": "GB/s", "frac": round(gbs / peak, 4),
             "algorithmic_bytes_per_launch": nbytes, "traffic": NCU_TRAFFIC_BYTES.get(key) if full else None}
        if bound == "alu" and fma_peak:
            tf = FLOPS[key] * V / avg_s / 1e12
            d.update({"achieved": round(tf, 2), "peak": round(fma_peak, 2), "unit": "TFLOP/s", "frac": round(tf / fma_peak, 4),
                      "hbm_GB/s": round(gbs, 1), "hbm_frac": round(gbs / peak, 4)})
        return d

    ds = in_place("dslash", "dslash")
    ff = in_place("fermion_force", "fermion_force")
    also = [x for x in (ff, in_place("dslash_dag_fused_r", "dslash_fused_r"), in_place("cg_update_xp", "cg_update_xp"),
                        in_place("gauge_force", "gauge_force", "alu"), in_place("link_update", "link_update")) if x]
    iso_ff = kernels.get("fermion_force_f64")
    if iso_ff:
        also.append({"kernel": "fermion_force", "where": "isolated, 20 launches", "avg_launch_us": iso_ff["us"], "bound": "hbm",
                     "achieved": iso_ff["GB/s"], "peak": peak, "unit": "GB/s", "frac": round(iso_ff["GB/s"] / peak, 4),
                     "traffic": NCU_TRAFFIC_BYTES.get("fermion_force") if full else None})
    shares = {name: round(ms / ev_ms, 4) for name, (ms, n) in per_class.items() if n}
    value = total_reals * 8 / (elapsed_ms * 1e-3) / 1e9
    roofline = {"kernel": ("hop_cb_kernel<float>" if args.action == "eo" and args.solver == "mixed" else
                           "hop_cb_kernel<double>" if args.action == "eo" else
                           "dslash_kernel<float>" if args.solver == "mixed" else "dslash_kernel<double>") + " (inside CG, %d launches)" % (ds["launches"] if ds else 0),
                "bound": "hbm", "achieved": ds["achieved"] if ds else None, "peak": peak, "unit": "GB/s",
                "frac": ds["frac"] if ds else None, "traffic": ds["traffic"] if ds else None,
                "frac_of_nominal_8TBs": round(ds["achieved"] / 8000.0, 4) if ds else None,
                "peak_source": peak_src, "avg_launch_us": ds["avg_launch_us"] if ds else None,
                "algorithmic_bytes_per_launch": ds["algorithmic_bytes_per_launch"] if ds else None,
                "timed_how": "%d extra steps after the headline region with lgt_timing_enable: plain launches, one CUDA-event pair "
                             "per launch on the handle's stream (%.1f ms per step against %.1f ms on the graph path)"
                             % (k_ev, ev_ms / k_ev, elapsed_ms / args.steps),
                # the metric's second named kernel, flat so that it survives a shallow copy of this object
                "fermion_force_kernel": "fermion_force_kernel<double,1> (fused Pi -= eps F, inside the MD step)",
                "fermion_force_achieved": ff["achieved"] if ff else None, "fermion_force_frac": ff["frac"] if ff else None,
                "fermion_force_avg_launch_us": ff["avg_launch_us"] if ff else None,
                "fermion_force_traffic": ff["traffic"] if ff else None,
                "fermion_force_isolated_frac": round(iso_ff["GB/s"] / peak, 4) if iso_ff else None,
                "fp64_fma_peak_tflops": round(fma_peak, 2) if fma_peak else None,
                "clocks_during_event_pass": clocks_ev,
                "also": also, "share_of_step": shares}
    out = {
        "metric": METRIC,
        "value": round(value, 1),
        "unit": "GB/s",
        "n_gpus": world,
        "steps": args.steps,
        "warmup": args.warmup,
        "ms_per_step": round(elapsed_ms / args.steps, 3),
        "higher_is_better": True,
        "scaling": "weak",
        "vs_baseline": None,
        "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_name(args.config, dims),
                   "beta": beta, "kappa": kappa, "bc": list(bc), "dt": dt, "cg_tol": tol,
                   "cg_iters_per_step": iters, "parallelism": "replicas x%d" % world,
                   "solver": args.solver, "fermion_action": args.action, "stout_levels": args.smear,
                   "launch_path": "CUDA graphs for the CG chunks, per-kernel timing off",
                   "l2": "inputs exceed L2 (links 604 MB, each spinor 201 MB at 32^4)"},
        "gflops": round(total_flops / (elapsed_ms * 1e-3) / 1e9, 1),
        "clocks": clocks,
        "e2e": {"value": round(e2e_reals * 8 / e2e_s / 1e9, 1), "unit": "GB/s", "steps": k_e2e,
                "ms_per_step": round(e2e_s / k_e2e * 1e3, 2), "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches_all),
        "roofline": roofline,
        "peaks": peaks,
        "kernels": kernels,
    }
    if decomposed is not None:
        out["decomposed"] = decomposed
    if cfg4 is not None:
        out["configs4"] = cfg4
    if extras:
        out["extras"] = extras
    if world == 1 and not args.skip_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg, sample_iters=args.cpu_sample_iters)
    if dd_hung:
        print(json.dumps(out), flush=True)
        os._exit(0)
    dist.shutdown()
    print(json.dumps(out), flush=True)


def run_extras(args, lgt, synth, lat, cfg, hU, hP, hphi, reset_state, md_step, local, stream):
    """--extras: the non-headline arms: mixed-precision solver, even/odd action, both, one stout level; the
    decomposed path with all slabs on this GPU; the paper's own lattice sizes (24^4 force evaluation, 16^4 HMC)."""
    import torch

    ctx = lat.ctx
    dims, beta, kappa, bc = cfg["dims"], cfg["beta"], cfg["kappa"], cfg["bc"]
    tol, dt = cfg.get("cg_tol", 1e-12), cfg.get("dt", 0.01)
    V = synth.volume(dims)
    max_iter = 10 * V
    extras = {}
    a, b = event_pair()

    def timed_steps(n=2):
        reset_state()
        md_step()
        reset_state()
        torch.cuda.synchronize()
        a.record()
        its = [md_step() for _ in range(n)]
        b.record()
        torch.cuda.synchronize()
        return round(a.elapsed_time(b) / n, 3), its

    lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    ms, its = timed_steps()
    extras["mixed_precision_cg"] = {"ms_per_step": ms, "fp32_cg_iters_per_step": its, "inner_tol": 1e-5, "true_residual_tol": tol,
                                    "note": "same step and tolerance, fp32 inner CG + fp64 defect correction"}
    lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_CG)
    # even/odd preconditioned action (another pseudofermion action for the same determinant)
    lgt.lgt_set_fermion_action(ctx, lgt.LGT_ACTION_EO)
    reset_state()
    md_step()
    reset_state()
    lgt.lgt_timing_reset(ctx)
    lgt.lgt_timing_enable(ctx, True)
    torch.cuda.synchronize()
    a.record()
    eo_iters = [md_step() for _ in range(2)]
    b.record()
    torch.cuda.synchronize()
    lgt.lgt_timing_enable(ctx, False)
    hop_ms, hop_n = lgt.lgt_timing_read(ctx, lgt.LGT_K_DSLASH)
    hopr_ms, hopr_n = lgt.lgt_timing_read(ctx, lgt.LGT_K_DSLASH_R)
    lgt.lgt_timing_reset(ctx)
    hop_bytes = 2 * (8 * 9 + 12 + 12) * 8 * (V // 2)  # per half-lattice hop: 8 links + in + out per output site
    extras["even_odd_action"] = {
        "ms_per_step_with_event_pairs": round(a.elapsed_time(b) / 2, 3), "cg_iters_per_step": eo_iters,
        "hop_kernel_avg_us": round(hop_ms / max(hop_n, 1) * 1e3, 2),
        "hop_kernel_GB/s": round(hop_bytes / (hop_ms / max(hop_n, 1) * 1e-3) / 1e9, 1) if hop_n else None,
        "hop_fused_r_avg_us": round(hopr_ms / max(hopr_n, 1) * 1e3, 2),
        "note": "S_F = phi_e^dag (M^dag M)^-1 phi_e, CG on the Schur complement to the same 1e-12"}
    ms, its = timed_steps()
    extras["even_odd_action"]["ms_per_step"] = ms
    # both together: fp32 CG on the Schur complement inside an fp64 defect correction
    lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    ms, its = timed_steps()
    extras["even_odd_mixed_precision"] = {
        "ms_per_step": ms, "fp32_cg_iters_per_step": its,
        "note": "even/odd action + mixed-precision solver, true fp64 residual 1e-12: the fastest configuration of the step"}
    # the paper's motivating compositional action: the fermions on one level of stout links,
    # rho = 0.3; the step then also builds the smeared links and pulls the force back through the level
    lgt.lgt_set_smearing(ctx, 1, 0.3)
    ms, its = timed_steps()
    extras["stout_1_level_even_odd_mixed"] = {
        "ms_per_step": ms, "fp32_cg_iters_per_step": its, "rho": 0.3,
        "note": "same step with the Dirac operator on one level of stout links: smeared links rebuilt after the "
                "drift, force recursion through the level (stout_local / stout_chain kernels)"}
    lgt.lgt_set_smearing(ctx, 0, 0.0)
    lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_CG)
    lgt.lgt_set_fermion_action(ctx, lgt.LGT_ACTION_FULL)
    # the decomposed path (lgt_dd_*) on this one GPU: 1 and 4 time slabs in one process, halo exchange by device copies
    U_np, P_np, phi_np = hU.numpy(), hP.numpy(), hphi.numpy()
    for nr, halo, grid, fast in ((1, "exchange", None, False), (1, "push", None, False), (4, "exchange", None, False), (4, "overlap", None, False),
                                 (4, "half", None, False), (4, "exchange", (2, 2), False), (4, "exchange", None, True)):
        if dims[3] % nr or (dims[0] * dims[1] * dims[2]) % 32 or (grid and (dims[3] % grid[0] or dims[2] % grid[1])):
            continue
        dd = lgt.DecomposedLattice(dims, nr, list(range(nr)), beta, kappa, bc, lgt.LGT_F64, local, stream, grid=grid)
        lgt.lgt_dd_set_halo_mode(dd.d, {"push": lgt.LGT_DD_PUSH, "overlap": lgt.LGT_DD_OVERLAP, "half": lgt.LGT_DD_HALF}.get(halo, lgt.LGT_DD_EXCHANGE))
        if fast:  # the fastest configuration of the step, on slabs
            lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
            lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)

        def dd_reset():
            dd.set_links(U_np)
            dd.set_momenta(P_np)
            dd.set_pseudofermion(phi_np)

        def dd_step():
            it = lgt.lgt_dd_md_kick(dd.d, dt, tol, max_iter)
            lgt.lgt_dd_md_drift(dd.d, dt)
            return it

        dd_reset()
        dd_step()
        dd_reset()
        torch.cuda.synchronize()
        a.record()
        dd_iters = [dd_step() for _ in range(2)]
        b.record()
        torch.cuda.synchronize()
        shape = ("%dx%d_grid" % grid) if grid else "%d_slabs" % nr
        extras["decomposed_%s_%s%s_one_gpu" % (shape, halo, "_even_odd_mixed" if fast else "")] = {
            "ms_per_step": round(a.elapsed_time(b) / 2, 3), "cg_iters_per_step": dd_iters,
            "note": "same MD step through lgt_dd_* with %s resident on this GPU, halo mode %s: the cost of the "
                    "ghost slices, halo traffic and split reductions, not a multi-GPU number" %
                    (("a %d x %d (t, z) grid of ranks" % grid) if grid else "%d time slab(s)" % nr, halo)}
        dd.close()
        del dd

    # the paper's own timing workload (Table I: one Wilson-fermion force evaluation at 24^4;
    # 3.39 s / 4.61 s on an H100 through JACC.jl, kappa and solver tolerance not stated): context, not a baseline
    d24 = (24, 24, 24, 24)
    c24 = dict(cfg, dims=d24, seed_links=2401)
    lat24 = lgt.Lattice(d24, beta, kappa, bc, lgt.LGT_F64, local, stream)
    lat24.set_links(synth.config_links(c24))
    eta24 = lat24.to_device(synth.gaussian_spinor(d24, 2402))
    phi24 = lat24.empty(synth.volume(d24), 4, 3)
    lgt.lgt_dslash(lat24.ctx, eta24, phi24, True)
    lgt.lgt_set_pseudofermion(lat24.ctx, phi24)
    F24 = lat24.empty(synth.volume(d24), 4, 3, 3)
    t24 = {}
    for name, solver, action in (("plain_fp64_cg", lgt.LGT_SOLVER_CG, lgt.LGT_ACTION_FULL),
                                 ("even_odd_mixed", lgt.LGT_SOLVER_MIXED_CG, lgt.LGT_ACTION_EO)):
        lgt.lgt_set_solver(lat24.ctx, solver, 1e-5)
        lgt.lgt_set_fermion_action(lat24.ctx, action)
        if action == lgt.LGT_ACTION_EO:
            lgt.lgt_pseudofermion_heatbath(lat24.ctx, 24, 0)
        lgt.lgt_fermion_force(lat24.ctx, None, None, F24, tol, max_iter)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        it24 = [lgt.lgt_fermion_force(lat24.ctx, None, None, F24, tol, max_iter) for _ in range(3)]
        torch.cuda.synchronize()
        t24[name] = {"ms": round((time.perf_counter() - t0) / 3 * 1e3, 2), "cg_iters": it24[0]}
    extras["paper_table1_workload_24^4"] = {
        "one_fermion_force_evaluation": t24, "kappa": kappa, "cg_tol": tol,
        "paper_H100_s": {"hand_written": 4.61, "llvm_ad": 3.39},
        "note": "wall clock incl. the solve, warm links eps = 0.3; the paper states neither kappa nor the solver tolerance, "
                "so this is context (PAPER.md:143-148), not a like-for-like ratio"}
    lat24.close()

    # the whole method end to end on the paper's other lattice size: HMC trajectories at 16^4 with everything on
    d16 = (16, 16, 16, 16)
    lat16 = lgt.Lattice(d16, beta, kappa, bc, lgt.LGT_F64, local, stream)
    lat16.set_links(synth.warm_links(d16, 0.3, 1601))
    lgt.lgt_set_fermion_action(lat16.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(lat16.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    lgt.lgt_set_smearing(lat16.ctx, 1, 0.3)
    lgt.lgt_set_integrator(lat16.ctx, lgt.LGT_INT_SEXTON_WEINGARTEN, 10)
    lgt.lgt_hmc_trajectory(lat16.ctx, 10, 0.02, 16, 0, tol=1e-10)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res16 = [lgt.lgt_hmc_trajectory(lat16.ctx, 10, 0.02, 16, t, tol=1e-10) for t in range(1, 5)]
    torch.cuda.synchronize()
    extras["hmc_trajectory_16^4"] = {
        "ms_per_trajectory": round((time.perf_counter() - t0) / 4 * 1e3, 2), "md_steps": 10, "dt": 0.02,
        "dH": [round(r[0], 4) for r in res16], "accepted": [bool(r[1]) for r in res16], "cg_iters": [r[2] for r in res16],
        "plaquette": round(lgt.lgt_plaquette(lat16.ctx), 5),
        "note": "heat baths, even/odd action, mixed-precision solver (true residual 1e-10), one stout level rho = 0.3, "
                "Sexton-Weingarten with 10 inner gauge steps, Metropolis: the paper's second HMC set-up (PAPER.md:154-156) at 16^4"}
    lat16.close()
    return extras


# ------------------------------------------------------------------------------------------------ the oracle, timed
def oracle_step(oracle, cfg, U, P, phi, sample_iters):
    """One bounded sample of the MD step on the CPU oracle: same kick + drift, CG capped at sample_iters."""
    dims, beta, kappa, bc = cfg["dims"], cfg["beta"], cfg["kappa"], cfg["bc"]
    t0 = time.perf_counter()
    P1, it, _ = oracle.kick(dims, beta, kappa, bc, U, phi, P, cfg.get("dt", 0.01), cfg.get("cg_tol", 1e-12), sample_iters)
    oracle.drift(dims, cfg.get("dt", 0.01), P1, U)
    return time.perf_counter() - t0, it


def oracle_kernels(oracle, cfg, U, eta, phi):
    """The metric's two named kernels on the oracle alone: one Dslash and one fermion force on given
    spinor fields, with all host threads and with one (the paper's CPU column is single-threaded)."""
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    V = 1
    for d in dims:
        V *= d
    n_all, out = oracle.num_threads(), {}
    try:
        for threads in sorted({n_all, 1}, reverse=True):
            oracle.set_num_threads(threads)
            for name, fn in (("dslash", lambda: oracle.dslash(dims, kappa, bc, U, eta)),
                             ("fermion_force", lambda: oracle.fermion_force(dims, kappa, bc, U, eta, phi))):
                best = float("inf")
                for _ in range(2):
                    t0 = time.perf_counter()
                    fn()
                    best = min(best, time.perf_counter() - t0)
                out["%s_%d_threads" % (name, threads)] = {"ms": round(best * 1e3, 1),
                                                           "GB/s": round(REALS[name] * 8 * V / best / 1e9, 3),
                                                           "GFLOP/s": round(FLOPS[name] * V / best / 1e9, 2)}
    finally:
        oracle.set_num_threads(n_all)
    return out


def cpu_baseline(cfg, sample_iters, steps=1, warmup=0, per_kernel=True):
    import oracle
    from paper_2602_20516_b200 import synth

    V = synth.volume(cfg["dims"])
    U, P, eta = make_inputs(cfg)
    phi = oracle.dslash(cfg["dims"], cfg["kappa"], cfg["bc"], U, eta, dagger=True)
    for _ in range(warmup):
        oracle_step(oracle, cfg, U, P, phi, sample_iters)
    t, reals = 0.0, 0
    for _ in range(steps):
        dt_s, it = oracle_step(oracle, cfg, U, P, phi, sample_iters)
        t += dt_s
        reals += step_reals(it) * V
    return {"value": round(reals * 8 / t / 1e9, 3), "unit": "GB/s", "cores": oracle.num_threads(), "kind": "oracle",
            "seconds_per_sample": round(t / steps, 2), "kernels": oracle_kernels(oracle, cfg, U, eta, phi) if per_kernel else None,
            "sample": "same %s lattice and fields; one MD step with CG capped at %d iterations "
                      "(gauge force + %d x (2 Dslash + BLAS-1) + Y = D X + fermion force + drift), same byte accounting"
                      % ("x".join(map(str, cfg["dims"])), sample_iters, sample_iters)}


# ------------------------------------------------------------------------------------------------ one lattice on N GPUs
def decomposed_steps(args, rank, world, local, steps, warmup, with_e2e=True):
    """ONE lattice cut into `world` time slabs (lgt_dd_*): the same MD step, every rank its slab.  Returns rank 0's result
    dict (None elsewhere).  Transport: the library's NCCL communicator, or with --transport host gloo through host memory
    (--same-gpu puts every rank on cuda:0 -- the only way to run the inter-process path on a one-GPU box)."""
    import torch

    from paper_2602_20516_b200 import dist, lgt, synth

    torch.cuda.set_device(local)  # the current device is per thread, and the guarded leg runs in one
    cfg = dict(synth.CONFIGS[args.config])
    if args.lattice:
        cfg["dims"] = tuple(args.lattice)
    dims, beta, kappa, bc = cfg["dims"], cfg["beta"], cfg["kappa"], cfg["bc"]
    tol, dt = cfg.get("cg_tol", 1e-12), cfg.get("dt", 0.01)
    V = synth.volume(dims)
    max_iter = 10 * V
    U, P, eta = make_inputs(cfg)  # every rank draws the same global fields and keeps its slab
    stream = torch.cuda.current_stream().cuda_stream
    grid = tuple(args.grid) if args.grid else None
    if grid is not None and grid[0] * grid[1] != world:
        raise SystemExit("--grid PT PZ needs PT * PZ = the number of ranks")
    dd = dist.decomposed_lattice(dims, beta, kappa, bc, lgt.LGT_F64, local, stream, halo=args.halo, transport=args.transport, grid=grid)
    if args.action == "eo":
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    if args.solver == "mixed":
        lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    if args.smear:
        lgt.lgt_dd_set_smearing(dd.d, args.smear, 0.3)
    import numpy as np

    mine = (lambda a: np.ascontiguousarray(dd.slab(a, rank)))  # this rank's time slab, or its (t, z) block on a grid
    hU, hP = torch.from_numpy(mine(U)).pin_memory(), torch.from_numpy(mine(P)).pin_memory()
    ctx = dd.ranks[0]
    lgt.lgt_set_links_host(ctx, hU)
    d_eta = torch.from_numpy(mine(eta)).cuda()
    d_phi = torch.empty_like(d_eta)
    lgt.lgt_dd_dslash(dd.d, [d_eta], [d_phi], True)
    hphi = d_phi.cpu().pin_memory()
    hU_out, hP_out = torch.empty_like(hU).pin_memory(), torch.empty_like(hP).pin_memory()
    del U, P, eta, d_eta

    def reset_state():
        lgt.lgt_set_links_host(ctx, hU)
        lgt.lgt_set_momenta_host(ctx, hP)
        lgt.lgt_set_pseudofermion_host(ctx, hphi)

    def md_step():
        it = lgt.lgt_dd_md_kick(dd.d, dt, tol, max_iter)
        lgt.lgt_dd_md_drift(dd.d, dt)
        return it

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    reset_state()
    for _ in range(warmup):
        md_step()
    sampler = ClockSampler(local)
    launches0 = lgt.lgt_launch_count(ctx)
    e0, e1 = event_pair()
    sampler.start()
    barrier()
    e0.record()
    iters = [md_step() for _ in range(steps)]
    e1.record()
    barrier()
    clocks = sampler.stop()
    elapsed_ms = e0.elapsed_time(e1)
    launches = lgt.lgt_launch_count(ctx) - launches0
    k_e2e, e2e_s, e2e_iters = max(1, min(steps, 3)), 0.0, []
    if with_e2e:
        barrier()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            reset_state()
            e2e_iters.append(md_step())
            lgt.lgt_get_links_host(ctx, hU_out)
            lgt.lgt_get_momenta_host(ctx, hP_out)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
    on_cpu = args.transport == "host"
    (elapsed_ms, e2e_s), (launches_all,) = dist.aggregate([elapsed_ms, e2e_s], [launches], device="cpu" if on_cpu else "cuda")
    dd.close()
    if rank != 0:
        return None
    total_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in iters) * V  # the whole lattice: strong scaling
    res = {"value": round(total_reals * 8 / (elapsed_ms * 1e-3) / 1e9, 1), "unit": "GB/s", "ms_per_step": round(elapsed_ms / steps, 3),
           "steps": steps, "cg_iters_per_step": iters, "gpu_launches": int(launches_all), "clocks": clocks,
           "parallelism": "dd%d: ONE %s lattice in %s, halo %s, transport %s%s" %
                          (world, "x".join(map(str, dims)), ("a %d x %d (t, z) grid" % grid) if grid else "%d time slabs" % world, args.halo,
                           args.transport, ", every rank on cuda:0" if args.same_gpu else "")}
    if with_e2e:
        e2e_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in e2e_iters) * V
        res["e2e"] = {"value": round(e2e_reals * 8 / e2e_s / 1e9, 1), "unit": "GB/s", "steps": k_e2e, "ms_per_step": round(e2e_s / k_e2e * 1e3, 2),
                      "h2d_bytes_per_step": (hU.numel() + hP.numel() + hphi.numel()) * 16 * world,
                      "d2h_bytes_per_step": (hU_out.numel() + hP_out.numel()) * 16 * world}
    return res


def guarded_decomposed_leg(args, rank, world, local):
    """The decomposed step as an extra inside the default N > 1 run.  The inter-process NCCL path has never run on more than
    one GPU (no multi-GPU box existed while this was written), so a watchdog bounds it: if it has not finished within
    --dd-leg-timeout seconds the process reports that and the headline line is printed without it."""
    result, done = {}, threading.Event()

    def work():
        try:
            result["res"] = decomposed_steps(args, rank, world, local, steps=max(1, min(args.steps, 3)), warmup=1, with_e2e=False)
        except Exception as e:
            result["res"] = {"error": "%s: %s" % (type(e).__name__, e)}
        done.set()

    t = threading.Thread(target=work, daemon=True)
    t.start()
    if not done.wait(args.dd_leg_timeout):
        return {"error": "timed out after %d s (the other legs of this line are unaffected)" % args.dd_leg_timeout}
    return result.get("res")


def run_decomposed(args):
    """--parallelism dd: ONE configs[3] lattice cut into N time slabs (lgt_dd_*), strong scaling, as the headline."""
    import torch

    from paper_2602_20516_b200 import dist, lgt, synth

    rank, world, local = dist.env_rank_world()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    if args.same_gpu:
        local = 0
    torch.cuda.set_device(local)
    if args.nccl_debug:
        os.environ.setdefault("NCCL_DEBUG", "INFO")  # leaves the communicator lines ("comm ... rank r nranks N") in the output
    dist.init("gloo" if args.transport == "host" else "nccl", None if args.transport == "host" else torch.device("cuda", local))
    lgt.lib()
    cfg = dict(synth.CONFIGS[args.config])
    dims = tuple(args.lattice) if args.lattice else cfg["dims"]
    res = decomposed_steps(args, rank, world, local, args.steps, args.warmup)
    if rank == 0:
        out = {
            "metric": METRIC, "value": res["value"], "unit": "GB/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": res["ms_per_step"],
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config, dims) + "; " + res["parallelism"],
                       "beta": cfg["beta"], "kappa": cfg["kappa"], "bc": list(cfg["bc"]), "dt": cfg.get("dt", 0.01),
                       "cg_tol": cfg.get("cg_tol", 1e-12), "cg_iters_per_step": res["cg_iters_per_step"],
                       "parallelism": res["parallelism"], "solver": args.solver, "fermion_action": args.action,
                       "stout_levels": args.smear,
                       "l2": "inputs exceed L2 at 32^4 up to 8 slabs (links 604 MB / N per rank)"},
            "clocks": res["clocks"], "e2e": res.get("e2e"), "gpu_launches": res["gpu_launches"],
        }
        print(json.dumps(out), flush=True)
    dist.shutdown()


def run_reference(args):
    from paper_2602_20516_b200 import dist, synth

    rank, world, _ = dist.env_rank_world()
    if rank != 0:
        return

    cfg = dict(synth.CONFIGS[args.config])
    if args.lattice:
        cfg["dims"] = tuple(args.lattice)
    t0 = time.perf_counter()
    base = cpu_baseline(cfg, args.cpu_sample_iters, steps=args.steps, warmup=args.warmup, per_kernel=False)
    out = {
        "impl": "reference", "metric": METRIC, "value": base["value"], "unit": "GB/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(base["seconds_per_sample"] * 1e3, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(args.config, cfg["dims"]),
                   "beta": cfg["beta"], "kappa": cfg["kappa"], "bc": list(cfg["bc"]), "dt": cfg.get("dt", 0.01),
                   "cg_tol": cfg.get("cg_tol", 1e-12), "sample": base["sample"]},
        "cpu_baseline": base,
        "e2e": {"value": base["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "wall_s": round(time.perf_counter() - t0, 1),
    }
    print(json.dumps(out), flush=True)


def run_peaks(args):
    """--peaks: the measured roofline denominators only (fp64 and fp32 FMA peak, copy bandwidth), one JSON line."""
    import torch

    from paper_2602_20516_b200 import lgt

    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    sampler.start()
    out = {}
    for prec, tag in ((lgt.LGT_F64, "f64"), (lgt.LGT_F32, "f32")):
        lat = lgt.Lattice((32, 32, 32, 32), 5.6, 0.12, (1, 1, 1, -1), prec, 0, torch.cuda.current_stream().cuda_stream)
        out[tag] = lgt.lgt_measure_peaks(lat.ctx, 50)
        lat.close()
    out["clocks"] = sampler.stop()
    out["how"] = ("lgt_measure_peaks: 8 independent FMA chains per thread, 8 x 256 threads per SM, 2 flops per FMA; plain copy of the "
                  "native link field (604 / 302 MB), read + write bytes; CUDA events, 50 launches, best and mean")
    print(json.dumps({"peaks": out}), flush=True)


def run_kernel_variants(args):
    """`--kernel-variants`: the alternative implementations kept in the library (lgt_set_kernel_variant) on the headline
    lattice, one after another in one process: isolated launches (CUDA events, inputs exceed L2), one CG solve each, and
    whether the results equal variant 0's bit for bit.  This is the command behind profiles/r02*_variants.md."""
    import torch

    from paper_2602_20516_b200 import lgt, synth

    torch.cuda.set_device(0)
    cfg = dict(synth.CONFIGS[args.config])
    if args.lattice:
        cfg["dims"] = tuple(args.lattice)
    dims, kappa, bc = cfg["dims"], cfg["kappa"], cfg["bc"]
    V = synth.volume(dims)
    U, _, eta = make_inputs(cfg)
    f32 = args.variant_precision == "f32"
    if f32 and args.variant_class != "dslash":
        raise SystemExit("--variant-precision f32 is for --variant-class dslash")
    lat = lgt.Lattice(dims, cfg["beta"], kappa, bc, lgt.LGT_F32 if f32 else lgt.LGT_F64, 0, torch.cuda.current_stream().cuda_stream)
    ctx = lat.ctx
    lgt.lgt_set_links_host(ctx, torch.from_numpy(U.astype("complex64") if f32 else U).pin_memory())
    nat = [lat.native_spinor() for _ in range(4)]
    lgt.lgt_spinor_to_native(ctx, lat.to_device(eta), nat[0])
    del U, eta
    esize = 4 if f32 else 8
    cg_tol = 1e-5 if f32 else cfg.get("cg_tol", 1e-12)
    out = {"lattice": "x".join(map(str, dims)), "dtype": "f32" if f32 else "f64", "kernel_class": args.variant_class, "variants": {}}
    kclass = lgt.KERNEL_CLASSES.index(args.variant_class)
    ref = {}
    names = VARIANT_NAMES[args.variant_class]
    only = [int(v) for v in args.only_variants.split(",")] if args.only_variants else range(len(names))
    for v in only:
        lgt.lgt_set_kernel_variant(ctx, kclass, v)
        res = {"what": names[v]}
        if args.variant_class == "dslash":
            for dag in (False, True):
                t = time_calls(lambda: lgt.lgt_dslash_native(ctx, nat[0], nat[1], dag), n=args.variant_launches,
                               warm=min(5, args.variant_launches))
                key = "dslash_dagger" if dag else "dslash"
                res[key] = {"us": round(t * 1e6, 1), "GB/s": round(REALS["dslash"] * esize * V / t / 1e9, 1)}
                got = nat[1].clone()
                res[key]["bitwise_variant0"] = bool(torch.equal(got, ref.setdefault(key, got)))
            if args.variant_no_cg:  # ncu captures: the isolated launches only
                out["variants"][str(v)] = res
                continue
            lgt.lgt_dslash_native(ctx, nat[0], nat[2], True)  # phi = D^dag eta
            for _ in range(2):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                it, rel, ok = lgt.lgt_cg_native(ctx, nat[2], nat[3], None, cg_tol, 10 * V)
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
            got = nat[3].clone()
            res["cg"] = {"iters": it, "converged": ok, "us_per_iter": round(dt * 1e6 / max(it, 1), 1),
                         "bitwise_variant0": bool(torch.equal(got, ref.setdefault("x", got)))}
        else:
            lgt.lgt_set_momenta_host(ctx, torch.zeros((V, 4, 3, 3), dtype=torch.complex128).pin_memory())
            t = time_calls(lambda: lgt.lgt_gauge_force_accumulate(ctx, 1e-3), n=args.variant_launches,
                           warm=min(5, args.variant_launches))
            res["gauge_force"] = {"us": round(t * 1e6, 1), "GB/s": round(REALS["gauge_force"] * 8 * V / t / 1e9, 1),
                                  "GFLOP/s": round(FLOPS["gauge_force"] * V / t / 1e9, 1)}
            lgt.lgt_set_momenta_host(ctx, torch.zeros((V, 4, 3, 3), dtype=torch.complex128).pin_memory())
            lgt.lgt_gauge_force_accumulate(ctx, 1.0)
            got = torch.empty((V, 4, 3, 3), dtype=torch.complex128, device="cuda")
            lgt.lgt_get_momenta(ctx, got)
            base = ref.setdefault("F", got)
            res["gauge_force"]["max_abs_diff_variant0"] = float((got - base).abs().max())
        out["variants"][str(v)] = res
    lat.close()
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (3 = 32^4 MD step)")
    ap.add_argument("--lattice", type=int, nargs=4, default=None, help="override dims (debugging only)")
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="profiling runs only: leave the oracle leg out")
    ap.add_argument("--solver", default="cg", choices=["cg", "mixed"],
                    help="non-default: time the step with the mixed-precision solver (not the headline configuration)")
    ap.add_argument("--action", default="full", choices=["full", "eo"],
                    help="non-default: time the step with the even/odd preconditioned action (not the headline configuration)")
    ap.add_argument("--halo", default="exchange", choices=["exchange", "push", "overlap", "half"],
                    help="decomposed lattice: separate exchange of the halo slices, or halos stored into the neighbours' ghost "
                         "slices by the Dslash kernels (CUDA IPC between processes)")
    ap.add_argument("--transport", default="nccl", choices=["nccl", "host"],
                    help="decomposed lattice: the library's NCCL communicator, or gloo through host memory (lgt_dd_set_host_transport)")
    ap.add_argument("--same-gpu", action="store_true",
                    help="--parallelism dd --transport host only: every rank on cuda:0 (runs the inter-process path on a one-GPU box)")
    ap.add_argument("--grid", type=int, nargs=2, default=None, metavar=("PT", "PZ"),
                    help="--parallelism dd: two split directions (lgt_dd_create_grid), PT * PZ = ranks; default: time slabs")
    ap.add_argument("--nccl-debug", action="store_true", help="--parallelism dd: NCCL_DEBUG=INFO, so that the output shows every rank's communicator")
    ap.add_argument("--smear", type=int, default=0,
                    help="non-default: the fermions see this many levels of stout-smeared links (rho = 0.3); not the headline")
    ap.add_argument("--extras", action="store_true", help="also time the non-headline arms (solvers, stout, slabs on one GPU, 24^4, 16^4 HMC)")
    ap.add_argument("--skip-extras", action="store_true", help="(default now; kept for old command lines)")
    ap.add_argument("--skip-config4", action="store_true", help="leave the 48^3 x 96 sweep (configs[4]) out")
    ap.add_argument("--skip-dd-leg", action="store_true", help="N > 1: leave the decomposed-lattice pass out of the replicas run")
    ap.add_argument("--dd-leg-timeout", type=int, default=240)
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "dd"],
                    help="N > 1: 'replicas' = N independent lattices (default, weak scaling, plus one guarded decomposed pass); "
                         "'dd' = ONE lattice cut into N time slabs (lgt_dd_*, strong scaling) as the headline")
    ap.add_argument("--cpu-sample-iters", type=int, default=20, help="CG iterations in the oracle's bounded sample")
    ap.add_argument("--kernel-variants", action="store_true",
                    help="time every implementation variant of one kernel class on the headline lattice (profiles/r02*_variants.md)")
    ap.add_argument("--variant-class", default="dslash", choices=sorted(VARIANT_NAMES))
    ap.add_argument("--only-variants", default="", help="comma-separated variant numbers (default: all)")
    ap.add_argument("--variant-launches", type=int, default=20)
    ap.add_argument("--variant-precision", default="f64", choices=["f64", "f32"],
                    help="--kernel-variants --variant-class dslash: precision of the handle (f32: CG to 1e-5)")
    ap.add_argument("--variant-no-cg", action="store_true", help="--kernel-variants: isolated launches only (for ncu captures)")
    ap.add_argument("--peaks", action="store_true", help="print the measured fp64 / fp32 FMA and copy peaks and exit")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.same_gpu and args.transport != "host":
        ap.error("--same-gpu needs --transport host (NCCL refuses two ranks on one device)")
    if args.peaks:
        run_peaks(args)
    elif args.kernel_variants:
        run_kernel_variants(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.parallelism == "dd":
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
