#!/usr/bin/env python
"""bench.py -- one JSON line for the HMC MD-step hot path on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one molecular-dynamics step of BASELINE.json configs[3] in the reading DESIGN.md A-13:
kick(dt) = gauge force + CG on D^dag D to 1e-12 + Y = D X + fused fermion force, then drift(dt) = link update,
on a 32^4 SU(3) lattice in fp64 (beta 5.6, kappa 0.12, antiperiodic time, dt 0.01, seeded warm-start links).
`value` is the algorithmic HBM traffic of all kernels of the step divided by
the device time of the step; `kernels` holds the metric's two named kernels (Dslash, fermion force) timed
in isolation; `roofline` is the dominant kernel (Dslash inside CG) timed in place with CUDA events.
N > 1: N independent replicas (one lattice per GPU, no data-path collective), weak scaling.
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

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the ncu --set full capture
# summarised in profiles/ (None until captured for the current kernel).
NCU_TRAFFIC_BYTES = {"dslash_f64_32^4": 1019771616}  # profiles/r01f_ncu_cg.md, dslash_kernel<double,0,1,0>: 1.0198 GB


# even/odd action, per site of the FULL lattice: a half-lattice hop reads 8 links + 1 spinor and writes 1 spinor per
# output site, and there are V/2 output sites
REALS_EO = dict(hop=(2 * (72 + 12 + 12)) // 2, hop_fused_r=(2 * (72 + 12 + 2 * 12)) // 2, update_xp=(2 * 5 * 12) // 2)
REALS_EO["cg_iter"] = 3 * REALS_EO["hop"] + REALS_EO["hop_fused_r"] + REALS_EO["update_xp"]   # -> 3408 B fp64


# one stout level, forward (staples -> A, exp(A) U -> U') and backward (local: A, F' rw, G; chain: U, G, Fdir, out rw)
REALS_STOUT_LEVEL = (2 * 36 + 32) + (32 + 2 * 2 * 36) + (32 + 2 * 32 + 32) + (2 * 36 + 32 + 32 + 2 * 32)


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


def measured_peaks():
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

    # ---- timed region: K steps, device time by CUDA events on the handle's stream, max over ranks
    sampler = ClockSampler(local)
    lgt.lgt_timing_reset(ctx)
    lgt.lgt_timing_enable(ctx, True)
    launches0 = lgt.lgt_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    barrier()
    e0.record()
    iters = [md_step() for _ in range(args.steps)]
    e1.record()
    barrier()
    clocks = sampler.stop()
    lgt.lgt_timing_enable(ctx, False)
    elapsed_ms = e0.elapsed_time(e1)
    launches = lgt.lgt_launch_count(ctx) - launches0
    per_class = {name: lgt.lgt_timing_read(ctx, k) for k, name in enumerate(lgt.KERNEL_CLASSES)}
    lgt.lgt_timing_reset(ctx)
    total_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in iters) * V
    total_flops = sum(step_flops(i) for i in iters) * V

    # ---- end to end: host buffers in, host buffers out, through the C ABI, every step
    k_e2e = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    e2e_iters = []
    for _ in range(k_e2e):
        reset_state()
        e2e_iters.append(md_step())
        lgt.lgt_get_links_host(ctx, hU_out)
        lgt.lgt_get_momenta_host(ctx, hP_out)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in e2e_iters) * V
    h2d = hU.numel() * 16 + hP.numel() * 16 + hphi.numel() * 16
    d2h = hU_out.numel() * 16 + hP_out.numel() * 16

    # ---- the same MD step with the mixed-precision solver; not the headline: `value` stays pure fp64
    extras = {}
    if rank == 0 and not args.skip_extras and not variant:
        lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
        reset_state()
        md_step()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reset_state()
        torch.cuda.synchronize()
        a.record()
        mixed_iters = [md_step() for _ in range(2)]
        b.record()
        torch.cuda.synchronize()
        extras["mixed_precision_cg"] = {"ms_per_step": round(a.elapsed_time(b) / 2, 3), "fp32_cg_iters_per_step": mixed_iters,
                                        "inner_tol": 1e-5, "true_residual_tol": tol,
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
            "ms_per_step": round(a.elapsed_time(b) / 2, 3), "cg_iters_per_step": eo_iters,
            "hop_kernel_avg_us": round(hop_ms / max(hop_n, 1) * 1e3, 2),
            "hop_kernel_GB/s": round(hop_bytes / (hop_ms / max(hop_n, 1) * 1e-3) / 1e9, 1) if hop_n else None,
            "hop_fused_r_avg_us": round(hopr_ms / max(hopr_n, 1) * 1e3, 2),
            "note": "S_F = phi_e^dag (M^dag M)^-1 phi_e, CG on the Schur complement to the same 1e-12"}
        # both together: fp32 CG on the Schur complement inside an fp64 defect correction
        lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
        reset_state()
        md_step()
        reset_state()
        torch.cuda.synchronize()
        a.record()
        eom_iters = [md_step() for _ in range(2)]
        b.record()
        torch.cuda.synchronize()
        extras["even_odd_mixed_precision"] = {
            "ms_per_step": round(a.elapsed_time(b) / 2, 3), "fp32_cg_iters_per_step": eom_iters,
            "note": "even/odd action + mixed-precision solver, true fp64 residual 1e-12: the fastest configuration of the step"}
        if not args.smear:
            # the paper's motivating compositional action: the fermions on one level of stout links,
            # rho = 0.3; the step then also builds the smeared links and pulls the force back through the level
            lgt.lgt_set_smearing(ctx, 1, 0.3)
            reset_state()
            md_step()
            reset_state()
            torch.cuda.synchronize()
            a.record()
            st_iters = [md_step() for _ in range(2)]
            b.record()
            torch.cuda.synchronize()
            extras["stout_1_level_even_odd_mixed"] = {
                "ms_per_step": round(a.elapsed_time(b) / 2, 3), "fp32_cg_iters_per_step": st_iters, "rho": 0.3,
                "note": "same step with the Dirac operator on one level of stout links: smeared links rebuilt after the "
                        "drift, force recursion through the level (stout_local / stout_chain kernels)"}
            lgt.lgt_set_smearing(ctx, 0, 0.0)
        lgt.lgt_set_solver(ctx, lgt.LGT_SOLVER_CG)
        lgt.lgt_set_fermion_action(ctx, lgt.LGT_ACTION_FULL)
        # the decomposed path (lgt_dd_*) on this one GPU: 1 and 4 time slabs in one process, halo exchange by device copies
        import numpy as np
        U_np, P_np, phi_np = hU.numpy(), hP.numpy(), hphi.numpy()
        for nr, halo in ((1, "exchange"), (1, "push"), (4, "exchange")):
            if dims[3] % nr or (dims[0] * dims[1] * dims[2]) % 32:
                continue
            dd = lgt.DecomposedLattice(dims, nr, list(range(nr)), beta, kappa, bc, lgt.LGT_F64, local, stream)
            lgt.lgt_dd_set_halo_mode(dd.d, lgt.LGT_DD_PUSH if halo == "push" else lgt.LGT_DD_EXCHANGE)

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
            extras["decomposed_%d_slabs_%s_one_gpu" % (nr, halo)] = {
                "ms_per_step": round(a.elapsed_time(b) / 2, 3), "cg_iters_per_step": dd_iters,
                "note": "same MD step through lgt_dd_* with %d time slab(s) resident on this GPU, halo mode %s: the cost of the "
                        "ghost slices, halo traffic and split reductions, not a multi-GPU number" % (nr, halo)}
            dd.close()
            del dd

    # ---- the paper's own timing workload (Table I: one Wilson-fermion force evaluation at 24^4;
    # 3.39 s / 4.61 s on an H100 through JACC.jl, kappa and solver tolerance not stated): context, not a baseline
    if rank == 0 and not args.skip_extras and not variant:
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

    # ---- the whole method end to end on the paper's other lattice size: HMC trajectories at 16^4 with everything on
    if rank == 0 and not args.skip_extras and not variant:
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

    # ---- max over ranks, aggregate
    (elapsed_ms, e2e_s), (total_reals, total_flops, e2e_reals, launches_all) = dist.aggregate(
        [elapsed_ms, e2e_s], [total_reals, total_flops, e2e_reals, launches], device="cuda")

    # ---- the metric's two kernels in isolation (inputs exceed L2: links 604 MB, spinors 201 MB each)
    kernels = {}

    def time_kernel(fn, n=20, warm=5):
        for _ in range(warm):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(n):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n * 1e-3

    def isolated(handle, real_bytes, tag):
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
            t = time_kernel(fn)
            kernels[name + tag] = {"us": round(t * 1e6, 2), "GB/s": round(REALS[key] * real_bytes * V / t / 1e9, 1),
                                   "GFLOP/s": round(FLOPS[key] * V / t / 1e9, 1)}

    if rank == 0:
        isolated(lat, 8, "_f64")
        lat32 = lgt.Lattice(dims, beta, kappa, bc, lgt.LGT_F32, local, stream)
        lgt.lgt_get_links(ctx, d_U := lat.empty(V, 4, 3, 3))
        lgt.lgt_set_links(lat32.ctx, d_U.to(torch.complex64))
        del d_U
        isolated(lat32, 4, "_f32")
        lat32.close()

    if rank != 0:
        lat.close()
        dist.shutdown()
        return

    peak, peak_src = measured_peaks()
    ds_ms, ds_n = per_class["dslash"]
    ds_avg_s = ds_ms / max(ds_n, 1) * 1e-3
    ds_bytes = (REALS_EO["hop"] if args.action == "eo" else REALS["dslash"]) * (4 if args.solver == "mixed" else 8) * V
    achieved = ds_bytes / ds_avg_s / 1e9 if ds_n else None
    shares = {name: round(ms / elapsed_ms, 4) for name, (ms, n) in per_class.items() if n}
    in_place = {}
    for name, key in (("dslash", "dslash"), ("dslash_dag_fused_r", "dslash_fused_r"), ("cg_blas1", "cg_update_xp"),
                      ("fermion_force", "fermion_force"), ("gauge_force", "gauge_force"), ("link_update", "link_update")):
        ms, n = per_class[name]
        if n:
            in_place[name] = {"launches": n, "avg_us": round(ms / n * 1e3, 2),
                              "GB/s": round(REALS[key] * 8 * V / (ms / n * 1e-3) / 1e9, 1)}
    value = total_reals * 8 / (elapsed_ms * 1e-3) / 1e9
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
        "config": {"workload": "configs[%d]: %s SU(3) one MD step = kick(dt) [gauge force, CG 1e-12 on D^dag D, Y = D X, "
                               "fermion force] + drift(dt)" % (args.config, "x".join(map(str, dims))),
                   "beta": beta, "kappa": kappa, "bc": list(bc), "dt": dt, "cg_tol": tol,
                   "cg_iters_per_step": iters, "parallelism": "replicas x%d" % world,
                   "solver": args.solver, "fermion_action": args.action, "stout_levels": args.smear,
                   "l2": "inputs exceed L2 (links 604 MB, each spinor 201 MB at 32^4)"},
        "gflops": round(total_flops / (elapsed_ms * 1e-3) / 1e9, 1),
        "clocks": clocks,
        "e2e": {"value": round(e2e_reals * 8 / e2e_s / 1e9, 1), "unit": "GB/s", "steps": k_e2e,
                "ms_per_step": round(e2e_s / k_e2e * 1e3, 2), "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches_all),
        "roofline": {"kernel": ("hop_cb_kernel<float> (mostly inside the fp32 CG, %d launches)" if args.action == "eo" and args.solver == "mixed" else
                                "hop_cb_kernel<double> (inside CG, %d launches)" if args.action == "eo" else
                                "dslash_kernel<float> (inside the fp32 CG, %d launches)" if args.solver == "mixed" else
                                "dslash_kernel<double> (inside CG, %d launches)") % ds_n, "bound": "hbm",
                     "achieved": round(achieved, 1) if achieved else None, "peak": peak, "unit": "GB/s",
                     "frac": round(achieved / peak, 4) if achieved else None,
                     "frac_of_nominal_8TBs": round(achieved / 8000.0, 4) if achieved else None,
                     "peak_source": peak_src, "avg_launch_us": round(ds_avg_s * 1e6, 2),
                     "algorithmic_bytes_per_launch": ds_bytes,
                     "traffic": NCU_TRAFFIC_BYTES.get("dslash_f64_32^4") if tuple(dims) == (32, 32, 32, 32) and not variant else None,
                     "share_of_step": shares, "kernels_in_place": in_place},
        "kernels": kernels,
        "extras": extras,
    }
    if world == 1 and not args.skip_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(cfg, sample_iters=args.cpu_sample_iters)
    lat.close()
    dist.shutdown()
    print(json.dumps(out), flush=True)


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
def run_decomposed(args):
    """--parallelism dd: ONE configs[3] lattice cut into N time slabs (lgt_dd_*), strong scaling.  The same MD step, the
    same byte accounting for the whole lattice; halo slices and CG sums go over the library's NCCL communicator.
    Verified on one GPU only (all slabs in one process, and NCCL with a single rank): DESIGN.md "Multi-GPU"."""
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
    dims, beta, kappa, bc = cfg["dims"], cfg["beta"], cfg["kappa"], cfg["bc"]
    tol, dt = cfg.get("cg_tol", 1e-12), cfg.get("dt", 0.01)
    V = synth.volume(dims)
    max_iter = 10 * V
    U, P, eta = make_inputs(cfg)  # every rank draws the same global fields and keeps its slab
    stream = torch.cuda.current_stream().cuda_stream
    dd = dist.decomposed_lattice(dims, beta, kappa, bc, lgt.LGT_F64, local, stream, halo=args.halo)
    if args.action == "eo":
        lgt.lgt_dd_set_fermion_action(dd.d, lgt.LGT_ACTION_EO)
    if args.solver == "mixed":
        lgt.lgt_dd_set_solver(dd.d, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    if args.smear:
        lgt.lgt_dd_set_smearing(dd.d, args.smear, 0.3)
    lo, hi = dist.slab_rows(dims, world, rank)
    hU, hP = torch.from_numpy(U[lo:hi].copy()).pin_memory(), torch.from_numpy(P[lo:hi].copy()).pin_memory()
    ctx = dd.ranks[0]
    lgt.lgt_set_links_host(ctx, hU)
    d_eta = torch.from_numpy(eta[lo:hi].copy()).cuda()
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
    for _ in range(args.warmup):
        md_step()
    sampler = ClockSampler(local)
    launches0 = lgt.lgt_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler.start()
    barrier()
    e0.record()
    iters = [md_step() for _ in range(args.steps)]
    e1.record()
    barrier()
    clocks = sampler.stop()
    elapsed_ms = e0.elapsed_time(e1)
    launches = lgt.lgt_launch_count(ctx) - launches0
    k_e2e = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    e2e_iters = []
    for _ in range(k_e2e):
        reset_state()
        e2e_iters.append(md_step())
        lgt.lgt_get_links_host(ctx, hU_out)
        lgt.lgt_get_momenta_host(ctx, hP_out)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    (elapsed_ms, e2e_s), (launches_all,) = dist.aggregate([elapsed_ms, e2e_s], [launches], device="cuda")
    if rank == 0:
        total_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in iters) * V  # the whole lattice: strong scaling
        e2e_reals = sum(step_reals(i, args.solver, args.action, args.smear) for i in e2e_iters) * V
        out = {
            "metric": METRIC, "value": round(total_reals * 8 / (elapsed_ms * 1e-3) / 1e9, 1), "unit": "GB/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(elapsed_ms / args.steps, 3),
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[%d]: ONE %s SU(3) lattice in %d time slabs, one MD step = kick(dt) + drift(dt), "
                                   "CG 1e-12" % (args.config, "x".join(map(str, dims)), world),
                       "beta": beta, "kappa": kappa, "bc": list(bc), "dt": dt, "cg_tol": tol, "cg_iters_per_step": iters,
                       "parallelism": "dd%d (time slabs, halo %s, NCCL all-reduce)" % (world, args.halo),
                       "solver": args.solver, "fermion_action": args.action, "stout_levels": args.smear,
                       "l2": "inputs exceed L2 at 32^4 up to 8 slabs (links 604 MB / N per rank)"},
            "clocks": clocks,
            "e2e": {"value": round(e2e_reals * 8 / e2e_s / 1e9, 1), "unit": "GB/s", "steps": k_e2e,
                    "ms_per_step": round(e2e_s / k_e2e * 1e3, 2),
                    "h2d_bytes_per_step": (hU.numel() + hP.numel() + hphi.numel()) * 16 * world,
                    "d2h_bytes_per_step": (hU_out.numel() + hP_out.numel()) * 16 * world},
            "gpu_launches": int(launches_all),
        }
        print(json.dumps(out), flush=True)
    dd.close()
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
        "config": {"workload": "configs[%d]: %s SU(3) MD step on the CPU oracle, bounded sample" %
                               (args.config, "x".join(map(str, cfg["dims"])))},
        "cpu_baseline": base,
        "e2e": {"value": base["value"], "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "wall_s": round(time.perf_counter() - t0, 1),
    }
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
    ap.add_argument("--halo", default="exchange", choices=["exchange", "push"],
                    help="--parallelism dd: NCCL send/recv of the halo slices, or halos stored into the neighbours' ghost "
                         "slices by the Dslash kernels (CUDA IPC between processes)")
    ap.add_argument("--smear", type=int, default=0,
                    help="non-default: the fermions see this many levels of stout-smeared links (rho = 0.3); not the headline")
    ap.add_argument("--skip-extras", action="store_true", help="profiling runs only: leave the non-headline solver arms out")
    ap.add_argument("--parallelism", default="replicas", choices=["replicas", "dd"],
                    help="N > 1: 'replicas' = N independent lattices (default, weak scaling); 'dd' = ONE lattice cut into N "
                         "time slabs with NCCL halo exchange (lgt_dd_*, strong scaling; verified on one GPU only, DESIGN.md)")
    ap.add_argument("--cpu-sample-iters", type=int, default=20, help="CG iterations in the oracle's bounded sample")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        run_reference(args)
    elif args.parallelism == "dd":
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
