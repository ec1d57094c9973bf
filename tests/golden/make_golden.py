"""Writes tests/golden/config0_oracle.json and config0_extensions.json from the CPU oracle only (never from the CUDA path).

    python tests/golden/make_golden.py
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_2602_20516_b200 import synth  # noqa: E402


def compute():
    c = synth.CONFIGS[0]
    dims, beta, kappa, bc, tol = c["dims"], c["beta"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(0)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    S_g, plaq = oracle.gauge_action(dims, beta, U)
    S_F, X, iters, ok = oracle.fermion_action(dims, kappa, bc, U, phi, tol, 10 * V)
    Y = oracle.dslash(dims, kappa, bc, U, X)
    Ff = oracle.fermion_force(dims, kappa, bc, U, X, Y)
    Fg = oracle.gauge_force(dims, beta, U)
    links = [(0, 0), (3, 1), (100, 2), (V - 1, 3)]

    def mat(m):
        return [[float(z.real), float(z.imag)] for z in m.ravel()]

    return {
        "config": "BASELINE.json configs[0]", "written_by": "tests/golden/make_golden.py (oracle only)",
        "S_g": S_g, "plaquette": plaq, "S_F": S_F, "eta_norm2": float(np.sum(np.abs(eta) ** 2)),
        "cg_iters": iters, "cg_converged": bool(ok),
        "fermion_force_norm2": float(np.sum(np.abs(Ff) ** 2)), "gauge_force_norm2": float(np.sum(np.abs(Fg) ** 2)),
        "links": [list(l) for l in links],
        "fermion_force": [mat(Ff[s, mu]) for s, mu in links],
        "gauge_force": [mat(Fg[s, mu]) for s, mu in links],
    }


def compute_extensions():
    """Regression values of the SURVEY 8(f) oracles on configs[0]: even/odd action, Philox heat baths, one stout level."""
    from oracle import evenodd as oeo
    from oracle import hmc as ohmc
    from oracle import stout as ost

    c = synth.CONFIGS[0]
    dims, kappa, bc, tol = c["dims"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(0)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    links = [(0, 0), (3, 1), (100, 2), (V - 1, 3)]

    def mat(m):
        return [[float(z.real), float(z.imag)] for z in m.ravel()]

    phi_eo = oeo.mhat(dims, kappa, bc, U, oeo.keep(eta, dims, 0), dagger=True)
    S_eo, _, it_eo, ok_eo = oeo.action(dims, kappa, bc, U, phi_eo, tol, 10 * V)
    F_eo, _, _ = oeo.fermion_force(dims, kappa, bc, U, phi_eo, tol, 10 * V)
    seed, traj = 20260220516, 3
    P, _ = ohmc.momentum_heatbath(dims, seed, traj)
    noise = ohmc.pseudofermion_noise(dims, seed, traj)
    rho = 0.3
    U1 = ost.smear(dims, rho, U)[0]
    phi_st = oracle.dslash(dims, kappa, bc, U1, eta, dagger=True)
    F_st, it_st, ok_st = ost.fermion_force(dims, kappa, bc, U, phi_st, 1, rho, tol, 10 * V)
    return {
        "config": "BASELINE.json configs[0]", "written_by": "tests/golden/make_golden.py (oracle only)", "links": [list(l) for l in links],
        "even_odd": {"S_F": S_eo, "cg_iters": it_eo, "cg_converged": bool(ok_eo), "force_norm2": float(np.sum(np.abs(F_eo) ** 2)),
                     "force": [mat(F_eo[s, mu]) for s, mu in links]},
        "heatbath": {"seed": seed, "trajectory": traj, "K": oracle.kinetic(dims, P), "eta_norm2": float(np.sum(np.abs(noise) ** 2)),
                     "momenta": [mat(P[s, mu]) for s, mu in links], "eta_site0": [[float(z.real), float(z.imag)] for z in noise[0].ravel()],
                     "metropolis_u": ohmc.metropolis_uniform(seed, traj)},
        "stout": {"rho": rho, "levels": 1, "smeared_plaquette": oracle.gauge_action(dims, 1.0, U1)[1], "cg_iters": it_st,
                  "cg_converged": bool(ok_st), "force_norm2": float(np.sum(np.abs(F_st) ** 2)),
                  "smeared_links": [mat(U1[s, mu]) for s, mu in links], "force": [mat(F_st[s, mu]) for s, mu in links]},
    }


if __name__ == "__main__":
    with open(os.path.join(HERE, "config0_oracle.json"), "w") as f:
        json.dump(compute(), f, indent=1)
    with open(os.path.join(HERE, "config0_extensions.json"), "w") as f:
        json.dump(compute_extensions(), f, indent=1)
    print("written")
