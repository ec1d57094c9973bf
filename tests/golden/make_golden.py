"""Writes tests/golden/config0_oracle.json from the CPU oracle only (never from the CUDA path).

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


if __name__ == "__main__":
    with open(os.path.join(HERE, "config0_oracle.json"), "w") as f:
        json.dump(compute(), f, indent=1)
    print("written")
