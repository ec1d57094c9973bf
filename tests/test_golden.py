"""tests/golden/config0_oracle.json: written by the oracle (make_golden.py); reproduced by the oracle on CPU,
matched by the CUDA path on GPU."""
import json
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
GOLD = json.load(open(os.path.join(HERE, "golden", "config0_oracle.json")))


def _mat(rows):
    return np.array([complex(a, b) for a, b in rows]).reshape(3, 3)


def test_oracle_reproduces_golden():
    import sys

    sys.path.insert(0, os.path.join(HERE, "golden"))
    import make_golden

    now = make_golden.compute()
    assert now["cg_iters"] == GOLD["cg_iters"] and GOLD["cg_converged"]
    for k in ("S_g", "plaquette", "S_F", "fermion_force_norm2", "gauge_force_norm2"):
        assert abs(now[k] - GOLD[k]) <= 1e-12 * abs(GOLD[k]), k
    # closed form (pin P6) holds for the stored numbers
    assert abs(GOLD["S_F"] - GOLD["eta_norm2"]) < 1e-12 * GOLD["eta_norm2"]


@pytest.mark.gpu
def test_cuda_path_matches_golden():
    import oracle
    from paper_2602_20516_b200 import lgt, synth

    c = synth.CONFIGS[0]
    dims, beta, kappa, bc, tol = c["dims"], c["beta"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(0)
    phi = oracle.dslash(dims, kappa, bc, U, synth.gaussian_spinor(dims, c["seed_eta"]), dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    S_g, S_F, K, it = lgt.lgt_action(lat.ctx, tol, 10 * V)
    assert it == GOLD["cg_iters"]
    assert abs(S_g - GOLD["S_g"]) < 1e-12 * abs(GOLD["S_g"])
    assert abs(S_F - GOLD["S_F"]) < 1e-11 * abs(GOLD["S_F"])
    assert abs(lgt.lgt_plaquette(lat.ctx) - GOLD["plaquette"]) < 1e-14
    Ff, _ = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    Fg = lat.gauge_force()
    for (s, mu), rf, rg in zip(GOLD["links"], GOLD["fermion_force"], GOLD["gauge_force"]):
        assert np.linalg.norm(Ff[s, mu] - _mat(rf)) < 1e-11 * np.linalg.norm(_mat(rf))
        assert np.linalg.norm(Fg[s, mu] - _mat(rg)) < 1e-12 * np.linalg.norm(_mat(rg))
    lat.close()
