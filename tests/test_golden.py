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


EXT = json.load(open(os.path.join(HERE, "golden", "config0_extensions.json")))


def test_oracle_reproduces_extension_golden():
    import sys

    sys.path.insert(0, os.path.join(HERE, "golden"))
    import make_golden

    now = make_golden.compute_extensions()
    for sec, keys in (("even_odd", ("S_F", "force_norm2")), ("heatbath", ("K", "eta_norm2", "metropolis_u")),
                      ("stout", ("smeared_plaquette", "force_norm2"))):
        for k in keys:
            assert abs(now[sec][k] - EXT[sec][k]) <= 1e-12 * abs(EXT[sec][k]), (sec, k)
    assert now["even_odd"]["cg_iters"] == EXT["even_odd"]["cg_iters"] and now["stout"]["cg_iters"] == EXT["stout"]["cg_iters"]


@pytest.mark.gpu
def test_cuda_path_matches_extension_golden():
    import oracle
    from oracle import evenodd as oeo
    from oracle import stout as ost
    from paper_2602_20516_b200 import lgt, synth

    c = synth.CONFIGS[0]
    dims, beta, kappa, bc, tol = c["dims"], c["beta"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(0)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    # heat baths
    hb = EXT["heatbath"]
    lgt.lgt_momentum_heatbath(lat.ctx, hb["seed"], hb["trajectory"])
    P = lat.get_momenta()
    for (s, mu), ref in zip(EXT["links"], hb["momenta"]):
        assert np.abs(P[s, mu] - _mat(ref)).max() < 1e-14
    assert abs(lgt.lgt_action(lat.ctx)[2] - hb["K"]) < 1e-12 * hb["K"]
    assert abs(lgt.lgt_pseudofermion_heatbath(lat.ctx, hb["seed"], hb["trajectory"]) - hb["eta_norm2"]) < 1e-12 * hb["eta_norm2"]
    # even/odd action
    eo = EXT["even_odd"]
    lat.set_pseudofermion(oeo.mhat(dims, kappa, bc, U, oeo.keep(eta, dims, 0), dagger=True))
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    F, it = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it == eo["cg_iters"]
    for (s, mu), ref in zip(EXT["links"], eo["force"]):
        assert np.linalg.norm(F[s, mu] - _mat(ref)) < 1e-11 * np.linalg.norm(_mat(ref))
    assert abs(lgt.lgt_action(lat.ctx, tol, 10 * V)[1] - eo["S_F"]) < 1e-11 * eo["S_F"]
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_FULL)
    # one stout level
    st = EXT["stout"]
    lgt.lgt_set_smearing(lat.ctx, st["levels"], st["rho"])
    U1 = lat.empty(V, 4, 3, 3)
    lgt.lgt_get_smeared_links(lat.ctx, U1)
    U1 = U1.cpu().numpy()
    for (s, mu), ref in zip(EXT["links"], st["smeared_links"]):
        assert np.abs(U1[s, mu] - _mat(ref)).max() < 1e-13
    lat.set_pseudofermion(oracle.dslash(dims, kappa, bc, ost.smear(dims, st["rho"], U)[0], eta, dagger=True))
    F, it = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it == st["cg_iters"]
    for (s, mu), ref in zip(EXT["links"], st["force"]):
        assert np.linalg.norm(F[s, mu] - _mat(ref)) < 1e-11 * np.linalg.norm(_mat(ref))
    lat.close()
