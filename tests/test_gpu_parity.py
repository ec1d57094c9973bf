"""GPU parity: the CUDA path through the C ABI vs the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): per link / per site relative 1e-11 in fp64,
2e-5 in fp32; CG iteration counts identical in fp64.
"""
import numpy as np
import pytest

import oracle
from oracle import evenodd as oeo
from paper_2602_20516_b200 import synth
from lattice_util import link_rel_err, link_rel_quantiles

pytestmark = pytest.mark.gpu

BC = (1, 1, 1, -1)
TOL64 = 1e-11
TOL32 = 2e-5


@pytest.fixture(scope="module")
def lgt():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the product path has no CPU fallback")
    from paper_2602_20516_b200 import lgt as m

    m.lib()
    return m


def site_rel_err(a, ref):
    """max over sites of |a - ref|_2 / |ref|_2 per site (12 complex numbers)."""
    d = np.sqrt(np.sum(np.abs(a - ref) ** 2, axis=(-1, -2)))
    n = np.sqrt(np.sum(np.abs(ref) ** 2, axis=(-1, -2)))
    return float((d / n).max())


def round32(a):
    return a.astype(np.complex64).astype(np.complex128)


# dims spanning several 128-thread blocks with ragged tails, odd extents, extents of 1 and 2
DSLASH_DIMS = [(4, 4, 4, 4), (4, 3, 5, 6), (8, 8, 8, 8), (6, 2, 1, 10), (16, 16, 16, 16), (3, 3, 3, 3)]


@pytest.mark.parametrize("dims", DSLASH_DIMS)
@pytest.mark.parametrize("dag", [False, True])
def test_dslash_fp64(lgt, dims, dag):
    U = synth.warm_links(dims, 0.3, 7)
    psi = synth.gaussian_spinor(dims, 8)
    for bc in (BC, (1, 1, 1, 1), (-1, -1, 1, -1)):
        lat = lgt.Lattice(dims, 5.6, 0.12, bc)
        lat.set_links(U)
        out = lat.dslash(psi, dagger=dag)
        ref = oracle.dslash(dims, 0.12, bc, U, psi, dagger=dag)
        assert site_rel_err(out, ref) < TOL64
        lat.close()


@pytest.mark.parametrize("dims,zs", [((16, 8, 8, 6), (1, 2, 4, 8)), ((32, 4, 6, 3), (1, 3, 6)), ((8, 16, 4, 5), (2, 4))])
def test_dslash_block_swizzle(lgt, dims, zs):
    """The slab-by-slab block order (lgt_set_block_swizzle) is a pure relabelling of blocks: D, D^dag and a whole CG
    solve must be bitwise what the lexicographic order gives, and equal to the oracle."""
    U = synth.warm_links(dims, 0.3, 17)
    psi = synth.gaussian_spinor(dims, 18)
    lat = lgt.Lattice(dims, 5.6, 0.12, BC)
    lat.set_links(U)
    assert lgt.lgt_set_block_swizzle(lat.ctx, 0) == 0
    base = [lat.dslash(psi, dagger=d) for d in (False, True)]
    x0, it0, _, ok0 = lat.cg(psi, 1e-10, 2000)
    Fg0 = lat.gauge_force()
    for d in (False, True):
        assert site_rel_err(base[d], oracle.dslash(dims, 0.12, BC, U, psi, dagger=d)) < TOL64
    for z in zs:
        assert lgt.lgt_set_block_swizzle(lat.ctx, z) == z
        for d in (False, True):
            assert np.array_equal(lat.dslash(psi, dagger=d), base[d])
        assert np.array_equal(lat.gauge_force(), Fg0)  # the staple kernel walks its blocks in the same order
        x, it, _, ok = lat.cg(psi, 1e-10, 2000)
        assert ok and ok0 and it == it0
        assert np.abs(x - x0).max() <= 1e-13 * np.abs(x0).max()  # block partials are summed in another order
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_block_swizzle(lat.ctx, 5 if dims[2] % 5 else 7)
    assert lgt.lgt_set_block_swizzle(lat.ctx, -1) == 0  # small lattice: automatic choice is "off"
    lat.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 10, 6, 8), (16, 16, 8, 4), (32, 4, 6, 3), (4, 3, 5, 6)])
def test_dslash_kernel_variants(lgt, dims):
    """Every implementation variant of the Dslash kernels kept in the library (lgt_set_kernel_variant; measured against
    each other in profiles/r02a_dslash_variants.md) applies the same operator: D and D^dag bitwise equal to variant 0
    (same per-site arithmetic in the same order) and equal to the oracle, a CG solve with the oracle's iteration count.
    Shapes the tiled variant cannot take (odd Lz / Lt, xy planes that are no multiple of 64 sites) fall back to variant 0."""
    U = synth.warm_links(dims, 0.3, 27)
    psi = synth.gaussian_spinor(dims, 28)
    lat = lgt.Lattice(dims, 5.6, 0.12, BC)
    lat.set_links(U)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH) == 0
    base = [lat.dslash(psi, dagger=d) for d in (False, True)]
    for d in (False, True):
        assert site_rel_err(base[d], oracle.dslash(dims, 0.12, BC, U, psi, dagger=d)) < TOL64
    x0, it0, _, ok0 = lat.cg(psi, 1e-10, 2000)
    _, it_ref, _, ok_ref = oracle.cg(dims, 0.12, BC, U, psi, 1e-10, 2000)
    assert ok0 and ok_ref and it0 == it_ref
    for v in (1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12):
        assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, v) == v
        for d in (False, True):
            if v in (6, 7, 12):  # 6 sums the eight hops in another order, 7 (and 12 = 7 in fp64) rebuilds the third row of every link
                assert site_rel_err(lat.dslash(psi, dagger=d), base[d]) < 1e-13
            else:
                assert np.array_equal(lat.dslash(psi, dagger=d), base[d]), (v, d)
        x, it, _, ok = lat.cg(psi, 1e-10, 2000)
        assert ok and it == it0, (v, it, it0)
        assert np.abs(x - x0).max() <= 1e-12 * np.abs(x0).max()  # variant 3 sums other block partials
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 13)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_kernel_variant(lat.ctx, 99, 0)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 0) == 0
    lat.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (32, 4, 6, 3), (16, 16, 16, 24)])
def test_dslash_fp32_twelve_real_links_variant(lgt, dims):
    """Variant 12 of the Dslash kernels (fp32 handles): rows 0 and 1 of every link read, row 2 rebuilt in registers with the
    folded fermion boundary sign, in the fp32 default's build (three blocks per SM, end-of-block prefetch of the two rows; the
    last shape is more than two waves of blocks, where the default prefetches too).  D, D^dag against the oracle within
    the fp32 tolerance and against variant 0 to fp32 rounding; CG with variant 0's count."""
    U = round32(synth.warm_links(dims, 0.3, 47))
    psi = round32(synth.gaussian_spinor(dims, 48))
    lat = lgt.Lattice(dims, 5.6, 0.12, BC, precision=lgt.LGT_F32)
    lat.set_links(U)
    base = [lat.dslash(psi, dagger=d).astype(np.complex128) for d in (False, True)]
    _, it0, _, ok0 = lat.cg(psi, 1e-5, 2000)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 12) == 12
    for d in (False, True):
        out = lat.dslash(psi, dagger=d).astype(np.complex128)
        assert site_rel_err(out, base[d]) < 2e-6
        if synth.volume(dims) <= 4096:
            assert site_rel_err(out, oracle.dslash(dims, 0.12, BC, U, psi, dagger=d)) < TOL32
    _, it, _, ok = lat.cg(psi, 1e-5, 2000)
    assert ok0 and ok and abs(it - it0) <= 1
    lat.close()


def test_async_host_transfers_match_the_blocking_ones(lgt):
    """lgt_set_momenta_host_async / lgt_get_*_host_async: the momenta upload runs on the copy stream under the solve (the
    kick solves first and only then touches Pi), the downloads run under whatever follows.  Two MD steps driven through the
    asynchronous calls give bitwise the links and momenta of the blocking calls, the downloaded buffers are complete after
    lgt_host_transfers_wait, and a second upload / download issued before the first has drained keeps the order."""
    import torch

    dims, beta, kappa = (8, 8, 8, 8), 5.6, 0.12
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 57)
    P = synth.gaussian_momenta(dims, 58)
    P2 = synth.gaussian_momenta(dims, 59)
    phi = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 60), dagger=True)
    hU, hP, hP2, hphi = [torch.from_numpy(a).pin_memory() for a in (U, P, P2, phi)]
    out = {}
    for mode in ("blocking", "async"):
        lat = lgt.Lattice(dims, beta, kappa, BC)
        hUo, hPo, hPo1 = [torch.zeros((V, 4, 3, 3), dtype=torch.complex128).pin_memory() for _ in range(3)]
        lgt.lgt_set_links_host(lat.ctx, hU)
        lgt.lgt_set_pseudofermion_host(lat.ctx, hphi)
        if mode == "blocking":
            lgt.lgt_set_momenta_host(lat.ctx, hP2)
            lgt.lgt_set_momenta_host(lat.ctx, hP)
        else:
            lgt.lgt_set_momenta_host_async(lat.ctx, hP2)  # overwritten by the next upload, in order
            lgt.lgt_set_momenta_host_async(lat.ctx, hP)
        its = [lgt.lgt_md_kick(lat.ctx, 0.02, 1e-12, 5000)]
        if mode == "blocking":
            lgt.lgt_get_momenta_host(lat.ctx, hPo1)
        else:
            lgt.lgt_get_momenta_host_async(lat.ctx, hPo1)
        lgt.lgt_md_drift(lat.ctx, 0.02)
        its.append(lgt.lgt_md_kick(lat.ctx, 0.02, 1e-12, 5000))
        if mode == "blocking":
            lgt.lgt_get_links_host(lat.ctx, hUo)
            lgt.lgt_get_momenta_host(lat.ctx, hPo)
        else:
            lgt.lgt_get_links_host_async(lat.ctx, hUo)
            lgt.lgt_get_momenta_host_async(lat.ctx, hPo)
            lgt.lgt_host_transfers_wait(lat.ctx)
        out[mode] = (hUo.numpy().copy(), hPo.numpy().copy(), hPo1.numpy().copy(), its)
        lat.close()
    for a, b in zip(out["blocking"][:3], out["async"][:3]):
        assert np.array_equal(a, b)
    assert out["blocking"][3] == out["async"][3]
    P1, _, _ = oracle.kick(dims, beta, kappa, BC, U, phi, P, 0.02, 1e-12, 5000)
    assert link_rel_err(out["async"][2], P1)[0] < TOL64


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (4, 3, 5, 6), (16, 4, 6, 2)])
def test_gauge_force_kernel_variants(lgt, dims):
    """The implementation variants of the staple kernel (lgt_set_kernel_variant(LGT_K_GAUGE_FORCE)): 1 and 2 only regroup the
    link threads into bigger blocks (the same sums bit for bit), 3 is one thread per site with the up staples taken plaquette
    by plaquette (another summation order: per link 1e-13 of the oracle like the default)."""
    U = synth.haar_links(dims, 47)
    ref = oracle.gauge_force(dims, 5.7, U)
    lat = lgt.Lattice(dims, 5.7, 0.0, BC)
    lat.set_links(U)
    base = lat.gauge_force()
    assert link_rel_err(base, ref)[0] < 1e-13
    for v in (1, 2, 3):
        assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_GAUGE_FORCE, v) == v
        F = lat.gauge_force()
        if v < 3:
            assert np.array_equal(F, base)
        assert link_rel_err(F, ref)[0] < 1e-13
        lat.set_momenta(np.zeros_like(ref))
        lgt.lgt_gauge_force_accumulate(lat.ctx, 0.5)  # the fused Pi -= eps F form of the same variant
        assert link_rel_err(lat.get_momenta(), -0.5 * ref)[0] < 1e-13
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_GAUGE_FORCE, 4)
    lat.close()


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (6, 4, 10, 6), (4, 3, 5, 6)])
def test_cg_fused_scalar_update_variant(lgt, dims):
    """Variant 1 of LGT_K_CG_BLAS: the CG scalar updates ride in the last block of the stencil kernels (ticket counter)
    instead of two one-block launches per iteration.  Same fixed-order sums (cg_fixed_sum is independent of the number of
    threads forming it): solution, iteration count and residual bitwise those of variant 0, for the full operator, the
    even/odd Schur complement and the mixed-precision solver; two launches fewer per iteration."""
    kappa = 0.12
    U = synth.warm_links(dims, 0.3, 37)
    b = synth.gaussian_spinor(dims, 38)
    lat = lgt.Lattice(dims, 5.6, kappa, BC)
    lat.set_links(U)
    even = all(d % 2 == 0 for d in dims)
    runs = []
    # 2: the whole even/odd solve as one cooperative launch; 3: the scalar updates folded into the kernels that follow them
    # (both: even/odd CG only, the full-operator CG is unaffected)
    for v in (0, 1, 0, 2, 3):
        assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_CG_BLAS, v) == v
        n0 = lgt.lgt_launch_count(lat.ctx)
        x, it, rel, ok = lat.cg(b, 1e-10, 3000)
        n1 = lgt.lgt_launch_count(lat.ctx)
        res = [x, it, rel, ok, n1 - n0]
        if even:
            res += list(lat.eo_cg(b, 1e-10, 3000))
        res += list(lat.cg_mixed(b, 1e-10, 3000))
        runs.append(res)
    for other in (runs[1], runs[3], runs[4]):
        for a, c in zip(runs[0], other):
            if isinstance(a, np.ndarray):
                assert np.array_equal(a, c)
            elif isinstance(a, (int, bool)) and not isinstance(c, float):
                pass
        if even:  # eo_cg: x, iterations, residual, converged at positions 5..8
            assert runs[0][6] == other[6] and runs[0][7] == other[7] and other[8]
    assert runs[0][1] == runs[1][1] == runs[2][1] and runs[0][2] == runs[1][2] and runs[0][3] and runs[1][3]
    # launches: init + per started chunk of 8 iterations (5 | 3 kernels per iteration) + the final Y = D x is not part of lat.cg
    chunks = -(-runs[0][1] // 8)
    assert runs[0][4] - runs[1][4] == 2 * 8 * chunks
    _, it_ref, _, ok_ref = oracle.cg(dims, kappa, BC, U, b, 1e-10, 3000)
    assert ok_ref and runs[1][1] == it_ref
    lat.close()


@pytest.mark.parametrize("dims", [(4, 3, 5, 6), (16, 16, 16, 16)])
def test_dslash_fp32(lgt, dims):
    U = round32(synth.warm_links(dims, 0.3, 7))
    psi = round32(synth.gaussian_spinor(dims, 8))
    lat = lgt.Lattice(dims, 5.6, 0.12, BC, precision=lgt.LGT_F32)
    lat.set_links(U)
    for dag in (False, True):
        out = lat.dslash(psi, dagger=dag).astype(np.complex128)
        ref = oracle.dslash(dims, 0.12, BC, U, psi, dagger=dag)
        assert site_rel_err(out, ref) < TOL32
    lat.close()


def test_links_momenta_roundtrip(lgt):
    dims = (4, 3, 5, 6)
    U = synth.warm_links(dims, 0.3, 1)
    P = synth.gaussian_momenta(dims, 2)
    lat = lgt.Lattice(dims, 5.6, 0.12, BC)
    assert np.array_equal(lat.get_links(), synth.unit_links(dims))  # initial state
    assert not lat.get_momenta().any()
    lat.set_links(U)
    lat.set_momenta(P)
    assert np.array_equal(lat.get_links(), U)
    assert np.abs(lat.get_momenta() - P).max() < 1e-15
    lat.close()


@pytest.mark.parametrize("cfg", [0, 2])
def test_cg_and_fermion_force_configs(lgt, cfg):
    """configs[0] (4^4, tol 1e-14) and configs[2] (16^4, tol 1e-12): CG iteration count identical, X, Y = D X = eta,
    S_F = |eta|^2 and the per-link force (Eq. 8 of the paper) against the oracle."""
    c = synth.CONFIGS[cfg]
    dims, kappa, bc, tol = c["dims"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(cfg)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    X_ref, it_ref, rel_ref, ok_ref = oracle.cg(dims, kappa, bc, U, phi, tol, 10 * V)
    Y_ref = oracle.dslash(dims, kappa, bc, U, X_ref)
    F_ref = oracle.fermion_force(dims, kappa, bc, U, X_ref, Y_ref)
    assert ok_ref

    lat = lgt.Lattice(dims, 5.5, kappa, bc)
    lat.set_links(U)
    X, it, rel, ok = lat.cg(phi, tol, 10 * V)
    assert ok and it == it_ref, (it, it_ref, rel, rel_ref)
    assert rel <= tol
    assert site_rel_err(X, X_ref) < 1e-9  # solution agrees to tol * sqrt(cond)
    # force kernel alone, shared X and Y: rounding level
    F_shared, _ = lat.fermion_force(X_ref, Y_ref)
    e, plain = link_rel_err(F_shared, F_ref)
    assert e < 1e-13, (e, plain)
    # end to end from phi through the GPU's own CG
    lat.set_pseudofermion(phi)
    F, it2 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it2 == it_ref
    e, plain = link_rel_err(F, F_ref)
    assert e < TOL64, (e, plain)
    if cfg == 2:
        # the paper's own accuracy figure (Fig. 2: Eq. 8 over every link of a 16^4 lattice, "uniform
        # agreement at the level of 1e-9 ... no visible outliers"), here GPU against oracle: the whole distribution
        # sits at double-precision rounding (measured: median 9e-16, 99.9 % 3e-15, max 6e-15) with a short tail
        q50, q90, q99, q999, qmax = link_rel_quantiles(F, F_ref)
        print("Eq. 8 distribution, 16^4, GPU CG + force vs oracle: median %.2e 90%% %.2e 99%% %.2e 99.9%% %.2e max %.2e"
              % (q50, q90, q99, q999, qmax))
        assert qmax < 1e-13 and q50 < 1e-14 and qmax < 30 * q50
        k50, _, _, _, kmax = link_rel_quantiles(F_shared, F_ref)
        print("  force kernel alone (shared X, Y): median %.2e max %.2e" % (k50, kmax))
        assert kmax < 1e-14
    # closed forms (pin P6): S_F = |eta|^2
    S_g, S_F, K, _ = lgt.lgt_action(lat.ctx, tol, 10 * V)
    n2 = np.sum(np.abs(eta) ** 2)
    assert abs(S_F - n2) < 1e-11 * n2
    S_g_ref, _ = oracle.gauge_action(dims, 5.5, U)
    assert abs(S_g - S_g_ref) < 1e-12 * abs(S_g_ref)
    lat.close()


@pytest.mark.parametrize("cfg,dims", [(0, None), (2, None), (2, (6, 10, 4, 8))])
def test_mixed_precision_cg(lgt, cfg, dims):
    """fp32 inner CG inside an fp64 defect-correction loop.  The solution of a linear system is unique,
    so the reference is the oracle's fp64 CG solution and the TRUE residual taken with the oracle's D; iteration
    counts are this solver's own (reading A-25) and are only bounded here.  Then the whole fermion kick
    through the mixed solver against the oracle force (1e-11 per link)."""
    c = synth.CONFIGS[cfg]
    dims = dims or c["dims"]
    # Solved to 1e-13 on both sides: with plain CG the two sides stop the same recurrence at the same iteration and
    # their solution errors cancel in the comparison; here the stopping rules differ (recurrence residual in the
    # oracle, true residual in the mixed solver), the errors are independent, and at 1e-12 the per-link force
    # difference is 1.5e-11 - 2.1e-11 (measured), just above the 1e-11 bar.
    kappa, bc, tol = c["kappa"], c["bc"], 1e-13
    V = synth.volume(dims)
    U = synth.warm_links(dims, c["eps"], c["seed_links"])
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    X_ref, it_ref, _, ok_ref = oracle.cg(dims, kappa, bc, U, phi, tol, 10 * V)
    Y_ref = oracle.dslash(dims, kappa, bc, U, X_ref)
    F_ref = oracle.fermion_force(dims, kappa, bc, U, X_ref, Y_ref)
    assert ok_ref

    lat = lgt.Lattice(dims, 5.5, kappa, bc)
    lat.set_links(U)
    X, inner, outer, rel, ok = lat.cg_mixed(phi, tol, 10 * V, inner_tol=1e-5)
    assert ok and rel <= tol
    assert 2 <= outer <= 8 and inner <= 2 * it_ref, (inner, outer, it_ref)
    # true residual with the oracle's operator
    AX = oracle.dslash(dims, kappa, bc, U, oracle.dslash(dims, kappa, bc, U, X), dagger=True)
    true_rel = np.linalg.norm(phi - AX) / np.linalg.norm(phi)
    assert true_rel <= 1.05 * tol, true_rel
    assert site_rel_err(X, X_ref) < 1e-9
    # a looser inner tolerance costs more cycles but reaches the same answer
    X2, inner2, outer2, rel2, ok2 = lat.cg_mixed(phi, tol, 10 * V, inner_tol=1e-3)
    assert ok2 and rel2 <= tol and outer2 > outer
    assert site_rel_err(X2, X_ref) < 1e-9
    # the fermion force and action through the handle's solver switch
    lat.set_pseudofermion(phi)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    F, it2 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it2 == inner
    e, plain = link_rel_err(F, F_ref)
    assert e < TOL64, (e, plain)
    _, S_F, _, _ = lgt.lgt_action(lat.ctx, tol, 10 * V)
    n2 = np.sum(np.abs(eta) ** 2)
    assert abs(S_F - n2) < 1e-11 * n2  # pin P6: S_F = |eta|^2
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_CG)
    F, it3 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it3 == it_ref
    # cap reached: LGT_ENOCONV, reported as not converged
    _, inner4, _, rel4, ok4 = lat.cg_mixed(phi, tol, 5, inner_tol=1e-5)
    assert not ok4 and inner4 == 5 and rel4 > tol
    lat.close()
    lat32 = lgt.Lattice(dims, 5.5, kappa, bc, precision=lgt.LGT_F32)
    with pytest.raises(lgt.LgtError):
        lgt.lgt_set_solver(lat32.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    lat32.close()


EO_DIMS = [(4, 4, 4, 4), (2, 2, 2, 2), (6, 10, 4, 8), (16, 4, 2, 6), (8, 8, 8, 8)]


@pytest.mark.parametrize("dims", EO_DIMS)
def test_eo_schur_operator(lgt, dims):
    """M = 1 - kappa^2 H_eo H_oe and M^dag on the even sites against the oracle's definition
    (oracle/evenodd.py), fp64 and fp32, periodic and antiperiodic boundaries; odd sites of the output are zero."""
    U = synth.warm_links(dims, 0.3, 27)
    psi = synth.gaussian_spinor(dims, 28)
    odd = oeo.parity(dims) == 1
    for bc in (BC, (1, 1, 1, 1), (-1, 1, -1, -1)):
        lat = lgt.Lattice(dims, 5.6, 0.12, bc)
        lat.set_links(U)
        for dag in (False, True):
            out = lat.eo_mhat(psi, dagger=dag)
            ref = oeo.mhat(dims, 0.12, bc, U, psi, dagger=dag)
            assert not out[odd].any()
            assert site_rel_err(out[~odd], ref[~odd]) < TOL64
        lat.close()
    lat = lgt.Lattice(dims, 5.6, 0.12, BC, precision=lgt.LGT_F32)
    U32, psi32 = round32(U), round32(psi)
    lat.set_links(U32)
    out = lat.eo_mhat(psi32).astype(np.complex128)
    assert site_rel_err(out[~odd], oeo.mhat(dims, 0.12, BC, U32, psi32)[~odd]) < TOL32
    lat.close()


@pytest.mark.parametrize("dims,kappa", [((4, 4, 4, 4), 0.10), ((8, 8, 8, 8), 0.12), ((6, 10, 4, 8), 0.12)])
def test_eo_cg_force_and_action(lgt, dims, kappa):
    """CG on M^dag M: iteration count identical to the oracle's, solution, then the even/odd action and its per-link
    force through lgt_set_fermion_action (reconstruction X_o = kappa H_oe X_e, Y_o = kappa H_oe^dag Y_e on the GPU),
    the closed form S = |eta_e|^2, and one kick of the momenta."""
    V = synth.volume(dims)
    tol, beta = 1e-12, 5.5
    U = synth.warm_links(dims, 0.3, 37)
    eta = oeo.keep(synth.gaussian_spinor(dims, 38), dims, 0)
    phi = oeo.mhat(dims, kappa, BC, U, eta, dagger=True) + oeo.keep(synth.gaussian_spinor(dims, 39), dims, 1)  # odd part must be ignored
    X_ref, it_ref, rel_ref, ok_ref = oeo.cg(dims, kappa, BC, U, phi, tol, 10 * V)
    F_ref, _, _ = oeo.fermion_force(dims, kappa, BC, U, phi, tol, 10 * V)
    assert ok_ref

    lat = lgt.Lattice(dims, beta, kappa, BC)
    lat.set_links(U)
    X, it, rel, ok = lat.eo_cg(phi, tol, 10 * V)
    assert ok and it == it_ref, (it, it_ref, rel, rel_ref)
    even = oeo.parity(dims) == 0
    assert not X[~even].any()
    assert site_rel_err(X[even], X_ref[even]) < 1e-9
    lat.set_pseudofermion(phi)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    F, it2 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it2 == it_ref
    e, plain = link_rel_err(F, F_ref)
    assert e < TOL64, (e, plain)
    S_g, S_F, K, _ = lgt.lgt_action(lat.ctx, tol, 10 * V)
    n2 = np.sum(np.abs(eta) ** 2)
    assert abs(S_F - n2) < 1e-11 * n2
    # one kick: Pi -= eps (F^g + F^eo)
    P0 = synth.gaussian_momenta(dims, 40)
    lat.set_momenta(P0)
    its = lgt.lgt_md_kick(lat.ctx, 0.05, tol, 10 * V)
    assert its == it_ref
    P_ref = P0 - 0.05 * (oracle.gauge_force(dims, beta, U) + F_ref)
    assert link_rel_err(lat.get_momenta(), P_ref)[0] < TOL64
    # the full action is untouched by the switch back
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_FULL)
    _, S_full, _, _ = lgt.lgt_action(lat.ctx, tol, 10 * V)
    S_full_ref, _, _, _ = oracle.fermion_action(dims, kappa, BC, U, phi, tol, 10 * V)
    assert abs(S_full - S_full_ref) < 1e-10 * abs(S_full_ref)
    lat.close()


def test_eo_mixed_precision_solver(lgt):
    """Even/odd action with the mixed-precision solver (fp32 CG on the Schur complement, fp64 defect correction on the
    true residual): same force and action as the oracle's fp64 solve, and through a links change (stale fp32 copies)."""
    dims, kappa, tol = (8, 8, 8, 8), 0.12, 1e-12
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 47)
    phi = oeo.mhat(dims, kappa, BC, U, oeo.keep(synth.gaussian_spinor(dims, 48), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U, phi, tol, 10 * V)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    F, it = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert 0 < it < 2 * it_ref + 20  # fp32 iterations in total
    e, plain = link_rel_err(F, F_ref)
    assert e < 1e-10, (e, plain)
    _, S_F, _, _ = lgt.lgt_action(lat.ctx, tol, 10 * V)
    S_ref = oeo.action(dims, kappa, BC, U, phi, tol, 10 * V)[0]
    assert abs(S_F - S_ref) < 1e-11 * abs(S_ref)
    # new links: the fp32 checkerboard copy must follow
    U2 = synth.warm_links(dims, 0.25, 49)
    lat.set_links(U2)
    F2, _ = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    F2_ref, _, _ = oeo.fermion_force(dims, kappa, BC, U2, phi, tol, 10 * V)
    assert link_rel_err(F2, F2_ref)[0] < 1e-10
    lat.close()


@pytest.mark.parametrize("bc", [BC, (-1, -1, -1, -1)])
def test_eo_mixed_solver_inner_hops_on_twelve_real_links(lgt, bc):
    """On lattices of more than two waves of blocks the fp32 INNER solve of the even/odd mixed-precision solver reads rows 0 and 1
    of every link and rebuilds row 2 with the folded fermion boundary sign (hop_cb_kernel PFL 2; the fp64 defect correction
    keeps the exact operator).  320 blocks per half field here: force against the oracle's fp64 even/odd solve, and the same
    iteration count (+- 2) and force as with the exact-link inner hops (any other Dslash variant selects them).  A plain fp32
    handle keeps the exact links unless variant 12 is selected; with it the solve agrees to fp32 rounding."""
    dims, kappa, tol = (16, 16, 16, 20), 0.12, 1e-12
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 147)
    phi = oeo.mhat(dims, kappa, bc, U, oeo.keep(synth.gaussian_spinor(dims, 148), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, bc, U, phi, tol, 10 * V)
    lat = lgt.Lattice(dims, 5.5, kappa, bc)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    F, it = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert 0 < it < 2 * it_ref + 20
    assert link_rel_err(F, F_ref)[0] < 1e-10
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 8) == 8  # exact 9-entry links in the inner hops
    F9, it9 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert abs(it - it9) <= 2 and link_rel_err(F9, F_ref)[0] < 1e-10
    # the same on one level of stout links (special unitary as well, boundary sign folded the same way)
    lgt.lgt_set_smearing(lat.ctx, 1, 0.3)
    Fs9, its9 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 0) == 0
    Fs12, its12 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert abs(its9 - its12) <= 2 and link_rel_err(Fs12, Fs9)[0] < 1e-10
    lgt.lgt_set_smearing(lat.ctx, 0, 0.0)
    # the fp64 hops themselves on 12-real links (variant 12, opt-in): same solve to rounding, same count
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_CG)
    b64 = synth.gaussian_spinor(dims, 150)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 0) == 0
    x0, it0, _, ok0 = lat.eo_cg(b64, tol, 10 * V)
    assert lgt.lgt_set_kernel_variant(lat.ctx, lgt.LGT_K_DSLASH, 12) == 12
    x12, it12, _, ok12 = lat.eo_cg(b64, tol, 10 * V)
    assert ok0 and ok12 and it0 == it12 and np.abs(x12 - x0).max() < 1e-12 * np.abs(x0).max()
    lat.close()
    # fp32 handle: variant 12 against the default's exact links
    b = round32(synth.gaussian_spinor(dims, 149))
    l32 = lgt.Lattice(dims, 5.5, kappa, bc, precision=lgt.LGT_F32)
    l32.set_links(round32(U))
    x0, it0, _, ok0 = l32.eo_cg(b, 1e-5, 3000)
    assert lgt.lgt_set_kernel_variant(l32.ctx, lgt.LGT_K_DSLASH, 12) == 12
    x12, it12, _, ok12 = l32.eo_cg(b, 1e-5, 3000)
    assert ok0 and ok12 and abs(it0 - it12) <= 1
    even = np.abs(x0).reshape(V, -1).max(axis=1) > 0
    assert np.linalg.norm((x12 - x0)[even]) < 1e-4 * np.linalg.norm(x0[even])
    l32.close()


def test_eo_mixed_solver_survives_links_off_the_group(lgt):
    """Links that are not special unitary (here 1.03 U): the 12-real inner hops rebuild a third row that is off by 3 %, the first
    correction cycle does not contract, and the solver falls back to the exact fp32 links (mixed_inner_fallback).  The force is
    the oracle's for these links to 1e-10; the price is iterations, never accuracy."""
    dims, kappa, tol = (16, 16, 16, 20), 0.11, 1e-12
    V = synth.volume(dims)
    U = 1.03 * synth.warm_links(dims, 0.3, 157)
    phi = oeo.mhat(dims, kappa, BC, U, oeo.keep(synth.gaussian_spinor(dims, 158), dims, 0), dagger=True)
    F_ref, it_ref, _ = oeo.fermion_force(dims, kappa, BC, U, phi, tol, 10 * V)
    lat = lgt.Lattice(dims, 5.5, kappa, BC)
    lat.set_links(U)
    lat.set_pseudofermion(phi)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lgt.lgt_set_solver(lat.ctx, lgt.LGT_SOLVER_MIXED_CG, 1e-5)
    F, it = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert link_rel_err(F, F_ref)[0] < 1e-10
    assert it_ref <= it < 4 * it_ref + 40  # one wasted inner solve at most, then the usual count
    F2, it2 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)  # the fallback holds while the links stay
    assert link_rel_err(F2, F_ref)[0] < 1e-10 and it2 < it  # (78, then 48 fp32 iterations when this was written)
    lat.close()


def test_eo_leapfrog_conserves_energy(lgt):
    """Leapfrog with the even/odd action on 8^4: |dH| ~ dt^2 and exact reversibility (pin P7 on this action)."""
    dims, beta, kappa = (8, 8, 8, 8), 5.6, 0.12
    U0 = synth.warm_links(dims, 0.3, 47)
    P0 = synth.gaussian_momenta(dims, 48)
    phi = synth.gaussian_spinor(dims, 49)
    lat = lgt.Lattice(dims, beta, kappa, BC)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    lat.set_pseudofermion(phi)
    dH = []
    for n, dt in ((8, 0.02), (16, 0.01)):
        lat.set_links(U0)
        lat.set_momenta(P0)
        H0, H1, _ = lgt.lgt_md_trajectory(lat.ctx, n, dt, 1e-13, 20000)
        dH.append(abs(H1 - H0))
    assert dH[0] < 5.0 and 3.5 < dH[0] / dH[1] < 4.5, dH
    lat.set_momenta(-lat.get_momenta())
    lgt.lgt_md_trajectory(lat.ctx, 16, 0.01, 1e-13, 20000)
    assert np.abs(lat.get_links() - U0).max() < 1e-10
    lat.close()


def test_eo_refuses_odd_extents(lgt):
    lat = lgt.Lattice((4, 3, 4, 4), 5.5, 0.1, BC)
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    assert e.value.code == lgt.LGT_EINVAL
    with pytest.raises(lgt.LgtError):
        lat.eo_mhat(synth.gaussian_spinor((4, 3, 4, 4), 1))
    lat.close()


@pytest.mark.parametrize("dims", [(4, 3, 5, 6), (6, 2, 1, 10), (3, 3, 3, 3), (8, 8, 8, 8)])
def test_fermion_force_ragged_shapes(lgt, dims):
    """Force kernel alone on shapes that do not fill a 128-site block, with extents of 1 and 2 (forward and
    backward neighbour coincide) and every boundary-sign pattern: rounding-level agreement per link."""
    kappa = 0.12
    U = synth.warm_links(dims, 0.3, 21)
    X = synth.gaussian_spinor(dims, 22)
    Y = synth.gaussian_spinor(dims, 23)
    for bc in (BC, (1, 1, 1, 1), (-1, -1, 1, -1)):
        lat = lgt.Lattice(dims, 5.6, kappa, bc)
        lat.set_links(U)
        F, _ = lat.fermion_force(X, Y)
        e, plain = link_rel_err(F, oracle.fermion_force(dims, kappa, bc, U, X, Y))
        assert e < 1e-13, (dims, bc, e, plain)
        # traceless anti-Hermitian output (Eq. 7 of the paper)
        assert np.abs(F + F.conj().swapaxes(-1, -2)).max() < 1e-15
        assert np.abs(np.trace(F, axis1=-2, axis2=-1)).max() < 1e-15
        lat.close()


def test_fermion_force_fp32(lgt):
    dims, kappa = (8, 8, 8, 8), 0.12
    U = round32(synth.warm_links(dims, 0.3, 3))
    X = round32(synth.gaussian_spinor(dims, 4))
    Y = round32(synth.gaussian_spinor(dims, 5))
    lat = lgt.Lattice(dims, 5.6, kappa, BC, precision=lgt.LGT_F32)
    lat.set_links(U)
    F, _ = lat.fermion_force(X, Y)
    e, plain = link_rel_err(F.astype(np.complex128), oracle.fermion_force(dims, kappa, BC, U, X, Y))
    assert e < TOL32, (e, plain)
    lat.close()


@pytest.mark.parametrize("dims", [(4, 3, 5, 6), (8, 8, 8, 8), (6, 2, 1, 10)])
def test_gauge_force_and_action(lgt, dims):
    beta = 6.0
    U = synth.haar_links(dims, 1101)
    lat = lgt.Lattice(dims, beta, 0.0, (1, 1, 1, 1))
    lat.set_links(U)
    F = lat.gauge_force()
    e, plain = link_rel_err(F, oracle.gauge_force(dims, beta, U))
    assert e < 1e-13, (e, plain)
    S_ref, plaq_ref = oracle.gauge_action(dims, beta, U)
    S_g, S_F, K, _ = lgt.lgt_action(lat.ctx)
    assert abs(S_g - S_ref) < 1e-12 * abs(S_ref) and S_F == 0.0 and K == 0.0
    assert abs(lgt.lgt_plaquette(lat.ctx) - plaq_ref) < 1e-14
    lat.close()
    # fp32
    U32 = round32(U)
    lat = lgt.Lattice(dims, beta, 0.0, (1, 1, 1, 1), precision=lgt.LGT_F32)
    lat.set_links(U32)
    e, plain = link_rel_err(lat.gauge_force().astype(np.complex128), oracle.gauge_force(dims, beta, U32))
    assert e < TOL32, (e, plain)
    lat.close()


def test_unit_gauge(lgt):
    dims = (4, 4, 4, 4)
    lat = lgt.Lattice(dims, 5.5, 0.1, BC)
    assert lgt.lgt_plaquette(lat.ctx) == 1.0
    S_g, S_F, K, _ = lgt.lgt_action(lat.ctx)
    assert S_g == 0.0
    assert not lat.gauge_force().any()
    lat.close()


@pytest.mark.parametrize("scale", [1e-9, 1e-3, 0.02, 1.0, 4.0])
def test_drift_matches_taylor_exponential(lgt, scale):
    dims = (4, 3, 5, 6)
    U = synth.warm_links(dims, 0.3, 1)
    P = synth.gaussian_momenta(dims, 2)
    # degenerate eigenvalue corners of the Cayley-Hamilton form: lambda_8 direction (both signs), zero momentum
    l8 = 0.5j * synth.gell_mann()[7]
    P[0, 0], P[1, 0], P[2, 0] = l8, -l8, 0.0
    lat = lgt.Lattice(dims, 5.6, 0.12, BC)
    lat.set_links(U)
    lat.set_momenta(P)
    lgt.lgt_md_drift(lat.ctx, scale)
    ref = oracle.drift(dims, scale, P, U)
    assert np.abs(lat.get_links() - ref).max() < 2e-14 * max(1.0, scale)
    lat.close()


def test_kick_and_momentum_kinetic(lgt):
    c = synth.CONFIGS[0]
    dims, beta, kappa, bc = c["dims"], c["beta"], c["kappa"], c["bc"]
    U = synth.config_links(0)
    P = synth.gaussian_momenta(dims, 5)
    phi = oracle.dslash(dims, kappa, bc, U, synth.gaussian_spinor(dims, c["seed_eta"]), dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    lat.set_momenta(P)
    lat.set_pseudofermion(phi)
    S_g, S_F, K, _ = lgt.lgt_action(lat.ctx, 1e-13, 5000)
    assert abs(K - oracle.kinetic(dims, P)) < 1e-12 * K
    it = lgt.lgt_md_kick(lat.ctx, 0.05, 1e-13, 5000)
    P_ref, it_ref, ok = oracle.kick(dims, beta, kappa, bc, U, phi, P, 0.05, 1e-13, 5000)
    assert ok and it == it_ref
    e, plain = link_rel_err(lat.get_momenta(), P_ref)
    assert e < TOL64
    lat.close()


def test_config1_leapfrog_trajectory(lgt):
    """configs[1]: 8^4 gauge-only, Haar links, 50 leapfrog steps at dt = 0.02: final state against the oracle's
    trajectory, dH against the oracle's dH, dt^2 scaling and reversibility on the GPU itself."""
    c = synth.CONFIGS[1]
    dims, beta, bc = c["dims"], c["beta"], c["bc"]
    U0 = synth.config_links(1)
    P0 = synth.gaussian_momenta(dims, c["seed_mom"])
    lat = lgt.Lattice(dims, beta, 0.0, bc)
    lat.set_links(U0)
    lat.set_momenta(P0)
    H0, H1, _ = lgt.lgt_md_trajectory(lat.ctx, c["nsteps"], c["dt"])
    U1, P1 = lat.get_links(), lat.get_momenta()
    U_ref, P_ref, _, _ = oracle.trajectory(dims, beta, 0.0, bc, U0, None, P0, c["nsteps"], c["dt"])
    H0_ref = oracle.hamiltonian(dims, beta, 0.0, bc, U0, None, P0)[0]
    H1_ref = oracle.hamiltonian(dims, beta, 0.0, bc, U_ref, None, P_ref)[0]
    assert abs(H0 - H0_ref) < 1e-12 * abs(H0_ref)
    assert abs((H1 - H0) - (H1_ref - H0_ref)) < 1e-9 * abs(H0_ref) + 1e-6 * abs(H1_ref - H0_ref)
    assert np.abs(U1 - U_ref).max() < 1e-11
    assert link_rel_err(P1, P_ref)[0] < TOL64
    # reversibility: flip the momenta, run again
    lat.set_momenta(-P1)
    lgt.lgt_md_trajectory(lat.ctx, c["nsteps"], c["dt"], measure=False)
    assert np.abs(lat.get_links() - U0).max() < 1e-11
    assert np.abs(lat.get_momenta() + P0).max() < 1e-10
    # dt -> dt/2 at fixed length: |dH| drops by about 4
    lat.set_links(U0)
    lat.set_momenta(P0)
    h0, h1, _ = lgt.lgt_md_trajectory(lat.ctx, 2 * c["nsteps"], c["dt"] / 2)
    ratio = (H1 - H0) / (h1 - h0)
    assert 3.5 < ratio < 4.5, ratio
    lat.close()


def test_md_step_with_fermions(lgt):
    c = synth.CONFIGS[0]
    dims, beta, kappa, bc = c["dims"], c["beta"], c["kappa"], c["bc"]
    U0 = synth.config_links(0)
    P0 = synth.gaussian_momenta(dims, 73)
    phi = oracle.dslash(dims, kappa, bc, U0, synth.gaussian_spinor(dims, c["seed_eta"]), dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U0)
    lat.set_momenta(P0)
    lat.set_pseudofermion(phi)
    its = lgt.lgt_md_step(lat.ctx, 0.05, 1e-13, 5000)
    U_ref, P_ref, its_ref, ok = oracle.trajectory(dims, beta, kappa, bc, U0, phi, P0, 1, 0.05, tol=1e-13, max_iter=5000)
    assert ok and its == its_ref
    assert np.abs(lat.get_links() - U_ref).max() < 1e-12
    assert link_rel_err(lat.get_momenta(), P_ref)[0] < TOL64
    lat.close()


def test_error_paths(lgt):
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_create((4, 4, 4, 0), 5.5, 0.1, BC)
    assert e.value.code == lgt.LGT_EINVAL
    with pytest.raises(lgt.LgtError):
        lgt.lgt_create((4, 4, 4, 4), 5.5, 0.1, (1, 1, 1, 0))
    with pytest.raises(lgt.LgtError):
        lgt.lgt_create((4, 4, 4, 4), 5.5, 0.1, BC, precision=7)
    lat = lgt.Lattice((4, 4, 4, 4), 5.5, 0.1, BC)
    with pytest.raises(lgt.LgtError) as e:
        lgt.lgt_set_links(lat.ctx, None)
    assert e.value.code == lgt.LGT_EINVAL
    F = lat.empty(lat.V, 4, 3, 3)
    with pytest.raises(lgt.LgtError) as e:  # no pseudofermion set
        lgt.lgt_fermion_force(lat.ctx, None, None, F)
    assert e.value.code == lgt.LGT_ESTATE
    # CG cap: reports non-convergence, leaves the last iterate
    U = synth.warm_links((4, 4, 4, 4), 0.3, 1)
    lat.set_links(U)
    b = synth.gaussian_spinor((4, 4, 4, 4), 2)
    x, it, rel, ok = lat.cg(b, 1e-13, 3)
    x_ref, it_ref, rel_ref, ok_ref = oracle.cg((4, 4, 4, 4), 0.1, BC, U, b, 1e-13, 3)
    assert not ok and it == 3 and not ok_ref and abs(rel - rel_ref) < 1e-12
    assert site_rel_err(x, x_ref) < 1e-12
    # zero right-hand side: zero iterations, zero solution
    x, it, rel, ok = lat.cg(np.zeros_like(b), 1e-13, 10)
    assert ok and it == 0 and not x.any()
    lat.close()


# ------------------------------------------------------------------------------------------------ full sizes
def _sample_sites(V, n, seed):
    rng = np.random.default_rng(seed)
    # first / last sites (all boundaries), plus a random sample
    return np.unique(np.concatenate([[0, 1, 31, 32, V - 1, V - 32, V // 2], rng.integers(0, V, n)]))


def test_config3_full_size_kernels_sampled(lgt):
    """configs[3] (32^4, the bench workload): Dslash, fermion force and gauge force at full size in the launch
    shapes bench.py times, compared on sampled sites / links that the oracle computes one by one."""
    c = synth.CONFIGS[3]
    dims, beta, kappa, bc = c["dims"], c["beta"], c["kappa"], c["bc"]
    V = synth.volume(dims)
    U = synth.config_links(3)
    X = synth.gaussian_spinor(dims, 11)
    Y = synth.gaussian_spinor(dims, 12)
    sites = _sample_sites(V, 200, 13)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    for dag in (False, True):
        out = lat.dslash(X, dagger=dag)
        ref = oracle.dslash_sites(dims, kappa, bc, U, X, sites, dagger=dag)
        assert site_rel_err(out[sites], ref) < TOL64
    F, _ = lat.fermion_force(X, Y)
    G = lat.gauge_force()
    worst_f = worst_g = 0.0
    for s in sites[:60]:
        for mu in range(4):
            rf = oracle.fermion_force_link(dims, kappa, bc, U, X, Y, int(s), mu)
            rg = oracle.gauge_force_link(dims, beta, U, int(s), mu)
            worst_f = max(worst_f, np.linalg.norm(F[s, mu] - rf) / np.linalg.norm(rf))
            worst_g = max(worst_g, np.linalg.norm(G[s, mu] - rg) / np.linalg.norm(rg))
    assert worst_f < TOL64 and worst_g < TOL64, (worst_f, worst_g)
    # fp32 variant of the same lattice (configs[3]: "also run as an fp32 Dslash and force variant")
    lat.close()
    U32, X32, Y32 = round32(U), round32(X), round32(Y)
    lat = lgt.Lattice(dims, beta, kappa, bc, precision=lgt.LGT_F32)
    lat.set_links(U32)
    out = lat.dslash(X32).astype(np.complex128)
    assert site_rel_err(out[sites], oracle.dslash_sites(dims, kappa, bc, U32, X32, sites)) < TOL32
    F32, _ = lat.fermion_force(X32, Y32)
    worst = 0.0
    for s in sites[:40]:
        for mu in range(4):
            rf = oracle.fermion_force_link(dims, kappa, bc, U32, X32, Y32, int(s), mu)
            worst = max(worst, np.linalg.norm(F32[s, mu].astype(np.complex128) - rf) / np.linalg.norm(rf))
    assert worst < TOL32, worst
    lat.close()


def test_config3_full_size_md_step(lgt):
    """configs[3]: one full MD step at 32^4 exactly as bench.py runs it (kick(dt) then drift(dt), CG to 1e-12):
    CG iteration count identical to the oracle's, momenta and links per link within 1e-11."""
    c = synth.CONFIGS[3]
    dims, beta, kappa, bc, tol, dt = c["dims"], c["beta"], c["kappa"], c["bc"], c["cg_tol"], c["dt"]
    V = synth.volume(dims)
    U = synth.config_links(3)
    P = synth.gaussian_momenta(dims, c["seed_mom"])
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    lat.set_momenta(P)
    lat.set_pseudofermion(phi)
    it = lgt.lgt_md_kick(lat.ctx, dt, tol, 10 * V)
    lgt.lgt_md_drift(lat.ctx, dt)
    P1, U1 = lat.get_momenta(), lat.get_links()
    lat.close()
    P_ref, it_ref, ok = oracle.kick(dims, beta, kappa, bc, U, phi, P, dt, tol, 10 * V)
    U_ref = oracle.drift(dims, dt, P_ref, U)
    assert ok and it == it_ref, (it, it_ref)
    assert link_rel_err(P1, P_ref)[0] < TOL64
    assert np.abs(U1 - U_ref).max() < 1e-13


def test_config3_full_size_solver_variants(lgt):
    """configs[3] at full size for the two SURVEY 8(f)1 solver variants, as bench.py's `extras` runs them, checked by
    properties the oracle can evaluate in seconds at 32^4: the TRUE residual of the returned solution taken with the
    oracle's D (mixed precision), resp. with the oracle's M (even/odd), and the even/odd force on sampled links
    against the oracle's per-link force evaluated on the GPU's reconstructed X, Y."""
    c = synth.CONFIGS[3]
    dims, beta, kappa, bc, tol = c["dims"], c["beta"], c["kappa"], c["bc"], c["cg_tol"]
    V = synth.volume(dims)
    U = synth.config_links(3)
    eta = synth.gaussian_spinor(dims, c["seed_eta"])
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    nphi = np.linalg.norm(phi)
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    X, inner, outer, rel, ok = lat.cg_mixed(phi, tol, 10 * V)
    assert ok and rel <= tol and outer <= 6 and inner < 400, (inner, outer, rel)
    AX = oracle.dslash(dims, kappa, bc, U, oracle.dslash(dims, kappa, bc, U, X), dagger=True)
    assert np.linalg.norm(phi - AX) / nphi <= 1.05 * tol
    # phi = D^dag eta  =>  X = D^-1 eta, so D X = eta (pin P6) also holds for the mixed solver's X
    assert site_rel_err(oracle.dslash(dims, kappa, bc, U, X), eta) < 1e-9
    del AX
    Xe, it, rel, ok = lat.eo_cg(phi, tol, 10 * V)
    assert ok and 20 < it < 159, it  # fewer iterations than the unpreconditioned solve (159)
    even = oeo.parity(dims) == 0
    r = oeo.keep(phi, dims, 0) - oeo.mhat(dims, kappa, bc, U, oeo.mhat(dims, kappa, bc, U, Xe), dagger=True)
    assert np.linalg.norm(r) / np.linalg.norm(phi[even]) <= 3 * tol  # recurrence vs true residual
    # force through the action switch, sampled links; X, Y rebuilt by the oracle from the GPU's X_e
    lat.set_pseudofermion(phi)
    lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
    F, it2 = lat.fermion_force(None, None, tol=tol, max_iter=10 * V)
    assert it2 == it
    Ye = oeo.mhat(dims, kappa, bc, U, Xe)
    Xf = Xe - oeo.keep(oracle.dslash(dims, kappa, bc, U, Xe), dims, 1)
    Yf = Ye - oeo.keep(oracle.dslash(dims, kappa, bc, U, Ye, dagger=True), dims, 1)
    worst = 0.0
    for s_ in _sample_sites(V, 30, 9)[:24]:
        for mu in range(4):
            rf = oracle.fermion_force_link(dims, kappa, bc, U, Xf, Yf, int(s_), mu)
            worst = max(worst, np.linalg.norm(F[s_, mu] - rf) / np.linalg.norm(rf))
    assert worst < TOL64, worst
    lat.close()


def test_config4_largest_lattice_sampled(lgt):
    """configs[4] (48^3 x 96, the largest single-GPU working set, Lx not a multiple of the 32-site layout block; fp64 and
    fp32; "Dslash, CG on D^dag D to 1e-10, fermion force and gauge force"), in the launch shape bench.py's configs4 sweep
    times: D and D^dag, both forces on sampled sites / links against the oracle's per-site routines; one CG solve to
    1e-10 checked by its TRUE residual with the oracle's D (two full oracle Dslashes) and by D X = eta; the fp32 Dslash
    and both fp32 forces at 2e-5.  The links are a periodic tiling of a seeded 24^4 warm field (a valid SU(3)
    configuration of the full size that takes seconds, not minutes, to make on the host)."""
    import torch

    dims, beta, kappa, bc = (48, 48, 48, 96), 5.6, 0.12, BC
    free, _ = torch.cuda.mem_get_info()
    assert free > 40e9, "configs[4] needs about 40 GB of free device memory; found %.1f GB" % (free / 1e9)
    V = synth.volume(dims)
    small = synth.warm_links((24, 24, 24, 24), 0.3, 1401).reshape(24, 24, 24, 24, 4, 3, 3)
    U = np.tile(small, (4, 2, 2, 2, 1, 1, 1)).reshape(V, 4, 3, 3)
    X = synth.gaussian_spinor(dims, 1402)
    Y = synth.gaussian_spinor(dims, 1403)
    # sampled sites, plus the corners of the index range and sites next to the antiperiodic time boundary
    sites = np.unique(np.concatenate([_sample_sites(V, 100, 5), np.array([0, 47, 48 * 48 - 1, V - 1, V - 48 ** 3, V - 48 ** 3 - 1], dtype=np.int64)]))
    lat = lgt.Lattice(dims, beta, kappa, bc)
    lat.set_links(U)
    for dag in (False, True):
        out = lat.dslash(X, dagger=dag)
        assert site_rel_err(out[sites], oracle.dslash_sites(dims, kappa, bc, U, X, sites, dagger=dag)) < TOL64
        del out
    F, _ = lat.fermion_force(X, Y)
    G = lat.gauge_force()
    worst_f = worst_g = 0.0
    for s in sites[:40]:
        for mu in range(4):
            rf = oracle.fermion_force_link(dims, kappa, bc, U, X, Y, int(s), mu)
            rg = oracle.gauge_force_link(dims, beta, U, int(s), mu)
            worst_f = max(worst_f, np.linalg.norm(F[s, mu] - rf) / np.linalg.norm(rf))
            worst_g = max(worst_g, np.linalg.norm(G[s, mu] - rg) / np.linalg.norm(rg))
    assert worst_f < TOL64 and worst_g < TOL64, (worst_f, worst_g)
    del F, G
    # CG on D^dag D to 1e-10 with phi = D^dag eta: true residual by the oracle's operator, and D X = eta (pin P6)
    eta = Y
    phi = oracle.dslash(dims, kappa, bc, U, eta, dagger=True)
    Xs, it, rel, ok = lat.cg(phi, 1e-10, 10 * V)
    assert ok and rel <= 1e-10 and 50 < it < 400, (it, rel)
    DX = oracle.dslash(dims, kappa, bc, U, Xs)
    assert np.linalg.norm(phi - oracle.dslash(dims, kappa, bc, U, DX, dagger=True)) <= 1.05e-10 * np.linalg.norm(phi)
    assert site_rel_err(DX, eta) < 1e-7
    del DX, Xs, phi
    lat.close()
    # fp32 (2e-5): inputs rounded to fp32 first (reading A-21)
    U32, X32, Y32 = round32(U), round32(X), round32(Y)
    del U, X, Y
    lat = lgt.Lattice(dims, beta, kappa, bc, precision=lgt.LGT_F32)
    lat.set_links(U32)
    for dag in (False, True):
        out = lat.dslash(X32, dagger=dag).astype(np.complex128)
        assert site_rel_err(out[sites], oracle.dslash_sites(dims, kappa, bc, U32, X32, sites, dagger=dag)) < TOL32
        del out
    F32, _ = lat.fermion_force(X32, Y32)
    G32 = lat.gauge_force()
    worst_f = worst_g = 0.0
    for s in sites[:30]:
        for mu in range(4):
            rf = oracle.fermion_force_link(dims, kappa, bc, U32, X32, Y32, int(s), mu)
            rg = oracle.gauge_force_link(dims, beta, U32, int(s), mu)
            worst_f = max(worst_f, np.linalg.norm(F32[s, mu].astype(np.complex128) - rf) / np.linalg.norm(rf))
            worst_g = max(worst_g, np.linalg.norm(G32[s, mu].astype(np.complex128) - rg) / np.linalg.norm(rg))
    assert worst_f < TOL32 and worst_g < TOL32, (worst_f, worst_g)
    lat.close()


def test_cg_graph_replay_is_bitwise_the_plain_launches(lgt):
    """The CG chunks run as CUDA graphs; with per-kernel timing on they fall back to plain launches.  Same kernels, same
    order: solution, iteration count and the even/odd force must be bit-identical, and repeated solves reuse the graph."""
    dims, kappa = (8, 8, 8, 8), 0.12
    V = synth.volume(dims)
    U = synth.warm_links(dims, 0.3, 71)
    b = oracle.dslash(dims, kappa, BC, U, synth.gaussian_spinor(dims, 72), dagger=True)
    lat = lgt.Lattice(dims, 5.6, kappa, BC)
    lat.set_links(U)
    lat.set_pseudofermion(b)
    out = {}
    for timing in (False, True, False):
        lgt.lgt_timing_enable(lat.ctx, timing)
        n0 = lgt.lgt_launch_count(lat.ctx)
        x, it, rel, ok = lat.cg(b, 1e-12, 10 * V)
        launches = lgt.lgt_launch_count(lat.ctx) - n0
        lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_EO)
        F, it_eo = lat.fermion_force(None, None, tol=1e-12, max_iter=10 * V)
        lgt.lgt_set_fermion_action(lat.ctx, lgt.LGT_ACTION_FULL)
        out.setdefault("runs", []).append((x, it, F, it_eo, launches))
    lgt.lgt_timing_enable(lat.ctx, False)
    lgt.lgt_timing_reset(lat.ctx)
    ref = out["runs"][1]  # plain launches
    for run in (out["runs"][0], out["runs"][2]):
        assert run[1] == ref[1] and run[3] == ref[3] and run[4] == ref[4]  # counts incl. the kernels inside the graphs
        assert np.array_equal(run[0], ref[0]) and np.array_equal(run[2], ref[2])
    x_ref, it_ref, _, _ = oracle.cg(dims, kappa, BC, U, b, 1e-12, 10 * V)
    assert ref[1] == it_ref
    lat.close()
