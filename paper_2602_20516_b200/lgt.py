"""Thin Python binding over the C-ABI CUDA library liblgt.so (include/lgt.h).

Argument marshalling only: every step of the path runs in the CUDA kernels.  Functions carry
the names of the C entry points; `Lattice` bundles a handle with torch-allocated buffers.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback: if the
library is not built or no CUDA device is present, calls raise.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblgt.so")

LGT_OK, LGT_EINVAL, LGT_ENOMEM, LGT_ECUDA, LGT_ENOCONV, LGT_ESTATE = 0, -1, -2, -3, -4, -5
LGT_F64, LGT_F32 = 0, 1
LGT_SOLVER_CG, LGT_SOLVER_MIXED_CG = 0, 1
LGT_ACTION_FULL, LGT_ACTION_EO = 0, 1
LGT_INT_LEAPFROG, LGT_INT_OMELYAN, LGT_INT_SEXTON_WEINGARTEN = 0, 1, 2
LGT_DD_EXCHANGE, LGT_DD_PUSH, LGT_DD_OVERLAP, LGT_DD_HALF = 0, 1, 2, 3
LGT_NOALLOC_MAX_SITES = 1 << 24

# every symbol include/lgt.h declares: (restype, argtypes)
_vp, _i, _d, _l = C.c_void_p, C.c_int, C.c_double, C.c_long
_ip, _dp, _lp = C.POINTER(C.c_int), C.POINTER(C.c_double), C.POINTER(C.c_long)
SYMBOLS = {
    "lgt_create": (_i, [C.POINTER(_vp), _ip, _d, _d, _ip, _i, _i, _vp]),
    "lgt_destroy": (_i, [_vp]),
    "lgt_last_error": (C.c_char_p, [_vp]),
    "lgt_version": (C.c_char_p, []),
    "lgt_set_links": (_i, [_vp, _vp]),
    "lgt_get_links": (_i, [_vp, _vp]),
    "lgt_set_momenta": (_i, [_vp, _vp]),
    "lgt_get_momenta": (_i, [_vp, _vp]),
    "lgt_set_pseudofermion": (_i, [_vp, _vp]),
    "lgt_set_links_host": (_i, [_vp, _vp]),
    "lgt_get_links_host": (_i, [_vp, _vp]),
    "lgt_set_momenta_host": (_i, [_vp, _vp]),
    "lgt_get_momenta_host": (_i, [_vp, _vp]),
    "lgt_set_pseudofermion_host": (_i, [_vp, _vp]),
    "lgt_set_momenta_host_async": (_i, [_vp, _vp]),
    "lgt_get_links_host_async": (_i, [_vp, _vp]),
    "lgt_get_momenta_host_async": (_i, [_vp, _vp]),
    "lgt_host_transfers_wait": (_i, [_vp]),
    "lgt_action": (_i, [_vp, _d, _i, _dp, _dp, _dp, _ip]),
    "lgt_plaquette": (_i, [_vp, _dp]),
    "lgt_dslash": (_i, [_vp, _vp, _vp, _i]),
    "lgt_cg": (_i, [_vp, _vp, _vp, _d, _i, _ip, _dp]),
    "lgt_gauge_force": (_i, [_vp, _vp]),
    "lgt_fermion_force": (_i, [_vp, _vp, _vp, _vp, _d, _i, _ip]),
    "lgt_md_kick": (_i, [_vp, _d, _d, _i, _ip]),
    "lgt_md_drift": (_i, [_vp, _d]),
    "lgt_md_step": (_i, [_vp, _d, _d, _i, _ip]),
    "lgt_md_trajectory": (_i, [_vp, _i, _d, _d, _i, _dp, _dp, _lp]),
    "lgt_native_spinor_bytes": (_l, [_vp]),
    "lgt_spinor_to_native": (_i, [_vp, _vp, _vp]),
    "lgt_spinor_from_native": (_i, [_vp, _vp, _vp]),
    "lgt_dslash_native": (_i, [_vp, _vp, _vp, _i]),
    "lgt_fermion_force_native": (_i, [_vp, _vp, _vp, _d]),
    "lgt_gauge_force_accumulate": (_i, [_vp, _d]),
    "lgt_cg_native": (_i, [_vp, _vp, _vp, _vp, _d, _i, _ip, _dp]),
    "lgt_timing_enable": (_i, [_vp, _i]),
    "lgt_timing_reset": (_i, [_vp]),
    "lgt_timing_read": (_i, [_vp, _i, _dp, _lp]),
    "lgt_measure_peaks": (_i, [_vp, _i, _dp, _dp, _dp, _dp]),
    "lgt_launch_count": (_l, [_vp]),
    "lgt_stream": (_vp, [_vp]),
    "lgt_set_block_swizzle": (_i, [_vp, _i, _ip]),
    "lgt_set_kernel_variant": (_i, [_vp, _i, _i, _ip]),
    "lgt_cg_mixed": (_i, [_vp, _vp, _vp, _d, _i, _d, _ip, _ip, _dp]),
    "lgt_set_solver": (_i, [_vp, _i, _d]),
    "lgt_eo_mhat": (_i, [_vp, _vp, _vp, _i]),
    "lgt_eo_cg": (_i, [_vp, _vp, _vp, _d, _i, _ip, _dp]),
    "lgt_set_fermion_action": (_i, [_vp, _i]),
    "lgt_dd_create": (_i, [C.POINTER(_vp), _ip, _i, _i, _ip, _d, _d, _ip, _i, _i, _vp]),
    "lgt_dd_create_grid": (_i, [C.POINTER(_vp), _ip, _ip, _i, _ip, _d, _d, _ip, _i, _i, _vp]),
    "lgt_dd_destroy": (_i, [_vp]),
    "lgt_dd_last_error": (C.c_char_p, [_vp]),
    "lgt_dd_nccl_unique_id": (_i, [_vp]),
    "lgt_dd_nccl_init": (_i, [_vp, _vp]),
    "lgt_dd_set_host_transport": (_i, [_vp, _vp, _vp, _vp]),
    "lgt_dd_halo_plan": (_i, [_i, _i, _i, _ip]),
    "lgt_dd_set_halo_mode": (_i, [_vp, _i]),
    "lgt_dd_ipc_export": (_i, [_vp, _vp]),
    "lgt_dd_ipc_import": (_i, [_vp, _vp, _vp]),
    "lgt_dd_local_ranks": (_i, [_vp]),
    "lgt_dd_rank": (_vp, [_vp, _i]),
    "lgt_dd_dslash": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp), _i]),
    "lgt_dd_cg": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp), _d, _i, _ip, _dp]),
    "lgt_dd_action": (_i, [_vp, _d, _i, _dp, _dp, _dp, _ip]),
    "lgt_dd_set_solver": (_i, [_vp, _i, _d]),
    "lgt_dd_set_fermion_action": (_i, [_vp, _i]),
    "lgt_dd_set_smearing": (_i, [_vp, _i, _d]),
    "lgt_dd_set_integrator": (_i, [_vp, _i, _i]),
    "lgt_dd_md_kick": (_i, [_vp, _d, _d, _i, _ip]),
    "lgt_dd_md_drift": (_i, [_vp, _d]),
    "lgt_dd_md_trajectory": (_i, [_vp, _i, _d, _d, _i, _dp, _dp, _lp]),
    "lgt_dd_hmc_trajectory": (_i, [_vp, _i, _d, _d, _i, C.c_ulonglong, C.c_uint, _dp, _ip, _lp, _dp]),
    "lgt_set_smearing": (_i, [_vp, _i, _d]),
    "lgt_get_smeared_links": (_i, [_vp, _vp]),
    "lgt_set_integrator": (_i, [_vp, _i, _i]),
    "lgt_momentum_heatbath": (_i, [_vp, C.c_ulonglong, C.c_uint]),
    "lgt_pseudofermion_heatbath": (_i, [_vp, C.c_ulonglong, C.c_uint, _dp]),
    "lgt_get_pseudofermion": (_i, [_vp, _vp]),
    "lgt_hmc_trajectory": (_i, [_vp, _i, _d, _d, _i, C.c_ulonglong, C.c_uint, _dp, _ip, _lp, _dp]),
    "lgt_plaquette_action_noalloc": (_i, [_ip, _d, _i, _i, _vp, _vp, _vp]),
    "lgt_noalloc_last_error": (C.c_char_p, []),
}

_lib = None


class LgtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lgt error %d: %s" % (code, msg))
        self.code = code


def lib():
    """Loads liblgt.so; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s not found: build it with `python -m paper_2602_20516_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array / int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return t.data_ptr()
    assert t.flags["C_CONTIGUOUS"]
    return t.ctypes.data


def _check(ctx, rc, allow=()):
    if rc != LGT_OK and rc not in allow:
        msg = lib().lgt_last_error(ctx)
        raise LgtError(rc, msg.decode() if msg else "")
    return rc


# ---- functions with the C names ---------------------------------------------------------------
def lgt_version():
    return lib().lgt_version().decode()


def lgt_create(dims, beta, kappa, bc, precision=LGT_F64, device=0, stream=None):
    h = _vp()
    d = (C.c_int * 4)(*[int(x) for x in dims])
    b = (C.c_int * 4)(*[int(x) for x in bc])
    rc = lib().lgt_create(C.byref(h), d, float(beta), float(kappa), b, int(precision), int(device), stream)
    if rc != LGT_OK:
        raise LgtError(rc, lib().lgt_last_error(None).decode())
    return h


def lgt_destroy(ctx):
    return lib().lgt_destroy(ctx)


def lgt_set_links(ctx, U):
    return _check(ctx, lib().lgt_set_links(ctx, _ptr(U)))


def lgt_get_links(ctx, U):
    return _check(ctx, lib().lgt_get_links(ctx, _ptr(U)))


def lgt_set_momenta(ctx, P):
    return _check(ctx, lib().lgt_set_momenta(ctx, _ptr(P)))


def lgt_get_momenta(ctx, P):
    return _check(ctx, lib().lgt_get_momenta(ctx, _ptr(P)))


def lgt_set_pseudofermion(ctx, phi):
    return _check(ctx, lib().lgt_set_pseudofermion(ctx, _ptr(phi)))


def lgt_set_links_host(ctx, U):
    return _check(ctx, lib().lgt_set_links_host(ctx, _ptr(U)))


def lgt_get_links_host(ctx, U):
    return _check(ctx, lib().lgt_get_links_host(ctx, _ptr(U)))


def lgt_set_momenta_host(ctx, P):
    return _check(ctx, lib().lgt_set_momenta_host(ctx, _ptr(P)))


def lgt_get_momenta_host(ctx, P):
    return _check(ctx, lib().lgt_get_momenta_host(ctx, _ptr(P)))


def lgt_set_pseudofermion_host(ctx, phi):
    return _check(ctx, lib().lgt_set_pseudofermion_host(ctx, _ptr(phi)))


def lgt_set_momenta_host_async(ctx, P):
    return _check(ctx, lib().lgt_set_momenta_host_async(ctx, _ptr(P)))


def lgt_get_links_host_async(ctx, U):
    return _check(ctx, lib().lgt_get_links_host_async(ctx, _ptr(U)))


def lgt_get_momenta_host_async(ctx, P):
    return _check(ctx, lib().lgt_get_momenta_host_async(ctx, _ptr(P)))


def lgt_host_transfers_wait(ctx):
    return _check(ctx, lib().lgt_host_transfers_wait(ctx))


def lgt_action(ctx, tol=1e-12, max_iter=100000):
    """Returns (S_g, S_F, K, cg_iters)."""
    sg, sf, k, it = C.c_double(), C.c_double(), C.c_double(), C.c_int()
    _check(ctx, lib().lgt_action(ctx, tol, max_iter, C.byref(sg), C.byref(sf), C.byref(k), C.byref(it)))
    return sg.value, sf.value, k.value, it.value


def lgt_plaquette(ctx):
    p = C.c_double()
    _check(ctx, lib().lgt_plaquette(ctx, C.byref(p)))
    return p.value


def lgt_noalloc_last_error():
    msg = lib().lgt_noalloc_last_error()
    return msg.decode() if msg else ""


def lgt_plaquette_action_noalloc(dims, beta, U, out, precision=LGT_F64, device=0, stream=None):
    """Enqueues the plaquette action of the caller's canonical device links U; `out` (device, two doubles) receives
    (S_g, average plaquette).  No allocation, no synchronisation; calls that overlap on the GPU race on the shared scratch."""
    d = (C.c_int * 4)(*[int(x) for x in dims])
    rc = lib().lgt_plaquette_action_noalloc(d, float(beta), int(precision), int(device), _ptr(U), _ptr(out), stream)
    if rc != LGT_OK:
        raise LgtError(rc, lgt_noalloc_last_error())
    return rc


def lgt_dslash(ctx, inp, out, dagger=False):
    return _check(ctx, lib().lgt_dslash(ctx, _ptr(inp), _ptr(out), int(bool(dagger))))


def lgt_cg(ctx, b, x, tol, max_iter):
    """Returns (iters, rel_resid, converged)."""
    it, rel = C.c_int(), C.c_double()
    rc = _check(ctx, lib().lgt_cg(ctx, _ptr(b), _ptr(x), tol, max_iter, C.byref(it), C.byref(rel)), allow=(LGT_ENOCONV,))
    return it.value, rel.value, rc == LGT_OK


def lgt_cg_mixed(ctx, b, x, tol, max_iter, inner_tol=1e-5):
    """Mixed-precision defect-correction CG.  Returns (inner_iters, outer_cycles, true_rel_resid, converged)."""
    it, outer, rel = C.c_int(), C.c_int(), C.c_double()
    rc = _check(ctx, lib().lgt_cg_mixed(ctx, _ptr(b), _ptr(x), tol, max_iter, inner_tol, C.byref(it), C.byref(outer),
                                        C.byref(rel)), allow=(LGT_ENOCONV,))
    return it.value, outer.value, rel.value, rc == LGT_OK


def lgt_eo_mhat(ctx, src, dst, dagger=False):
    return _check(ctx, lib().lgt_eo_mhat(ctx, _ptr(src), _ptr(dst), int(bool(dagger))))


def lgt_eo_cg(ctx, b, x, tol, max_iter):
    """CG on M^dag M (even sites).  Returns (iters, rel_resid, converged)."""
    it, rel = C.c_int(), C.c_double()
    rc = _check(ctx, lib().lgt_eo_cg(ctx, _ptr(b), _ptr(x), tol, max_iter, C.byref(it), C.byref(rel)), allow=(LGT_ENOCONV,))
    return it.value, rel.value, rc == LGT_OK


def lgt_set_fermion_action(ctx, action):
    return _check(ctx, lib().lgt_set_fermion_action(ctx, int(action)))


def lgt_set_solver(ctx, solver, inner_tol=1e-5):
    return _check(ctx, lib().lgt_set_solver(ctx, int(solver), float(inner_tol)))


def lgt_gauge_force(ctx, F):
    return _check(ctx, lib().lgt_gauge_force(ctx, _ptr(F)))


def lgt_fermion_force(ctx, X, Y, F, tol=1e-12, max_iter=100000):
    """X, Y None: solved from the handle's pseudofermion.  Returns cg_iters."""
    it = C.c_int()
    _check(ctx, lib().lgt_fermion_force(ctx, _ptr(X), _ptr(Y), _ptr(F), tol, max_iter, C.byref(it)))
    return it.value


def lgt_md_kick(ctx, eps, tol=1e-12, max_iter=100000):
    it = C.c_int()
    _check(ctx, lib().lgt_md_kick(ctx, eps, tol, max_iter, C.byref(it)))
    return it.value


def lgt_md_drift(ctx, eps):
    return _check(ctx, lib().lgt_md_drift(ctx, eps))


def lgt_md_step(ctx, dt, tol=1e-12, max_iter=100000):
    it = C.c_int()
    _check(ctx, lib().lgt_md_step(ctx, dt, tol, max_iter, C.byref(it)))
    return it.value


def lgt_md_trajectory(ctx, nsteps, dt, tol=1e-12, max_iter=100000, measure=True):
    """Returns (H_initial, H_final, cg_iters)."""
    h0, h1, its = C.c_double(), C.c_double(), C.c_long()
    _check(ctx, lib().lgt_md_trajectory(ctx, nsteps, dt, tol, max_iter,
                                        C.byref(h0) if measure else None, C.byref(h1) if measure else None,
                                        C.byref(its)))
    return h0.value, h1.value, its.value


def lgt_set_smearing(ctx, n_levels, rho=0.0):
    _check(ctx, lib().lgt_set_smearing(ctx, n_levels, rho))


def lgt_get_smeared_links(ctx, U):
    _check(ctx, lib().lgt_get_smeared_links(ctx, _ptr(U)))


def lgt_set_integrator(ctx, integrator, n_inner=1):
    _check(ctx, lib().lgt_set_integrator(ctx, integrator, n_inner))


def lgt_momentum_heatbath(ctx, seed, trajectory):
    _check(ctx, lib().lgt_momentum_heatbath(ctx, seed, trajectory))


def lgt_pseudofermion_heatbath(ctx, seed, trajectory):
    """Returns |eta|^2 (= S_F at the start of the trajectory)."""
    n2 = C.c_double()
    _check(ctx, lib().lgt_pseudofermion_heatbath(ctx, seed, trajectory, C.byref(n2)))
    return n2.value


def lgt_get_pseudofermion(ctx, phi):
    _check(ctx, lib().lgt_get_pseudofermion(ctx, _ptr(phi)))


def lgt_hmc_trajectory(ctx, nsteps, dt, seed, trajectory, tol=1e-12, max_iter=100000):
    """Returns (dH, accepted, cg_iters, H_initial, converged)."""
    dH, acc, its, H0 = C.c_double(), C.c_int(), C.c_long(), C.c_double()
    rc = _check(ctx, lib().lgt_hmc_trajectory(ctx, nsteps, dt, tol, max_iter, seed, trajectory, C.byref(dH), C.byref(acc),
                                              C.byref(its), C.byref(H0)), allow=(LGT_ENOCONV,))
    return dH.value, bool(acc.value), its.value, H0.value, rc == LGT_OK


def lgt_native_spinor_bytes(ctx):
    return lib().lgt_native_spinor_bytes(ctx)


def lgt_spinor_to_native(ctx, canonical, native):
    return _check(ctx, lib().lgt_spinor_to_native(ctx, _ptr(canonical), _ptr(native)))


def lgt_spinor_from_native(ctx, native, canonical):
    return _check(ctx, lib().lgt_spinor_from_native(ctx, _ptr(native), _ptr(canonical)))


def lgt_dslash_native(ctx, inp, out, dagger=False):
    return _check(ctx, lib().lgt_dslash_native(ctx, _ptr(inp), _ptr(out), int(bool(dagger))))


def lgt_fermion_force_native(ctx, X, Y, eps):
    return _check(ctx, lib().lgt_fermion_force_native(ctx, _ptr(X), _ptr(Y), eps))


def lgt_gauge_force_accumulate(ctx, eps):
    return _check(ctx, lib().lgt_gauge_force_accumulate(ctx, eps))


def lgt_cg_native(ctx, b, x, y, tol, max_iter):
    it, rel = C.c_int(), C.c_double()
    rc = _check(ctx, lib().lgt_cg_native(ctx, _ptr(b), _ptr(x), _ptr(y), tol, max_iter, C.byref(it), C.byref(rel)),
                allow=(LGT_ENOCONV,))
    return it.value, rel.value, rc == LGT_OK


(LGT_K_DSLASH, LGT_K_CG_BLAS, LGT_K_FERMION_FORCE, LGT_K_GAUGE_FORCE, LGT_K_LINK_UPDATE, LGT_K_OTHER,
 LGT_K_DSLASH_R, LGT_K_CG_UPDATE) = range(8)
KERNEL_CLASSES = ("dslash", "cg_scalars", "fermion_force", "gauge_force", "link_update", "other", "dslash_dag_fused_r", "cg_update_xp")


def lgt_measure_peaks(ctx, launches=10, fma=True, copy=True):
    """Returns {"fma_tflops_best", "fma_tflops_mean", "copy_gbs_best", "copy_gbs_mean"} (None where not measured)."""
    v = [C.c_double() for _ in range(4)]
    _check(ctx, lib().lgt_measure_peaks(ctx, launches, C.byref(v[0]) if fma else None, C.byref(v[1]) if fma else None,
                                        C.byref(v[2]) if copy else None, C.byref(v[3]) if copy else None))
    keys = ("fma_tflops_best", "fma_tflops_mean", "copy_gbs_best", "copy_gbs_mean")
    return {k: (x.value if (fma if i < 2 else copy) else None) for i, (k, x) in enumerate(zip(keys, v))}


def lgt_timing_enable(ctx, enable=True):
    return _check(ctx, lib().lgt_timing_enable(ctx, int(bool(enable))))


def lgt_timing_reset(ctx):
    return _check(ctx, lib().lgt_timing_reset(ctx))


def lgt_timing_read(ctx, kernel_class):
    """Returns (ms_total, launches) of one kernel class since the last reset."""
    ms, n = C.c_double(), C.c_long()
    _check(ctx, lib().lgt_timing_read(ctx, int(kernel_class), C.byref(ms), C.byref(n)))
    return ms.value, n.value


def lgt_stream(ctx):
    return lib().lgt_stream(ctx)


def lgt_last_error(ctx):
    msg = lib().lgt_last_error(ctx)
    return msg.decode() if msg else ""


def lgt_launch_count(ctx):
    return lib().lgt_launch_count(ctx)


def lgt_set_block_swizzle(ctx, z_planes=-1):
    """Block traversal order of the Dslash kernels (0 lexicographic, Z > 0 slabs of Z z-planes, < 0 automatic).
    Returns the value in effect."""
    out = C.c_int(0)
    _check(ctx, lib().lgt_set_block_swizzle(ctx, int(z_planes), C.byref(out)))
    return out.value


def lgt_set_kernel_variant(ctx, kernel_class, variant=-1):
    """Implementation variant of one kernel class (variant < 0 only queries).  Returns the value in effect."""
    out = C.c_int(0)
    _check(ctx, lib().lgt_set_kernel_variant(ctx, int(kernel_class), int(variant), C.byref(out)))
    return out.value


# ---- decomposed lattice (lgt_dd_*) -----------------------------------------------------------------
def _dd_check(d, rc, allow=()):
    if rc != LGT_OK and rc not in allow:
        msg = lib().lgt_dd_last_error(d)
        raise LgtError(rc, msg.decode() if msg else "")
    return rc


def _ptr_array(items):
    return (_vp * len(items))(*[_ptr(t) for t in items])


def lgt_dd_create(dims, nranks, local_ranks, beta, kappa, bc, precision=LGT_F64, device=0, stream=None):
    h = _vp()
    d4 = (C.c_int * 4)(*[int(x) for x in dims])
    b4 = (C.c_int * 4)(*[int(x) for x in bc])
    lr = (C.c_int * len(local_ranks))(*[int(r) for r in local_ranks])
    rc = lib().lgt_dd_create(C.byref(h), d4, nranks, len(local_ranks), lr, beta, kappa, b4, precision, device, stream)
    _dd_check(None, rc)
    return h


def lgt_dd_create_grid(dims, grid, local_ranks, beta, kappa, bc, precision=LGT_F64, device=0, stream=None):
    """Two split directions: grid = (Pt, Pz), rank = pt * Pz + pz."""
    h = _vp()
    d4 = (C.c_int * 4)(*[int(x) for x in dims])
    g2 = (C.c_int * 2)(*[int(x) for x in grid])
    b4 = (C.c_int * 4)(*[int(x) for x in bc])
    lr = (C.c_int * len(local_ranks))(*[int(r) for r in local_ranks])
    rc = lib().lgt_dd_create_grid(C.byref(h), d4, g2, len(local_ranks), lr, beta, kappa, b4, precision, device, stream)
    _dd_check(None, rc)
    return h


def lgt_dd_destroy(d):
    lib().lgt_dd_destroy(d)
    _host_transports.pop(getattr(d, "value", None), None)


def lgt_dd_last_error(d):
    msg = lib().lgt_dd_last_error(d)
    return msg.decode() if msg else ""


def lgt_dd_nccl_unique_id():
    """128 bytes (rank 0 calls this, everybody receives them by a broadcast)."""
    buf = C.create_string_buffer(128)
    _dd_check(None, lib().lgt_dd_nccl_unique_id(buf))
    return bytes(buf.raw)


def lgt_dd_nccl_init(d, id128):
    _dd_check(d, lib().lgt_dd_nccl_init(d, C.c_char_p(bytes(id128))))


SENDRECV_FN = C.CFUNCTYPE(_i, _vp, C.POINTER(_vp), _ip, C.POINTER(_vp), _ip, C.c_size_t)
ALLREDUCE_FN = C.CFUNCTYPE(_i, _vp, _dp, _i)
_host_transports = {}  # group address -> the ctypes callback objects (they must outlive the group)


def lgt_dd_halo_plan(nranks, rank, lt_local):
    """Host-only.  Returns (send_peer, send_slice, recv_peer, recv_slice), two entries each, in issue order."""
    plan = (C.c_int * 8)()
    rc = lib().lgt_dd_halo_plan(nranks, rank, lt_local, plan)
    if rc != LGT_OK:
        raise LgtError(rc, "lgt_dd_halo_plan: bad arguments")
    v = list(plan)
    return v[0:2], v[2:4], v[4:6], v[6:8]


def lgt_dd_set_host_transport(d, sendrecv, allreduce):
    """sendrecv(send_bufs, send_peers, recv_bufs, recv_peers): two numpy uint8 views each way over the library's pinned
    staging memory; allreduce(buf): numpy float64 view, summed over the ranks in place.  Exceptions become error codes."""
    import numpy as np

    def view(addr, n, ctype, dtype):
        return np.frombuffer((ctype * n).from_address(addr), dtype=dtype)

    def c_sendrecv(user, sb, sp, rb, rp, nbytes):
        try:
            sendrecv([view(sb[k], nbytes, C.c_ubyte, np.uint8) for k in range(2)], [sp[0], sp[1]],
                     [view(rb[k], nbytes, C.c_ubyte, np.uint8) for k in range(2)], [rp[0], rp[1]])
            return 0
        except Exception:  # never unwind through the C frames
            import traceback

            traceback.print_exc()
            return 1

    def c_allreduce(user, buf, count):
        try:
            allreduce(view(C.addressof(buf.contents), count, C.c_double, np.float64))
            return 0
        except Exception:
            import traceback

            traceback.print_exc()
            return 1

    fns = (SENDRECV_FN(c_sendrecv), ALLREDUCE_FN(c_allreduce))
    _dd_check(d, lib().lgt_dd_set_host_transport(d, C.cast(fns[0], _vp), C.cast(fns[1], _vp), None))
    _host_transports[d.value] = fns


def lgt_dd_set_halo_mode(d, mode):
    _dd_check(d, lib().lgt_dd_set_halo_mode(d, mode))


def lgt_dd_ipc_export(d):
    """128 bytes: the CUDA IPC handles of this rank's r and t fields."""
    buf = C.create_string_buffer(128)
    _dd_check(d, lib().lgt_dd_ipc_export(d, buf))
    return bytes(buf.raw)


def lgt_dd_ipc_import(d, lo_handles, hi_handles):
    _dd_check(d, lib().lgt_dd_ipc_import(d, C.c_char_p(bytes(lo_handles)), C.c_char_p(bytes(hi_handles))))


def lgt_dd_local_ranks(d):
    return lib().lgt_dd_local_ranks(d)


def lgt_dd_rank(d, local_index):
    h = lib().lgt_dd_rank(d, local_index)
    if not h:
        raise LgtError(LGT_EINVAL, "lgt_dd_rank: bad local index")
    return _vp(h)


def lgt_dd_dslash(d, ins, outs, dagger=False):
    _dd_check(d, lib().lgt_dd_dslash(d, _ptr_array(ins), _ptr_array(outs), int(bool(dagger))))


def lgt_dd_cg(d, bs, xs, tol, max_iter):
    """Returns (iters, rel_resid, converged)."""
    it, rel = C.c_int(), C.c_double()
    rc = _dd_check(d, lib().lgt_dd_cg(d, _ptr_array(bs), _ptr_array(xs), tol, max_iter, C.byref(it), C.byref(rel)), allow=(LGT_ENOCONV,))
    return it.value, rel.value, rc == LGT_OK


def lgt_dd_action(d, tol=1e-12, max_iter=100000):
    """Returns (S_g, S_F, K, cg_iters), global values."""
    sg, sf, k, it = C.c_double(), C.c_double(), C.c_double(), C.c_int()
    _dd_check(d, lib().lgt_dd_action(d, tol, max_iter, C.byref(sg), C.byref(sf), C.byref(k), C.byref(it)))
    return sg.value, sf.value, k.value, it.value


def lgt_dd_set_solver(d, solver, inner_tol=1e-5):
    _dd_check(d, lib().lgt_dd_set_solver(d, solver, inner_tol))


def lgt_dd_set_integrator(d, integrator, n_inner=1):
    _dd_check(d, lib().lgt_dd_set_integrator(d, integrator, n_inner))


def lgt_dd_set_smearing(d, n_levels, rho=0.0):
    _dd_check(d, lib().lgt_dd_set_smearing(d, n_levels, rho))


def lgt_dd_set_fermion_action(d, action):
    _dd_check(d, lib().lgt_dd_set_fermion_action(d, action))


def lgt_dd_md_kick(d, eps, tol=1e-12, max_iter=100000):
    it = C.c_int()
    _dd_check(d, lib().lgt_dd_md_kick(d, eps, tol, max_iter, C.byref(it)))
    return it.value


def lgt_dd_md_drift(d, eps):
    _dd_check(d, lib().lgt_dd_md_drift(d, eps))


def lgt_dd_md_trajectory(d, nsteps, dt, tol=1e-12, max_iter=100000, measure=True):
    """Returns (H_initial, H_final, cg_iters)."""
    h0, h1, its = C.c_double(), C.c_double(), C.c_long()
    _dd_check(d, lib().lgt_dd_md_trajectory(d, nsteps, dt, tol, max_iter, C.byref(h0) if measure else None,
                                            C.byref(h1) if measure else None, C.byref(its)))
    return h0.value, h1.value, its.value


def lgt_dd_hmc_trajectory(d, nsteps, dt, seed, trajectory, tol=1e-12, max_iter=100000):
    """Returns (dH, accepted, cg_iters, H_initial, converged)."""
    dH, acc, its, H0 = C.c_double(), C.c_int(), C.c_long(), C.c_double()
    rc = _dd_check(d, lib().lgt_dd_hmc_trajectory(d, nsteps, dt, tol, max_iter, seed, trajectory, C.byref(dH), C.byref(acc),
                                                  C.byref(its), C.byref(H0)), allow=(LGT_ENOCONV,))
    return dH.value, bool(acc.value), its.value, H0.value, rc == LGT_OK


# ---- convenience wrapper -----------------------------------------------------------------------
class Lattice:
    """A handle plus torch buffers in the canonical layout.  numpy in / numpy out helpers for tests."""

    def __init__(self, dims, beta, kappa, bc, precision=LGT_F64, device=0, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2602_20516_b200 needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.V = 1
        for d in self.dims:
            self.V *= d
        self.precision = precision
        self.cdtype = torch.complex128 if precision == LGT_F64 else torch.complex64
        self.device = torch.device("cuda", device)
        self.ctx = lgt_create(dims, beta, kappa, bc, precision, device, stream)

    def close(self):
        if self.ctx is not None:
            lgt_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # device tensors
    def empty(self, *shape):
        return self.torch.empty(shape, dtype=self.cdtype, device=self.device)

    def to_device(self, a):
        return self.torch.from_numpy(a).to(self.cdtype).to(self.device).contiguous()

    def native_spinor(self):
        return self.torch.empty(lgt_native_spinor_bytes(self.ctx), dtype=self.torch.uint8, device=self.device)

    # numpy helpers (upload, call, download)
    def set_links(self, U):
        lgt_set_links(self.ctx, self.to_device(U))

    def get_links(self):
        out = self.empty(self.V, 4, 3, 3)
        lgt_get_links(self.ctx, out)
        return out.cpu().numpy()

    def set_momenta(self, P):
        lgt_set_momenta(self.ctx, self.to_device(P))

    def get_momenta(self):
        out = self.empty(self.V, 4, 3, 3)
        lgt_get_momenta(self.ctx, out)
        return out.cpu().numpy()

    def set_pseudofermion(self, phi):
        lgt_set_pseudofermion(self.ctx, self.to_device(phi))

    def dslash(self, psi, dagger=False):
        out = self.empty(self.V, 4, 3)
        lgt_dslash(self.ctx, self.to_device(psi), out, dagger)
        return out.cpu().numpy()

    def cg(self, b, tol, max_iter):
        x = self.empty(self.V, 4, 3)
        it, rel, ok = lgt_cg(self.ctx, self.to_device(b), x, tol, max_iter)
        return x.cpu().numpy(), it, rel, ok

    def eo_mhat(self, psi, dagger=False):
        out = self.empty(self.V, 4, 3)
        lgt_eo_mhat(self.ctx, self.to_device(psi), out, dagger)
        return out.cpu().numpy()

    def eo_cg(self, b, tol, max_iter):
        x = self.empty(self.V, 4, 3)
        it, rel, ok = lgt_eo_cg(self.ctx, self.to_device(b), x, tol, max_iter)
        return x.cpu().numpy(), it, rel, ok

    def cg_mixed(self, b, tol, max_iter, inner_tol=1e-5):
        x = self.empty(self.V, 4, 3)
        it, outer, rel, ok = lgt_cg_mixed(self.ctx, self.to_device(b), x, tol, max_iter, inner_tol)
        return x.cpu().numpy(), it, outer, rel, ok

    def gauge_force(self):
        F = self.empty(self.V, 4, 3, 3)
        lgt_gauge_force(self.ctx, F)
        return F.cpu().numpy()

    def fermion_force(self, X=None, Y=None, tol=1e-12, max_iter=100000):
        F = self.empty(self.V, 4, 3, 3)
        it = lgt_fermion_force(self.ctx, None if X is None else self.to_device(X),
                               None if Y is None else self.to_device(Y), F, tol, max_iter)
        return F.cpu().numpy(), it


class DecomposedLattice:
    """A group of time slabs (lgt_dd_*) with numpy in / numpy out helpers.  `local_ranks` = all ranks: the
    single-device verification mode; one rank: the production mode (call nccl_init with the broadcast id)."""

    def __init__(self, dims, nranks, local_ranks, beta, kappa, bc, precision=LGT_F64, device=0, stream=None, grid=None):
        """nranks time slabs, or with grid = (Pt, Pz) a two-direction decomposition (nranks is then Pt * Pz)."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2602_20516_b200 needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.nranks, self.local_ranks = int(nranks), [int(r) for r in local_ranks]
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self.Vloc = self.V // self.nranks
        self.cdtype = torch.complex128 if precision == LGT_F64 else torch.complex64
        self.device = torch.device("cuda", device)
        self.grid = None if grid is None else (int(grid[0]), int(grid[1]))
        if self.grid is None:
            self.d = lgt_dd_create(dims, nranks, local_ranks, beta, kappa, bc, precision, device, stream)
        else:
            if self.grid[0] * self.grid[1] != self.nranks:
                raise ValueError("nranks must be Pt * Pz")
            self.d = lgt_dd_create_grid(dims, self.grid, local_ranks, beta, kappa, bc, precision, device, stream)
        self.ranks = [lgt_dd_rank(self.d, i) for i in range(len(self.local_ranks))]

    def close(self):
        if self.d is not None:
            lgt_dd_destroy(self.d)
            self.d = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def slab(self, a, rank):
        """Rows of a global canonical array [V, ...] that belong to `rank`: a run of time slices (t is the slowest index),
        or on a grid the block [Lt/Pt][Lz/Pz][Ly][Lx] of rank = pt * Pz + pz, flattened in lexicographic order."""
        if self.grid is None:
            return a[rank * self.Vloc:(rank + 1) * self.Vloc]
        from .dist import grid_block

        return grid_block(a, self.dims, self.grid, rank)

    def _up(self, a, rank):
        import numpy as np

        return self.torch.from_numpy(np.ascontiguousarray(self.slab(a, rank))).to(self.cdtype).to(self.device).contiguous()

    def _scatter(self, a, setter):
        for i, r in enumerate(self.local_ranks):
            setter(self.ranks[i], self._up(a, r))

    def _gather(self, getter, *shape):
        """Local slabs as a list of numpy arrays in local-rank order."""
        out = []
        for i in range(len(self.local_ranks)):
            t = self.torch.empty((self.Vloc,) + shape, dtype=self.cdtype, device=self.device)
            getter(self.ranks[i], t)
            out.append(t.cpu().numpy())
        return out

    def set_links(self, U):
        self._scatter(U, lgt_set_links)

    def set_momenta(self, P):
        self._scatter(P, lgt_set_momenta)

    def set_pseudofermion(self, phi):
        self._scatter(phi, lgt_set_pseudofermion)

    def get_links(self):
        return self._gather(lgt_get_links, 4, 3, 3)

    def get_momenta(self):
        return self._gather(lgt_get_momenta, 4, 3, 3)

    def dslash(self, psi, dagger=False):
        ins = [self._up(psi, r) for r in self.local_ranks]
        outs = [self.torch.empty_like(t) for t in ins]
        lgt_dd_dslash(self.d, ins, outs, dagger)
        return [t.cpu().numpy() for t in outs]

    def cg(self, b, tol, max_iter):
        bs = [self._up(b, r) for r in self.local_ranks]
        xs = [self.torch.empty_like(t) for t in bs]
        it, rel, ok = lgt_dd_cg(self.d, bs, xs, tol, max_iter)
        return [t.cpu().numpy() for t in xs], it, rel, ok
