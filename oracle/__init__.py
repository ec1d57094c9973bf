"""CPU oracle for the HMC force hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with paper_2602_20516_b200.

Thin ctypes/numpy marshalling over oracle/liblgt_oracle.so (lgt_oracle.cpp); all
arithmetic lives in the C++ file.  Arrays are complex128, canonical layout:
links U[V,4,3,3], spinors psi[V,4,3], momenta/forces P[V,4,3,3], site index
s = x + Lx*(y + Ly*(z + Lz*t)).
"""
import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.lgto_redot.restype = C.c_double
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _dims(dims):
    d = (C.c_int * 4)(*[int(x) for x in dims])
    V = int(np.prod([int(x) for x in dims]))
    return d, V


def _bc(bc):
    return (C.c_int * 4)(*[int(x) for x in bc])


def gamma(mu):
    out = np.empty((4, 4), np.complex128)
    lib().lgto_gamma(C.c_int(mu), _p(out))
    return out


def generator(a):
    out = np.empty((3, 3), np.complex128)
    lib().lgto_generator(C.c_int(a), _p(out))
    return out


def ta(M):
    M = _c(M, (3, 3))
    out = np.empty((3, 3), np.complex128)
    lib().lgto_ta(_p(M), _p(out))
    return out


def expm(A):
    A = _c(A, (3, 3))
    out = np.empty((3, 3), np.complex128)
    lib().lgto_expm(_p(A), _p(out))
    return out


def gauge_action(dims, beta, U):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    S, plaq = C.c_double(), C.c_double()
    lib().lgto_gauge_action(d, C.c_double(beta), _p(U), C.byref(S), C.byref(plaq))
    return S.value, plaq.value


def dslash(dims, kappa, bc, U, psi, dagger=False):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    psi = _c(psi, (V, 4, 3))
    out = np.empty_like(psi)
    lib().lgto_dslash(d, C.c_double(kappa), _bc(bc), _p(U), _p(psi), _p(out), C.c_int(int(dagger)))
    return out


def dslash_sites(dims, kappa, bc, U, psi, sites, dagger=False):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    psi = _c(psi, (V, 4, 3))
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites), 4, 3), np.complex128)
    lib().lgto_dslash_sites(d, C.c_double(kappa), _bc(bc), _p(U), _p(psi), C.c_int(int(dagger)),
                            _p(sites), C.c_long(len(sites)), _p(out))
    return out


def cg(dims, kappa, bc, U, b, tol, max_iter):
    """Returns (x, iters, rel_resid, converged)."""
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    b = _c(b, (V, 4, 3))
    x = np.empty_like(b)
    it, rel = C.c_int(), C.c_double()
    rc = lib().lgto_cg(d, C.c_double(kappa), _bc(bc), _p(U), _p(b), _p(x), C.c_double(tol),
                       C.c_int(max_iter), C.byref(it), C.byref(rel))
    return x, it.value, rel.value, rc == 0


def gauge_force(dims, beta, U):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    F = np.empty_like(U)
    lib().lgto_gauge_force(d, C.c_double(beta), _p(U), _p(F))
    return F


def gauge_force_link(dims, beta, U, s, mu):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    F = np.empty((3, 3), np.complex128)
    lib().lgto_gauge_force_link(d, C.c_double(beta), _p(U), C.c_long(s), C.c_int(mu), _p(F))
    return F


def fermion_force(dims, kappa, bc, U, X, Y):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    X = _c(X, (V, 4, 3))
    Y = _c(Y, (V, 4, 3))
    F = np.empty_like(U)
    lib().lgto_fermion_force(d, C.c_double(kappa), _bc(bc), _p(U), _p(X), _p(Y), _p(F))
    return F


def fermion_force_link(dims, kappa, bc, U, X, Y, s, mu):
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    X = _c(X, (V, 4, 3))
    Y = _c(Y, (V, 4, 3))
    F = np.empty((3, 3), np.complex128)
    lib().lgto_fermion_force_link(d, C.c_double(kappa), _bc(bc), _p(U), _p(X), _p(Y),
                                  C.c_long(s), C.c_int(mu), _p(F))
    return F


def kinetic(dims, P):
    d, V = _dims(dims)
    P = _c(P, (V, 4, 3, 3))
    K = C.c_double()
    lib().lgto_kinetic(d, _p(P), C.byref(K))
    return K.value


def redot(a, b):
    a = _c(a)
    b = _c(b, a.shape)
    return lib().lgto_redot(C.c_long(a.size), _p(a), _p(b))


def fermion_action(dims, kappa, bc, U, phi, tol, max_iter):
    """Returns (S_F, X, iters, converged)."""
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    phi = _c(phi, (V, 4, 3))
    X = np.empty_like(phi)
    S, it = C.c_double(), C.c_int()
    rc = lib().lgto_fermion_action(d, C.c_double(kappa), _bc(bc), _p(U), _p(phi), C.c_double(tol),
                                   C.c_int(max_iter), C.byref(S), _p(X), C.byref(it))
    return S.value, X, it.value, rc == 0


def drift(dims, eps, P, U):
    """Returns the updated links; inputs untouched."""
    d, V = _dims(dims)
    P = _c(P, (V, 4, 3, 3))
    U = _c(U, (V, 4, 3, 3)).copy()
    lib().lgto_drift(d, C.c_double(eps), _p(P), _p(U))
    return U


def kick(dims, beta, kappa, bc, U, phi, P, eps, tol=1e-12, max_iter=100000):
    """Returns (P_new, cg_iters, converged)."""
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3))
    P = _c(P, (V, 4, 3, 3)).copy()
    it = C.c_int()
    if phi is not None:
        phi = _c(phi, (V, 4, 3))
    rc = lib().lgto_kick(d, C.c_double(beta), C.c_double(kappa), _bc(bc), _p(U),
                         _p(phi) if phi is not None else None, _p(P), C.c_double(eps),
                         C.c_double(tol), C.c_int(max_iter), C.byref(it))
    return P, it.value, rc == 0


def trajectory(dims, beta, kappa, bc, U, phi, P, nsteps, dt, tol=1e-12, max_iter=100000):
    """Returns (U_new, P_new, total_cg_iters, converged)."""
    d, V = _dims(dims)
    U = _c(U, (V, 4, 3, 3)).copy()
    P = _c(P, (V, 4, 3, 3)).copy()
    if phi is not None:
        phi = _c(phi, (V, 4, 3))
    its = C.c_long()
    rc = lib().lgto_trajectory(d, C.c_double(beta), C.c_double(kappa), _bc(bc), _p(U),
                               _p(phi) if phi is not None else None, _p(P), C.c_int(nsteps),
                               C.c_double(dt), C.c_double(tol), C.c_int(max_iter), C.byref(its))
    return U, P, its.value, rc == 0


def hamiltonian(dims, beta, kappa, bc, U, phi, P, tol=1e-12, max_iter=100000):
    """H = K + S_g + S_F; returns (H, K, S_g, S_F)."""
    K = kinetic(dims, P)
    S_g, _ = gauge_action(dims, beta, U)
    S_F = 0.0
    if phi is not None and kappa != 0.0:
        S_F = fermion_action(dims, kappa, bc, U, phi, tol, max_iter)[0]
    return K + S_g + S_F, K, S_g, S_F


def num_threads():
    return lib().lgto_num_threads()


def set_num_threads(n):
    lib().lgto_set_num_threads(C.c_int(int(n)))
