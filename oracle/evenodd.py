"""CPU oracle for the even/odd (Schur) preconditioned pseudofermion action -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

SURVEY.md 8(f)1.  Only tests/ may import this module.  It shares no code with paper_2602_20516_b200: everything
here is the plain definition written with the pinned oracle operator `oracle.dslash` (D and D^dag of
BASELINE.json configs[0]) and numpy masks.

Definitions.  Sites are split by parity p(x) = (x+y+z+t) mod 2 (every extent even, so that parity survives the
periodic wrap).  With D = 1 - kappa H and H only connecting sites of opposite parity,

    D = [[1, -kappa H_eo], [-kappa H_oe, 1]],     M = 1 - kappa^2 H_eo H_oe  (Schur complement on the even sites),

det D = det M, and the two-flavour determinant det(D^dag D) of PAPER.md:377 (S3.1) is also represented by

    S_F^eo = phi_e^dag (M^dag M)^-1 phi_e.

Its variation follows S3.12 with D -> M: dS = -2 Re[Y_e^dag (dM) X_e], X_e = (M^dag M)^-1 phi_e,
Y_e = M X_e, dM = -kappa^2 (dH_eo H_oe + H_eo dH_oe).  Setting X_o = kappa H_oe X_e and Y_o = kappa (H_eo)^dag Y_e
turns this into -2 Re[Y^dag (dD) X] over the FULL lattice with dD = -kappa dH, i.e. the full-lattice force
formula evaluated on X = (X_e, X_o), Y = (Y_e, Y_o): `oracle.fermion_force(X, Y)`.

Pins (tests/test_oracle_eo_pins.py): M against the dense Schur complement of the dense D and det D = det M on a
2^4 lattice; M^dag against the conjugate transpose; the force against Richardson central differences of S_F^eo;
phi_e = M^dag eta_e  =>  S_F^eo = |eta_e|^2, Y_e = eta_e.
"""
import numpy as np

import oracle


def parity(dims):
    """p(s) = (x+y+z+t) mod 2 for every site of the canonical order s = x + Lx*(y + Ly*(z + Lz*t))."""
    Lx, Ly, Lz, Lt = [int(d) for d in dims]
    if any(d % 2 for d in (Lx, Ly, Lz, Lt)):
        raise ValueError("even/odd fields need every extent even")
    s = np.arange(Lx * Ly * Lz * Lt)
    return ((s % Lx) + (s // Lx) % Ly + (s // (Lx * Ly)) % Lz + s // (Lx * Ly * Lz)) % 2


def keep(psi, dims, p):
    """Copy of the spinor field with the sites of parity 1 - p set to zero."""
    out = np.array(psi, dtype=np.complex128, copy=True)
    out[parity(dims) != p] = 0.0
    return out


def mhat(dims, kappa, bc, U, x, dagger=False):
    """M x_e (dagger: M^dag x_e) on the even sites; odd sites of x are ignored, odd sites of the result are zero.

    D (x_e, 0) = (x_e, -kappa H_oe x_e) =: (x_e, y_o);  D (0, y_o) = (-kappa H_eo y_o, y_o) = (kappa^2 H_eo H_oe x_e, y_o);
    hence M x_e = x_e - [D (0, y_o)]_e.  D^dag has the same block structure with H -> H^dag."""
    xe = keep(x, dims, 0)
    yo = keep(oracle.dslash(dims, kappa, bc, U, xe, dagger=dagger), dims, 1)
    return xe - keep(oracle.dslash(dims, kappa, bc, U, yo, dagger=dagger), dims, 0)


def cg(dims, kappa, bc, U, b, tol, max_iter):
    """Textbook CG on A = M^dag M over the even sites, x0 = 0, the recurrence and stop rule of DESIGN.md reading A-10
    (stop on the recurrence residual, iters = applications of A).  Returns (x_e, iters, rel_resid, converged)."""
    be = keep(b, dims, 0)
    x = np.zeros_like(be)
    r = be.copy()
    p = be.copy()
    rr = oracle.redot(r, r)
    bb = rr
    k = 0
    if bb == 0.0:
        return x, 0, 0.0, True
    while rr > tol * tol * bb and k < max_iter:
        u = mhat(dims, kappa, bc, U, p)
        q = mhat(dims, kappa, bc, U, u, dagger=True)
        alpha = rr / oracle.redot(p, q)
        x += alpha * p
        r -= alpha * q
        rr_new = oracle.redot(r, r)
        p = r + (rr_new / rr) * p
        rr = rr_new
        k += 1
    return x, k, float(np.sqrt(rr / bb)), not (rr > tol * tol * bb)


def solve_xy(dims, kappa, bc, U, phi, tol, max_iter):
    """X = (X_e, kappa H_oe X_e), Y = (Y_e, kappa H_oe^dag Y_e) with X_e = (M^dag M)^-1 phi_e, Y_e = M X_e.
    kappa H_oe x_e = -[D (x_e, 0)]_o and kappa (H^dag)_oe y_e = -[D^dag (y_e, 0)]_o.  Returns (X, Y, iters, converged)."""
    Xe, it, _, ok = cg(dims, kappa, bc, U, phi, tol, max_iter)
    Ye = mhat(dims, kappa, bc, U, Xe)
    Xo = -keep(oracle.dslash(dims, kappa, bc, U, Xe), dims, 1)
    Yo = -keep(oracle.dslash(dims, kappa, bc, U, Ye, dagger=True), dims, 1)
    return Xe + Xo, Ye + Yo, it, ok


def action(dims, kappa, bc, U, phi, tol, max_iter):
    """S_F^eo = Re phi_e^dag (M^dag M)^-1 phi_e.  Returns (S, X_e, iters, converged)."""
    Xe, it, _, ok = cg(dims, kappa, bc, U, phi, tol, max_iter)
    return oracle.redot(keep(phi, dims, 0), Xe), Xe, it, ok


def fermion_force(dims, kappa, bc, U, phi, tol, max_iter):
    """Per-link force of S_F^eo: the full-lattice formula on the reconstructed X, Y.  Returns (F, iters, converged)."""
    X, Y, it, ok = solve_xy(dims, kappa, bc, U, phi, tol, max_iter)
    return oracle.fermion_force(dims, kappa, bc, U, X, Y), it, ok
