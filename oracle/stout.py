"""CPU oracle for stout-smeared Wilson fermions -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

SURVEY.md 8(f)3: the paper's motivating "compositional action" and its second HMC set-up,
Wilson fermions on stout links with rho = 0.3.  Only tests/ may import this module.  It shares
no code with paper_2602_20516_b200.  The paper gives no formula (it differentiates the code); the smearing is that of
its ref. [6], restated here in the conventions of DESIGN.md section 2:

    one level:   U'_mu(x) = exp(A_mu(x)) U_mu(x),   A_mu(x) = -rho P_su(3)[U_mu(x) V_mu(x)],   V = sum of the six staples
                 (ref. [6]: U' = exp(iQ) U with Omega = C U^dag, C = rho V^dag, iQ = P_su(3)[Omega] = -rho P_su(3)[U V])
    n levels:    U^(0) = U, U^(k+1) = smear(U^(k));   fermions see U^(n), the gauge action the thin links U^(0).
    S_F[U] = phi^dag (D[U^(n)]^dag D[U^(n)])^-1 phi.

The forward map is composed from pinned pieces only: P_su(3)[U V] = oracle.gauge_force at beta = 6 and
exp(A) U = oracle.drift.  The force is the chain rule written out, NOT the closed Cayley-Hamilton recursion of
ref. [6] (that one is the GPU's): with F' the force with respect to U' (the pinned oracle.fermion_force on U'),

    dU' U'^-1 = Phi_A(dA) + Ad_{exp A}(dU U^-1),   Phi_A = sum_k ad_A^k / (k+1)!  (the differential of exp),
    dS = -2 sum tr[(dU' U'^-1) F']
       = -2 sum tr[(dU U^-1) exp(-A) F' exp(A)]                                   (direct term)
         -2 sum tr[dA G],   G = Phi_{-A}(F')  (ad_A is skew for the trace form)    (through the exponent)
    and with dA = -rho P_su(3)[d(U V)]:   -2 tr[dA G] = 2 rho Re tr[d(U V) G], so the second part is the force of
    W[U] = 2 rho sum_{x,mu} Re tr[U_mu(x) V_mu(x) G_mu(x)] at fixed G -- a sum of plaquette loops with one insertion of
    G, differentiated link by link by `loop_force`: for a closed loop Re tr[M_1 ... M_n], replacing U -> exp(t tau) U in
    the factor M_i gives Re tr[tau R_i] with R_i the loop rotated to start at M_i (and a minus sign, rotated to start
    after it, if M_i is a dagger); the force is -1/2 P_su(3)[R_i] per unit coefficient.

Pins (tests/test_oracle_stout_pins.py): central finite differences of the smeared action along every generator on
sampled links for one and two levels; Phi_{-A} against the block-triangular matrix exponential of a library routine;
gauge covariance of the smearing; rho = 0 is the identity; the unit field is a fixed point; W's force against a
finite difference of the pinned gauge force along G.
"""
import numpy as np

import oracle


# ---------------------------------------------------------------------------------------------- helpers
def _grid(f, dims):
    Lx, Ly, Lz, Lt = [int(d) for d in dims]
    return f.reshape((Lt, Lz, Ly, Lx) + f.shape[1:])


def _shift(f, dims, mu, d):
    """f'(x) = f(x + d mu_hat), periodic; fields are [V, ...] in the canonical site order."""
    V = f.shape[0]
    return np.roll(_grid(f, dims), -d, axis=3 - mu).reshape((V,) + f.shape[1:])


def _dag(M):
    return M.conj().swapaxes(-1, -2)


def _ta(M):
    A = 0.5 * (M - _dag(M))
    tr = np.trace(A, axis1=-2, axis2=-1) / 3.0
    return A - tr[..., None, None] * np.eye(3)


# ---------------------------------------------------------------------------------------------- forward map
def smear(dims, rho, U):
    """One stout level.  Returns (U', A) with A[V,4,3,3] the su(3) exponent of every link."""
    A = -rho * oracle.gauge_force(dims, 6.0, U)  # gauge_force = (beta/6) P_su(3)[U V]
    return oracle.drift(dims, 1.0, A, U), A


def smear_levels(dims, rho, n, U):
    """Returns ([U^(0), ..., U^(n)], [A^(1), ..., A^(n)])."""
    Us, As = [np.ascontiguousarray(U, dtype=np.complex128)], []
    for _ in range(n):
        U1, A = smear(dims, rho, Us[-1])
        Us.append(U1)
        As.append(A)
    return Us, As


def fermion_action(dims, kappa, bc, U, phi, n, rho, tol=1e-12, max_iter=100000):
    """S_F on n-level stout links.  Returns (S_F, X, iters, converged)."""
    Us, _ = smear_levels(dims, rho, n, U)
    return oracle.fermion_action(dims, kappa, bc, Us[-1], phi, tol, max_iter)


# ---------------------------------------------------------------------------------------------- chain rule
def phi_minus(A, F, terms=60):
    """G = Phi_{-A}(F) = sum_k (-ad_A)^k F / (k+1)!, link by link ([..., 3, 3] arrays)."""
    term = np.array(F, dtype=np.complex128, copy=True)
    G = term.copy()
    for k in range(1, terms):
        term = -(A @ term - term @ A) / (k + 1.0)
        G += term
    return G


def loop_force(dims, coeff, factors):
    """Force of  coeff * sum_x Re tr[M_1(x) ... M_n(x)]  with respect to the links.

    factors: list of entries  ("U", mu, offset, dagger)  -- the link field U_mu taken at x + offset (offset a 4-tuple),
    daggered if dagger -- or  ("G", field)  -- a fixed [V,3,3] field, already shifted, that is not differentiated.
    U is passed through `fields`: factors hold the arrays themselves, see `_factor`.  Returns F[V,4,3,3] with
    d/dt (coeff * sum) under U_mu(x) -> exp(t tau^a) U_mu(x) equal to -2 tr[tau^a F_mu(x)]."""
    mats = [f["mat"] for f in factors]
    n = len(mats)
    V = mats[0].shape[0]
    F = np.zeros((V, 4, 3, 3), np.complex128)
    for i, f in enumerate(factors):
        if f["kind"] != "U":
            continue
        if not f["dagger"]:
            order = list(range(i, n)) + list(range(0, i))   # rotated to start at M_i:  Re tr[tau M_i ... M_{i-1}]
            sign = 1.0
        else:
            order = list(range(i + 1, n)) + list(range(0, i + 1))  # d(U^dag) = -U^dag tau: starts after M_i
            sign = -1.0
        R = mats[order[0]]
        for j in order[1:]:
            R = R @ mats[j]
        contrib = -0.5 * coeff * sign * _ta(R)  # Re tr[tau R] = tr[tau P_su(3) R];  dS = -2 tr[tau F]
        # the factor sits at x + offset: move the contribution to the link's own site
        off = f["offset"]
        for mu in range(4):
            if off[mu]:
                contrib = _shift(contrib, dims, mu, -off[mu])
        F[:, f["mu"]] += contrib
    return F


def _factor(dims, U, mu, offset, dagger):
    m = U[:, mu]
    for d in range(4):
        if offset[d]:
            m = _shift(m, dims, d, offset[d])
    return dict(kind="U", mu=mu, offset=tuple(offset), dagger=dagger, mat=_dag(m) if dagger else m)


def w_force(dims, rho, U, G):
    """Force of W[U] = 2 rho sum_{x,mu} Re tr[U_mu(x) V_mu(x) G_mu(x)] at fixed G (module docstring)."""
    F = np.zeros_like(U)
    e = np.eye(4, dtype=int)
    for mu in range(4):
        g = dict(kind="G", mat=G[:, mu])
        for nu in range(4):
            if nu == mu:
                continue
            # U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x) G_mu(x)
            up = [_factor(dims, U, mu, 0 * e[mu], False), _factor(dims, U, nu, e[mu], False),
                  _factor(dims, U, mu, e[nu], True), _factor(dims, U, nu, 0 * e[nu], True), g]
            F += loop_force(dims, 2.0 * rho, up)
            # U_mu(x) U_nu^dag(x+mu-nu) U_mu^dag(x-nu) U_nu(x-nu) G_mu(x)
            dn = [_factor(dims, U, mu, 0 * e[mu], False), _factor(dims, U, nu, e[mu] - e[nu], True),
                  _factor(dims, U, mu, -e[nu], True), _factor(dims, U, nu, -e[nu], False), g]
            F += loop_force(dims, 2.0 * rho, dn)
    return F


def pull_back(dims, rho, U, A, Fp):
    """Force with respect to U from the force Fp with respect to U' = exp(A) U of one stout level.
    Returns (F, F_direct, G)."""
    E = oracle.drift(dims, 1.0, A, U) @ _dag(U)  # exp(A), U unitary
    F_direct = _dag(E) @ Fp @ E
    G = phi_minus(A, Fp)
    return F_direct + w_force(dims, rho, U, G), F_direct, G


def fermion_force(dims, kappa, bc, U, phi, n, rho, tol=1e-12, max_iter=100000):
    """Force of S_F on n-level stout links with respect to the thin links.  Returns (F, iters, converged)."""
    Us, As = smear_levels(dims, rho, n, U)
    S, X, it, ok = oracle.fermion_action(dims, kappa, bc, Us[-1], phi, tol, max_iter)
    Y = oracle.dslash(dims, kappa, bc, Us[-1], X)
    F = oracle.fermion_force(dims, kappa, bc, Us[-1], X, Y)
    for k in range(n - 1, -1, -1):
        F = pull_back(dims, rho, Us[k], As[k], F)[0]
    return F, it, ok
