// lgt_oracle.cpp -- plain CPU oracle for the HMC force hot path.
//
// TEST INFRASTRUCTURE, NOT PRODUCT CODE (see lgt_oracle.h).  Slow and written to be
// checked against the definitions by eye: full 4x4 gamma matrices on full 4-spinors
// (no half-spinor trick), explicit 3x3 complex products, lexicographic site loops,
// matrix exponential by a scaled Taylor series, textbook CG.  complex<double> throughout.
// OpenMP only parallelises loops whose iterations write disjoint outputs; every global
// sum is taken serially in site order over per-site partials, so results do not depend
// on the thread count.
//
// What is computed (citations: PAPER.md line / equation; "configs[0]" = BASELINE.json):
//   gauge action   S_g = beta sum_P (1 - Re tr U_P / 3)                       configs[0]
//   Wilson-Dirac   D = 1 - kappa sum_mu [(1-g_mu) U_mu(x) d_{x+mu} + (1+g_mu) U_mu^dag(x-mu) d_{x-mu}]   configs[0]
//   pseudofermion  S_f = phi^dag (D^dag D)^-1 phi                              PAPER.md:377 (S3.1)
//   solve          A chi = phi, A = D^dag D, by CG, not differentiated
//   eta = D chi ;  dS_f = -2 Re[eta^dag (dD) chi]                              PAPER.md:417 (S3.10), 425 (S3.12)
//   projector      P[A] = (A - A^dag)/2 - tr(A - A^dag)/(2N)                   PAPER.md:109 (7), 294 (S2.9)
//   MD             U <- exp(dt Pi) U ; Pi <- Pi - dt F                         PAPER.md:261-263 (S2.1, S2.2)
// Pi here is the paper's iP (anti-Hermitian), reading A-1.
// Force normalisation: F = sum_a tau^a d_a S with d_a S = d/dt S(exp(t tau^a) U)|_0,
// i.e. d_a S = -2 tr(tau^a F); pinned by finite differences in tests/.

#include "lgt_oracle.h"

#include <cmath>
#include <complex>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef std::complex<double> cd;
const cd I_(0.0, 1.0);

struct Mat3 {
    cd e[3][3];
};
struct Spinor {
    cd c[4][3];  // [spin][colour]
};

Mat3 zero3() {
    Mat3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.e[i][j] = 0.0;
    return r;
}
Mat3 ident3() {
    Mat3 r = zero3();
    for (int i = 0; i < 3; i++) r.e[i][i] = 1.0;
    return r;
}
Mat3 mul(const Mat3& a, const Mat3& b) {
    Mat3 r = zero3();
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            for (int k = 0; k < 3; k++) r.e[i][j] += a.e[i][k] * b.e[k][j];
    return r;
}
Mat3 dag(const Mat3& a) {
    Mat3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.e[i][j] = std::conj(a.e[j][i]);
    return r;
}
Mat3 add(const Mat3& a, const Mat3& b) {
    Mat3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.e[i][j] = a.e[i][j] + b.e[i][j];
    return r;
}
Mat3 scale(const Mat3& a, cd s) {
    Mat3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) r.e[i][j] = s * a.e[i][j];
    return r;
}
cd trace(const Mat3& a) { return a.e[0][0] + a.e[1][1] + a.e[2][2]; }
double frob2(const Mat3& a) {
    double s = 0;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) s += std::norm(a.e[i][j]);
    return s;
}

// P_su(3)[M]  (Eq. 7 with N_c = 3)
Mat3 TA(const Mat3& m) {
    Mat3 d = add(m, scale(dag(m), -1.0));  // M - M^dag
    cd tr = trace(d);
    Mat3 r = scale(d, 0.5);
    for (int i = 0; i < 3; i++) r.e[i][i] -= tr / 6.0;
    return r;
}

// exp(A): scale A by 2^-s until ||A||_F < 1/16, 30-term Taylor series, square s times.
Mat3 expm(const Mat3& A) {
    double nrm = std::sqrt(frob2(A));
    int s = 0;
    while (std::ldexp(nrm, -s) >= 1.0 / 16.0) s++;
    Mat3 B = scale(A, std::ldexp(1.0, -s));
    Mat3 E = ident3();
    Mat3 T = ident3();
    for (int k = 1; k <= 30; k++) {
        T = scale(mul(T, B), 1.0 / k);
        E = add(E, T);
    }
    for (int q = 0; q < s; q++) E = mul(E, E);
    return E;
}

// ---- gamma matrices: chiral basis, gamma_mu = [[0, sigma_mu], [sigma_mu^dag, 0]] (A-6)
struct Gammas {
    cd g[5][4][4];
    Gammas() {
        cd sig[4][2][2] = {
            {{0.0, -I_}, {-I_, 0.0}},  // x
            {{0.0, -1.0}, {1.0, 0.0}},  // y
            {{-I_, 0.0}, {0.0, I_}},  // z
            {{1.0, 0.0}, {0.0, 1.0}},  // t
        };
        for (int mu = 0; mu < 4; mu++) {
            for (int a = 0; a < 4; a++)
                for (int b = 0; b < 4; b++) g[mu][a][b] = 0.0;
            for (int a = 0; a < 2; a++)
                for (int b = 0; b < 2; b++) {
                    g[mu][a][2 + b] = sig[mu][a][b];
                    g[mu][2 + a][b] = std::conj(sig[mu][b][a]);
                }
        }
        // gamma_5 = gamma_x gamma_y gamma_z gamma_t
        cd t1[4][4], t2[4][4];
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) {
                t1[a][b] = 0.0;
                for (int k = 0; k < 4; k++) t1[a][b] += g[0][a][k] * g[1][k][b];
            }
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) {
                t2[a][b] = 0.0;
                for (int k = 0; k < 4; k++) t2[a][b] += t1[a][k] * g[2][k][b];
            }
        for (int a = 0; a < 4; a++)
            for (int b = 0; b < 4; b++) {
                g[4][a][b] = 0.0;
                for (int k = 0; k < 4; k++) g[4][a][b] += t2[a][k] * g[3][k][b];
            }
    }
};
const Gammas GAM;

// ---- Gell-Mann matrices, tau^a = i lambda^a / 2
Mat3 generator(int a) {
    Mat3 l = zero3();
    switch (a) {
        case 0: l.e[0][1] = 1.0; l.e[1][0] = 1.0; break;
        case 1: l.e[0][1] = -I_; l.e[1][0] = I_; break;
        case 2: l.e[0][0] = 1.0; l.e[1][1] = -1.0; break;
        case 3: l.e[0][2] = 1.0; l.e[2][0] = 1.0; break;
        case 4: l.e[0][2] = -I_; l.e[2][0] = I_; break;
        case 5: l.e[1][2] = 1.0; l.e[2][1] = 1.0; break;
        case 6: l.e[1][2] = -I_; l.e[2][1] = I_; break;
        case 7: {
            double r = 1.0 / std::sqrt(3.0);
            l.e[0][0] = r; l.e[1][1] = r; l.e[2][2] = -2.0 * r;
            break;
        }
    }
    return scale(l, 0.5 * I_);
}

// ---- lattice geometry
struct Lattice {
    int L[4];
    long V;
    explicit Lattice(const int* dims) {
        V = 1;
        for (int m = 0; m < 4; m++) {
            L[m] = dims[m];
            V *= L[m];
        }
    }
    void coords(long s, int x[4]) const {
        for (int m = 0; m < 4; m++) {
            x[m] = (int)(s % L[m]);
            s /= L[m];
        }
    }
    long index(const int x[4]) const {
        return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3]));
    }
    long fwd(long s, int mu) const {
        int x[4];
        coords(s, x);
        x[mu] = (x[mu] + 1) % L[mu];
        return index(x);
    }
    long bwd(long s, int mu) const {
        int x[4];
        coords(s, x);
        x[mu] = (x[mu] + L[mu] - 1) % L[mu];
        return index(x);
    }
    // fermion sign carried by the link U_mu(s): bc[mu] if the link crosses the boundary
    double link_sign(long s, int mu, const int* bc) const {
        int x[4];
        coords(s, x);
        return (x[mu] == L[mu] - 1) ? (double)bc[mu] : 1.0;
    }
};

const Mat3& link(const double* U, long s, int mu) {
    return *reinterpret_cast<const Mat3*>(U + (s * 4 + mu) * 18);
}
Mat3& link(double* U, long s, int mu) { return *reinterpret_cast<Mat3*>(U + (s * 4 + mu) * 18); }
const Spinor& spinor(const double* p, long s) {
    return *reinterpret_cast<const Spinor*>(p + s * 24);
}
Spinor& spinor(double* p, long s) { return *reinterpret_cast<Spinor*>(p + s * 24); }

// colour multiplication, spin by spin:  (M psi)[alpha][a] = sum_b M[a][b] psi[alpha][b]
Spinor colour_mul(const Mat3& M, const Spinor& p) {
    Spinor r;
    for (int al = 0; al < 4; al++)
        for (int a = 0; a < 3; a++) {
            cd acc = 0.0;
            for (int b = 0; b < 3; b++) acc += M.e[a][b] * p.c[al][b];
            r.c[al][a] = acc;
        }
    return r;
}
// (1 + sgn*gamma_mu) psi
Spinor one_plus_gamma(int mu, double sgn, const Spinor& p) {
    Spinor r;
    for (int al = 0; al < 4; al++)
        for (int a = 0; a < 3; a++) {
            cd acc = p.c[al][a];
            for (int be = 0; be < 4; be++) acc += sgn * GAM.g[mu][al][be] * p.c[be][a];
            r.c[al][a] = acc;
        }
    return r;
}

// (D psi)(s), or (D^dag psi)(s) for dagger: gamma_mu -> -gamma_mu  (gamma5-hermiticity)
Spinor dslash_site(const Lattice& lat, double kappa, const int* bc, const double* U,
                   const double* in, long s, int dagger) {
    const double g = dagger ? -1.0 : 1.0;
    Spinor out = spinor(in, s);
    for (int mu = 0; mu < 4; mu++) {
        long sf = lat.fwd(s, mu);
        double sgf = lat.link_sign(s, mu, bc);
        Spinor hop = one_plus_gamma(mu, -g, colour_mul(link(U, s, mu), spinor(in, sf)));
        long sb = lat.bwd(s, mu);
        double sgb = lat.link_sign(sb, mu, bc);
        Spinor hopb = one_plus_gamma(mu, +g, colour_mul(dag(link(U, sb, mu)), spinor(in, sb)));
        for (int al = 0; al < 4; al++)
            for (int a = 0; a < 3; a++)
                out.c[al][a] -= kappa * (sgf * hop.c[al][a] + sgb * hopb.c[al][a]);
    }
    return out;
}

void dslash(const Lattice& lat, double kappa, const int* bc, const double* U, const double* in,
            double* out, int dagger) {
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) spinor(out, s) = dslash_site(lat, kappa, bc, U, in, s, dagger);
}

// Re <a,b> with a serial sum in index order
double redot(long n, const double* a, const double* b) {
    double acc = 0.0;
    for (long i = 0; i < n; i++) acc += a[2 * i] * b[2 * i] + a[2 * i + 1] * b[2 * i + 1];
    return acc;
}

// Textbook CG on A = D^dag D, x0 = 0 (reading A-10)
int cg(const Lattice& lat, double kappa, const int* bc, const double* U, const double* b,
       double* x, double tol, int max_iter, int* iters, double* rel_resid) {
    const long n = lat.V * 12;  // complex numbers per spinor field
    std::vector<double> r(2 * n), p(2 * n), t(2 * n), q(2 * n);
    for (long i = 0; i < 2 * n; i++) {
        x[i] = 0.0;
        r[i] = b[i];
        p[i] = b[i];
    }
    double rr = redot(n, r.data(), r.data());
    const double bb = rr;
    int k = 0;
    if (bb == 0.0) {
        *iters = 0;
        *rel_resid = 0.0;
        return 0;
    }
    while (rr > tol * tol * bb && k < max_iter) {
        dslash(lat, kappa, bc, U, p.data(), t.data(), 0);  // t = D p
        dslash(lat, kappa, bc, U, t.data(), q.data(), 1);  // q = D^dag t = A p
        double pq = redot(n, p.data(), q.data());
        double alpha = rr / pq;
        for (long i = 0; i < 2 * n; i++) x[i] += alpha * p[i];
        for (long i = 0; i < 2 * n; i++) r[i] -= alpha * q[i];
        double rr_new = redot(n, r.data(), r.data());
        double beta = rr_new / rr;
        for (long i = 0; i < 2 * n; i++) p[i] = r[i] + beta * p[i];
        rr = rr_new;
        k++;
    }
    *iters = k;
    *rel_resid = std::sqrt(rr / bb);
    return (rr > tol * tol * bb) ? 1 : 0;
}

// U_P = U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)
Mat3 plaquette(const Lattice& lat, const double* U, long s, int mu, int nu) {
    long smu = lat.fwd(s, mu), snu = lat.fwd(s, nu);
    return mul(mul(link(U, s, mu), link(U, smu, nu)), mul(dag(link(U, snu, mu)), dag(link(U, s, nu))));
}

// V_mu(x) = sum_{nu != mu} [ U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)
//                           + U_nu^dag(x+mu-nu) U_mu^dag(x-nu) U_nu(x-nu) ]
Mat3 staple_sum(const Lattice& lat, const double* U, long s, int mu) {
    Mat3 V = zero3();
    long smu = lat.fwd(s, mu);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        long snu = lat.fwd(s, nu);
        Mat3 up = mul(mul(link(U, smu, nu), dag(link(U, snu, mu))), dag(link(U, s, nu)));
        long sdn = lat.bwd(s, nu);
        long smudn = lat.bwd(smu, nu);
        Mat3 dn = mul(mul(dag(link(U, smudn, nu)), dag(link(U, sdn, mu))), link(U, sdn, nu));
        V = add(V, add(up, dn));
    }
    return V;
}

Mat3 gauge_force_link(const Lattice& lat, double beta, const double* U, long s, int mu) {
    return scale(TA(mul(link(U, s, mu), staple_sum(lat, U, s, mu))), beta / 6.0);
}

// C_mu(x)_{ab} = sum_alpha { [(1-g_mu) X(x+mu)]_{alpha a} conj(Y(x)_{alpha b})
//                          + [(1+g_mu) Y(x+mu)]_{alpha a} conj(X(x)_{alpha b}) }
// F = -kappa TA( s_mu(x) U_mu(x) C_mu(x) )        from dS_f = -2 Re[Y^dag (dD) X]
Mat3 fermion_force_link(const Lattice& lat, double kappa, const int* bc, const double* U,
                        const double* X, const double* Y, long s, int mu) {
    long sf = lat.fwd(s, mu);
    Spinor a = one_plus_gamma(mu, -1.0, spinor(X, sf));
    Spinor b = one_plus_gamma(mu, +1.0, spinor(Y, sf));
    const Spinor& xs = spinor(X, s);
    const Spinor& ys = spinor(Y, s);
    Mat3 C = zero3();
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            for (int al = 0; al < 4; al++)
                C.e[i][j] += a.c[al][i] * std::conj(ys.c[al][j]) + b.c[al][i] * std::conj(xs.c[al][j]);
    double sg = lat.link_sign(s, mu, bc);
    return scale(TA(scale(mul(link(U, s, mu), C), sg)), -kappa);
}

}  // namespace

extern "C" {

void lgto_gamma(int mu, double* out) {
    cd* o = reinterpret_cast<cd*>(out);
    for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) o[a * 4 + b] = GAM.g[mu][a][b];
}

void lgto_generator(int a, double* out) { *reinterpret_cast<Mat3*>(out) = generator(a); }

void lgto_ta(const double* M, double* out) {
    *reinterpret_cast<Mat3*>(out) = TA(*reinterpret_cast<const Mat3*>(M));
}

void lgto_expm(const double* A, double* out) {
    *reinterpret_cast<Mat3*>(out) = expm(*reinterpret_cast<const Mat3*>(A));
}

void lgto_gauge_action(const int* dims, double beta, const double* U, double* S_g, double* plaq) {
    Lattice lat(dims);
    std::vector<double> part(lat.V);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++) {
        double acc = 0.0;
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) acc += trace(plaquette(lat, U, s, mu, nu)).real() / 3.0;
        part[s] = acc;
    }
    double sum = 0.0;
    for (long s = 0; s < lat.V; s++) sum += part[s];
    *S_g = beta * (6.0 * (double)lat.V - sum);
    *plaq = sum / (6.0 * (double)lat.V);
}

void lgto_dslash(const int* dims, double kappa, const int* bc, const double* U, const double* in,
                 double* out, int dagger) {
    Lattice lat(dims);
    dslash(lat, kappa, bc, U, in, out, dagger);
}

void lgto_dslash_sites(const int* dims, double kappa, const int* bc, const double* U,
                       const double* in, int dagger, const long* sites, long n, double* out) {
    Lattice lat(dims);
    for (long i = 0; i < n; i++) spinor(out, i) = dslash_site(lat, kappa, bc, U, in, sites[i], dagger);
}

int lgto_cg(const int* dims, double kappa, const int* bc, const double* U, const double* b,
            double* x, double tol, int max_iter, int* iters, double* rel_resid) {
    Lattice lat(dims);
    return cg(lat, kappa, bc, U, b, x, tol, max_iter, iters, rel_resid);
}

void lgto_gauge_force(const int* dims, double beta, const double* U, double* F) {
    Lattice lat(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) link(F, s, mu) = gauge_force_link(lat, beta, U, s, mu);
}

void lgto_gauge_force_link(const int* dims, double beta, const double* U, long s, int mu, double* F) {
    Lattice lat(dims);
    *reinterpret_cast<Mat3*>(F) = gauge_force_link(lat, beta, U, s, mu);
}

void lgto_fermion_force(const int* dims, double kappa, const int* bc, const double* U,
                        const double* X, const double* Y, double* F) {
    Lattice lat(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) link(F, s, mu) = fermion_force_link(lat, kappa, bc, U, X, Y, s, mu);
}

void lgto_fermion_force_link(const int* dims, double kappa, const int* bc, const double* U,
                             const double* X, const double* Y, long s, int mu, double* F) {
    Lattice lat(dims);
    *reinterpret_cast<Mat3*>(F) = fermion_force_link(lat, kappa, bc, U, X, Y, s, mu);
}

void lgto_kinetic(const int* dims, const double* P, double* K) {
    Lattice lat(dims);
    double acc = 0.0;
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) acc += frob2(link(P, s, mu));
    *K = acc;
}

double lgto_redot(long n, const double* a, const double* b) { return redot(n, a, b); }

int lgto_fermion_action(const int* dims, double kappa, const int* bc, const double* U,
                        const double* phi, double tol, int max_iter, double* S_F, double* X,
                        int* iters) {
    Lattice lat(dims);
    std::vector<double> x(lat.V * 24);
    double rel;
    int rc = cg(lat, kappa, bc, U, phi, x.data(), tol, max_iter, iters, &rel);
    *S_F = redot(lat.V * 12, phi, x.data());
    if (X) std::memcpy(X, x.data(), sizeof(double) * x.size());
    return rc;
}

void lgto_drift(const int* dims, double eps, const double* P, double* U) {
    Lattice lat(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; s++)
        for (int mu = 0; mu < 4; mu++) {
            Mat3 E = expm(scale(link(P, s, mu), eps));
            link(U, s, mu) = mul(E, link(U, s, mu));
        }
}

int lgto_kick(const int* dims, double beta, double kappa, const int* bc, const double* U,
              const double* phi, double* P, double eps, double tol, int max_iter, int* iters) {
    Lattice lat(dims);
    const long nl = lat.V * 4 * 18;
    std::vector<double> F(nl);
    int rc = 0;
    *iters = 0;
    lgto_gauge_force(dims, beta, U, F.data());
    for (long i = 0; i < nl; i++) P[i] -= eps * F[i];
    if (phi != nullptr && kappa != 0.0) {
        std::vector<double> X(lat.V * 24), Y(lat.V * 24);
        double rel;
        rc = cg(lat, kappa, bc, U, phi, X.data(), tol, max_iter, iters, &rel);
        dslash(lat, kappa, bc, U, X.data(), Y.data(), 0);  // Y = D X
        lgto_fermion_force(dims, kappa, bc, U, X.data(), Y.data(), F.data());
        for (long i = 0; i < nl; i++) P[i] -= eps * F[i];
    }
    return rc;
}

int lgto_trajectory(const int* dims, double beta, double kappa, const int* bc, double* U,
                    const double* phi, double* P, int nsteps, double dt, double tol, int max_iter,
                    long* cg_iters) {
    int rc = 0, it = 0;
    long total = 0;
    if (nsteps <= 0) {
        if (cg_iters) *cg_iters = 0;
        return 0;
    }
    rc |= lgto_kick(dims, beta, kappa, bc, U, phi, P, 0.5 * dt, tol, max_iter, &it);
    total += it;
    for (int n = 0; n < nsteps; n++) {
        lgto_drift(dims, dt, P, U);
        double e = (n == nsteps - 1) ? 0.5 * dt : dt;
        rc |= lgto_kick(dims, beta, kappa, bc, U, phi, P, e, tol, max_iter, &it);
        total += it;
    }
    if (cg_iters) *cg_iters = total;
    return rc;
}

int lgto_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void lgto_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

}  // extern "C"
