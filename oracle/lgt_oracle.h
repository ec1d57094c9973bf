/*
 * lgt_oracle.h -- C ABI of the CPU oracle.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code with the CUDA path (paper_2602_20516_b200/csrc) and
 * neither side includes or imports the other.
 *
 * Every function is stateless and takes HOST pointers in the canonical layout:
 *
 *   site index  s = x + Lx*(y + Ly*(z + Lz*t))      (x fastest)   dims = {Lx,Ly,Lz,Lt}
 *   links       U[s][mu][i][j]   complex double (re,im), row-major 3x3, mu = 0..3 = x,y,z,t
 *   spinors     psi[s][alpha][a] complex double, alpha = 0..3 spin, a = 0..2 colour
 *   momenta / forces  P[s][mu][i][j]  traceless anti-Hermitian 3x3
 *
 * bc[mu] = +1 / -1 is the fermion boundary sign picked up by a hop across the
 * mu boundary (gauge links themselves stay periodic).
 *
 * Citations are to /root/reference/PAPER.md (line numbers) and to
 * BASELINE.json configs[0], which states the Wilson actions the paper only names.
 */
#ifndef LGT_ORACLE_H
#define LGT_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

/* gamma_mu (mu=0..3) and gamma_5 (mu=4) as 4x4 complex row-major: out[16] complex. */
void lgto_gamma(int mu, double* out);

/* tau^a = i lambda^a / 2, a = 0..7 (Gell-Mann), out[9] complex row-major. */
void lgto_generator(int a, double* out);

/* P_su(3)[M] = (M - M^dag)/2 - tr(M - M^dag)/6   (PAPER.md:109 Eq. 7, :294 Eq. S2.9). */
void lgto_ta(const double* M, double* out);

/* exp(A) of a 3x3 complex matrix by scaled Taylor series + repeated squaring. */
void lgto_expm(const double* A, double* out);

/* S_g = beta * sum_x sum_{mu<nu} (1 - Re tr U_P / 3);  plaq = mean of Re tr U_P / 3. */
void lgto_gauge_action(const int* dims, double beta, const double* U,
                       double* S_g, double* plaq);

/* out = D in (dagger = 0) or D^dag in (dagger = 1); Wilson-Dirac, BASELINE.json configs[0]. */
void lgto_dslash(const int* dims, double kappa, const int* bc, const double* U,
                 const double* in, double* out, int dagger);

/* (D psi)(site) for a list of sites only: out[n][4][3]. */
void lgto_dslash_sites(const int* dims, double kappa, const int* bc, const double* U,
                       const double* in, int dagger, const long* sites, long n, double* out);

/* CG on D^dag D x = b from x0 = 0 (PAPER.md:397-401 Eq. S3.6, :454).
 * Stops when rr <= tol^2 * bb or after max_iter applications of D^dag D.
 * Returns 0 if converged, 1 if the cap was hit. */
int lgto_cg(const int* dims, double kappa, const int* bc, const double* U,
            const double* b, double* x, double tol, int max_iter,
            int* iters, double* rel_resid);

/* F^g_mu(x) = (beta/6) TA(U_mu(x) V_mu(x)), V = sum of the six staples. */
void lgto_gauge_force(const int* dims, double beta, const double* U, double* F);

/* Force for ONE link only (s, mu): F[9] complex. */
void lgto_gauge_force_link(const int* dims, double beta, const double* U,
                           long s, int mu, double* F);

/* F^f_mu(x) = -kappa TA(s_mu(x) U_mu(x) C_mu(x))  (PAPER.md:425 Eq. S3.12), X = (D^dag D)^-1 phi, Y = D X. */
void lgto_fermion_force(const int* dims, double kappa, const int* bc, const double* U,
                        const double* X, const double* Y, double* F);

/* Force for ONE link only (s, mu): F[9] complex. */
void lgto_fermion_force_link(const int* dims, double kappa, const int* bc, const double* U,
                             const double* X, const double* Y, long s, int mu, double* F);

/* K = sum_{x,mu} ||P_mu(x)||_F^2. */
void lgto_kinetic(const int* dims, const double* P, double* K);

/* Re <a, b> = Re sum conj(a) b over n complex numbers. */
double lgto_redot(long n, const double* a, const double* b);

/* S_F = Re phi^dag X with X from CG (PAPER.md:377 Eq. S3.1).  X (optional, may be NULL) receives the solution. */
int lgto_fermion_action(const int* dims, double kappa, const int* bc, const double* U,
                        const double* phi, double tol, int max_iter,
                        double* S_F, double* X, int* iters);

/* U_mu(x) <- expm(eps P_mu(x)) U_mu(x)   (PAPER.md:97 Eq. 5, :261 Eq. S2.1). */
void lgto_drift(const int* dims, double eps, const double* P, double* U);

/* P <- P - eps (F^g + F^f)   (PAPER.md:263 Eq. S2.2).  phi == NULL or kappa == 0: gauge only.
 * Returns 0, or 1 if CG failed to converge. */
int lgto_kick(const int* dims, double beta, double kappa, const int* bc, const double* U,
              const double* phi, double* P, double eps, double tol, int max_iter, int* iters);

/* Leapfrog: kick(dt/2) {drift(dt) kick(dt)}^(n-1) drift(dt) kick(dt/2).  cg_iters: total over kicks. */
int lgto_trajectory(const int* dims, double beta, double kappa, const int* bc,
                    double* U, const double* phi, double* P,
                    int nsteps, double dt, double tol, int max_iter, long* cg_iters);

/* Number of OpenMP threads the loops over sites use. */
int lgto_num_threads(void);
void lgto_set_num_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
