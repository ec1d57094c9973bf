/*
 * lgt.h -- C ABI of the B200-native HMC molecular-dynamics force library (liblgt.so).
 *
 * The hot path of arXiv 2602.20516 ("Lattice Gauge Theory via LLVM-Level Automatic
 * Differentiation"), hand-written as CUDA kernels for sm_100a:
 *   Wilson plaquette action and staple force, Wilson-Dirac operator D / D^dag, CG on
 *   D^dag D, two-flavour Wilson fermion force, su(3) projection, leapfrog kick / drift.
 * Citations "PAPER.md:n" are lines of the paper text; "configs[0]" is BASELINE.json's
 * statement of the two Wilson actions, which the paper names but does not write out.
 *
 * Conventions (DESIGN.md has the derivations and every reading of the paper):
 *   dims = {Lx,Ly,Lz,Lt}; V = Lx*Ly*Lz*Lt; canonical site index s = x + Lx*(y + Ly*(z + Lz*t)).
 *   CANONICAL LAYOUT, used by every pointer argument unless the call says "native":
 *     links     U[s][mu][i][j]    complex (re,im), 3x3 row-major, mu = 0..3 = x,y,z,t
 *     spinors   psi[s][alpha][a]  complex, alpha = 0..3 spin (chiral basis, gamma5 = diag(1,1,-1,-1)),
 *                                 a = 0..2 colour
 *     momenta and forces  P[s][mu][i][j]  traceless anti-Hermitian 3x3 (the paper's iP)
 *   Element type is complex double for an LGT_F64 handle, complex float for LGT_F32.
 *   All field pointers are DEVICE pointers to caller-owned buffers, unless the call's name ends
 *   in _host.  Output scalars are written through HOST pointers.
 *   The handle owns its copies of U, Pi, phi and all workspaces in the internal ("native")
 *   structure-of-arrays layout; set/get calls convert.
 *   Every call returns LGT_OK or a negative error code and never throws or aborts; after an
 *   error lgt_last_error(ctx) gives a message.  Work is enqueued on the handle's stream; calls
 *   that return host scalars synchronise that stream only.  A handle is not thread-safe.
 *   There is no CPU fallback: without a CUDA device lgt_create fails with LGT_ECUDA.
 *
 * MD equations (Eqs. S2.1-S2.2, with Pi = iP anti-Hermitian):
 *     U_mu(x) <- exp(dt Pi_mu(x)) U_mu(x),      Pi_mu(x) <- Pi_mu(x) - dt F_mu(x),
 *   F = P_su(3)[...] (Eq. 7), normalised so that
 *     d/dt S(exp(t tau^a) U_mu(x))|_0 = -2 tr(tau^a F_mu(x)),  tau^a = i lambda^a / 2,
 *   and H = K + S_g + S_F with K = sum_{x,mu} ||Pi_mu(x)||_F^2.
 */
#ifndef LGT_H
#define LGT_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct lgt_ctx lgt_ctx; /* opaque */

enum { LGT_OK = 0, LGT_EINVAL = -1, LGT_ENOMEM = -2, LGT_ECUDA = -3, LGT_ENOCONV = -4, LGT_ESTATE = -5 };
enum { LGT_F64 = 0, LGT_F32 = 1 };
enum { LGT_SOLVER_CG = 0, LGT_SOLVER_MIXED_CG = 1 };
enum { LGT_ACTION_FULL = 0, LGT_ACTION_EO = 1 };
enum { LGT_INT_LEAPFROG = 0, LGT_INT_OMELYAN = 1, LGT_INT_SEXTON_WEINGARTEN = 2 };

/* ---- lifetime -------------------------------------------------------------------------- */

/* Creates a handle for one lattice on CUDA device `device`.
 * dims[4] >= 1 each; beta = gauge coupling of S_g; kappa = hopping parameter of D (0 => gauge only);
 * bc[4] = fermion boundary signs, each +1 or -1 (configs use {1,1,1,-1}); precision = LGT_F64 / LGT_F32;
 * cuda_stream = a cudaStream_t to enqueue on, or NULL for the default stream.
 * Links start as the unit field, momenta and pseudofermion as zero ("not set").
 * Errors: LGT_EINVAL (bad argument), LGT_ECUDA (no device / CUDA failure), LGT_ENOMEM. */
int lgt_create(lgt_ctx** out, const int dims[4], double beta, double kappa, const int bc[4],
               int precision, int device, void* cuda_stream);
int lgt_destroy(lgt_ctx* ctx);
/* Message of the last error on this handle (or of the last failed lgt_create if ctx == NULL).
 * Owned by the library; valid until the next call. */
const char* lgt_last_error(const lgt_ctx* ctx);
/* Library version string, static. */
const char* lgt_version(void);

/* ---- state upload / download (canonical layout, device pointers) ------------------------ */
int lgt_set_links(lgt_ctx* ctx, const void* U);           /* [V][4][3][3] complex */
int lgt_get_links(lgt_ctx* ctx, void* U);
int lgt_set_momenta(lgt_ctx* ctx, const void* P);         /* [V][4][3][3]; only the traceless anti-Hermitian part is kept */
int lgt_get_momenta(lgt_ctx* ctx, void* P);
int lgt_set_pseudofermion(lgt_ctx* ctx, const void* phi); /* [V][4][3] complex */

/* Same as the three setters / two getters above with HOST buffers (pageable or pinned): the
 * host<->device copy is made by the library on the handle's stream and the call synchronises. */
int lgt_set_links_host(lgt_ctx* ctx, const void* U);
int lgt_get_links_host(lgt_ctx* ctx, void* U);
int lgt_set_momenta_host(lgt_ctx* ctx, const void* P);
int lgt_get_momenta_host(lgt_ctx* ctx, void* P);
int lgt_set_pseudofermion_host(lgt_ctx* ctx, const void* phi);

/* Asynchronous forms (undivided lattices; LGT_ESTATE on a slab handle): the transfer and the layout conversion are enqueued --
 * the copies on the handle's own copy stream -- and the call returns at once.  The library orders them against its kernels:
 * a kernel that touches Pi waits for a pending upload of Pi (lgt_md_kick solves first, which does not need Pi, so the upload
 * overlaps the solve), an upload starts after everything enqueued before it, a download converts on the handle's stream and
 * copies behind it, so that the next step's uploads and kernels run under it.  HOST buffers (pinned, for any overlap to
 * happen) must stay valid, and a downloaded buffer is complete, only after lgt_host_transfers_wait(ctx) has returned. */
int lgt_set_momenta_host_async(lgt_ctx* ctx, const void* P);
int lgt_get_links_host_async(lgt_ctx* ctx, void* U);
int lgt_get_momenta_host_async(lgt_ctx* ctx, void* P);
int lgt_host_transfers_wait(lgt_ctx* ctx);

/* ---- A1: actions (configs[0]; PAPER.md:377 Eq. S3.1) ------------------------------------ */
/* S_g = beta sum_x sum_{mu<nu} (1 - Re tr U_P/3);  S_F = Re phi^dag (D^dag D)^-1 phi (CG to `tol`,
 * 0 if kappa == 0 or no pseudofermion is set);  K = sum ||Pi||_F^2.  Any output pointer may be NULL.
 * cg_iters (may be NULL) receives the CG iteration count.  LGT_ENOCONV if CG hit max_iter. */
int lgt_action(lgt_ctx* ctx, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters);
/* Mean plaquette (1/6V) sum Re tr U_P / 3. */
int lgt_plaquette(lgt_ctx* ctx, double* plaq);

/* ---- A2: Wilson-Dirac operator (configs[0]) --------------------------------------------- */
/* (D psi)(x) = psi(x) - kappa sum_mu [ (1-gamma_mu) s_mu(x) U_mu(x) psi(x+mu)
 *                                     + (1+gamma_mu) s_mu(x-mu) U_mu^dag(x-mu) psi(x-mu) ],
 * s_mu(x) = bc[mu] on links that cross the mu boundary, else 1.  dagger != 0 applies D^dag
 * (gamma_mu -> -gamma_mu).  in, out: canonical spinors [V][4][3], in != out. */
int lgt_dslash(lgt_ctx* ctx, const void* in, void* out, int dagger);

/* ---- A3: solver (PAPER.md:397-401 Eq. S3.6; :454) ---------------------------------------- */
/* Solves (D^dag D) x = b by conjugate gradient from x0 = 0; stops when the recurrence residual
 * satisfies |r|^2 <= tol^2 |b|^2 or after max_iter applications of D^dag D.
 * iters, rel_resid (= |r|/|b|) may be NULL.  Returns LGT_ENOCONV if the cap was hit (x holds the
 * last iterate). */
int lgt_cg(lgt_ctx* ctx, const void* b, void* x, double tol, int max_iter, int* iters, double* rel_resid);

/* Mixed-precision variant (LGT_F64 handles only).  Same system, same x0 = 0, same answer to
 * tolerance: defect correction x <- x + e where e ~ (D^dag D)^-1 r comes from a CG run entirely in fp32 on the
 * residual scaled to unit norm, to relative residual max(inner_tol, tol |b| / (4 |r|)); then r = b - D^dag D x in
 * fp64.  Stops when the TRUE residual satisfies |r| <= tol |b| (so rel_resid is a true, not a recurrence, residual).
 * From the second cycle on the inner CG keeps the previous cycle's last search direction (p = r + beta p_k, a reliable update
 * instead of a restart) as long as the previous cycle delivered the reduction it was asked for.
 * inner_iters = fp32 CG iterations in total (capped by max_iter), outer_cycles = corrections; any may be NULL.
 * LGT_ENOCONV if the cap (or 40 cycles) was hit; x then holds the last iterate. */
int lgt_cg_mixed(lgt_ctx* ctx, const void* b, void* x, double tol, int max_iter, double inner_tol,
                 int* inner_iters, int* outer_cycles, double* rel_resid);
/* Chooses the solver used wherever the library solves the pseudofermion system itself (lgt_action, lgt_fermion_force
 * with X = Y = NULL, lgt_md_*): LGT_SOLVER_CG (default; the plain CG of lgt_cg, iteration counts identical to the
 * oracle's in fp64) or LGT_SOLVER_MIXED_CG with the given inner_tol (ignored for LGT_SOLVER_CG).  cg_iters outputs
 * then count fp32 iterations.  Combines with LGT_ACTION_EO: fp32 CG on the Schur complement M^dag M inside the same
 * fp64 defect correction on the true residual (the fastest configuration of the MD step, bench.py "extras"). */
int lgt_set_solver(lgt_ctx* ctx, int solver, double inner_tol);

/* ---- even/odd (Schur) preconditioning (every extent of the lattice must be even) ---------- */
/* With sites split by parity p = (x+y+z+t) mod 2, D = [[1, -kappa H_eo], [-kappa H_oe, 1]] and
 *   M = 1 - kappa^2 H_eo H_oe   (acts on even sites),   det D = det M,
 * so phi_e^dag (M^dag M)^-1 phi_e is a pseudofermion action for the same two-flavour determinant as
 * phi^dag (D^dag D)^-1 phi, with a better conditioned solve on half the sites.
 * lgt_eo_mhat: out = M in (dagger != 0: M^dag in) on the even sites of canonical full-size spinors; odd sites of
 *   `in` are ignored and odd sites of `out` are set to zero.
 * lgt_eo_cg: solves (M^dag M) x_e = b_e by the same CG recurrence and stop rule as lgt_cg (x0 = 0, recurrence
 *   residual, iters = applications of M^dag M); canonical full-size spinors, odd sites ignored / zeroed. */
int lgt_eo_mhat(lgt_ctx* ctx, const void* in, void* out, int dagger);
int lgt_eo_cg(lgt_ctx* ctx, const void* b, void* x, double tol, int max_iter, int* iters, double* rel_resid);
/* Chooses the pseudofermion action used by lgt_action, lgt_fermion_force (X = Y = NULL) and lgt_md_*:
 *   LGT_ACTION_FULL (default): S_F = phi^dag (D^dag D)^-1 phi, the paper's form;
 *   LGT_ACTION_EO: S_F = phi_e^dag (M^dag M)^-1 phi_e (only the even sites of the pseudofermion are used).  Its force
 *     is the same fused per-link kernel applied to X = (X_e, kappa H_oe X_e), Y = (Y_e, kappa H_oe^dag Y_e) with
 *     X_e = (M^dag M)^-1 phi_e, Y_e = M X_e (DESIGN.md derives this from S3.12).
 * LGT_EINVAL if an extent is odd. */
int lgt_set_fermion_action(lgt_ctx* ctx, int action);

/* ---- A4, A5: forces (PAPER.md:105-109 Eq. 7; :425 Eq. S3.12; :462-506 S4) ----------------- */
/* F^g_mu(x) = (beta/6) P_su(3)[ U_mu(x) V_mu(x) ], V = sum of the six staples. F: [V][4][3][3]. */
int lgt_gauge_force(lgt_ctx* ctx, void* F);
/* F^f_mu(x) = -kappa P_su(3)[ s_mu(x) U_mu(x) C_mu(x) ],
 * C_mu(x) = sum_spin (1-gamma_mu)X(x+mu) (x) Y(x)^dag + (1+gamma_mu)Y(x+mu) (x) X(x)^dag (colour outer products).
 * X, Y: canonical spinors with X = (D^dag D)^-1 phi, Y = D X; if both are NULL they are obtained from the
 * handle's pseudofermion by CG to (tol, max_iter).  cg_iters may be NULL. */
int lgt_fermion_force(lgt_ctx* ctx, const void* X, const void* Y, void* F,
                      double tol, int max_iter, int* cg_iters);

/* ---- A6, A7: molecular dynamics (PAPER.md:95-99 Eq. 5; :261-263) -------------------------- */
/* Pi <- Pi - eps (F^g + F^f); the fermion part (CG, Y = D X, fused force) runs if kappa != 0 and a
 * pseudofermion is set.  cg_iters may be NULL. */
int lgt_md_kick(lgt_ctx* ctx, double eps, double tol, int max_iter, int* cg_iters);
/* U_mu(x) <- exp(eps Pi_mu(x)) U_mu(x), exponential by Cayley-Hamilton (ref. [6]). */
int lgt_md_drift(lgt_ctx* ctx, double eps);
/* One leapfrog step: kick(dt/2) drift(dt) kick(dt/2). cg_iters: sum over the two kicks. */
int lgt_md_step(lgt_ctx* ctx, double dt, double tol, int max_iter, int* cg_iters);
/* Leapfrog trajectory kick(dt/2) {drift(dt) kick(dt)}^(n-1) drift(dt) kick(dt/2), with H = K + S_g + S_F
 * evaluated before and after (either pointer may be NULL to skip that evaluation). */
int lgt_md_trajectory(lgt_ctx* ctx, int nsteps, double dt, double tol, int max_iter,
                      double* H_initial, double* H_final, long* cg_iters);

/* ---- HMC around the trajectory (leapfrog, Sexton-Weingarten with inner gauge steps) ---- */
/* Integrator used by lgt_md_trajectory and lgt_hmc_trajectory (a step = dt, adjacent kicks merged; K = kick with both
 * forces, Kg / Kf = gauge / fermion force only, D = drift):
 *   LGT_INT_LEAPFROG (default):   K(dt/2) D(dt) K(dt/2)
 *   LGT_INT_OMELYAN:              K(l dt) D(dt/2) K((1-2l) dt) D(dt/2) K(l dt), l = 0.1931833275037836 (2nd-order minimum norm)
 *   LGT_INT_SEXTON_WEINGARTEN:    Kf(dt/2) [Kg(h/2) D(h) Kg(h/2)]^n_inner Kf(dt/2), h = dt / n_inner (n_inner >= 1; ignored else)
 * lgt_md_step / lgt_md_kick / lgt_md_drift are not affected. */
int lgt_set_integrator(lgt_ctx* ctx, int integrator, int n_inner);
/* Heat baths from the counter-based generator Philox4x32-10, a pure function of (seed, trajectory, element) so that
 * the oracle reproduces them (reading A-25: key = seed, counter = (element, draw, stream, trajectory)):
 *   momenta:        Pi_mu(x) = sum_a pi^a tau^a, pi^a ~ N(0,1), weight exp(-K);
 *   pseudofermion:  eta ~ exp(-eta^dag eta), then phi = D^dag eta (LGT_ACTION_FULL) or phi_e = M^dag eta_e, phi_o = 0
 *                   (LGT_ACTION_EO), so that S_F = |eta|^2 (resp. |eta_e|^2), returned through eta_norm2 (may be NULL).
 * LGT_ESTATE if kappa == 0. */
int lgt_momentum_heatbath(lgt_ctx* ctx, unsigned long long seed, unsigned trajectory);
int lgt_pseudofermion_heatbath(lgt_ctx* ctx, unsigned long long seed, unsigned trajectory, double* eta_norm2);
/* The handle's pseudofermion in the canonical layout, [V][4][3] complex, device pointer.  LGT_ESTATE if none is set. */
int lgt_get_pseudofermion(lgt_ctx* ctx, void* phi);
/* One HMC trajectory: both heat baths (the pseudofermion one if kappa != 0), H_0 = K + S_g + |eta|^2, nsteps steps of
 * the handle's integrator, H_1 = K + S_g + S_F (one more solve), Metropolis test "u < exp(-(H_1 - H_0))" with u the
 * generator's stream-3 uniform of this trajectory; on rejection the links of the start are restored.  The momenta are
 * left as integrated.  Outputs (any may be NULL): dH = H_1 - H_0, accepted = 0 / 1, cg_iters = solver iterations in
 * total, H_initial = H_0.  LGT_ENOCONV if a solve hit max_iter (the trajectory is still completed). */
int lgt_hmc_trajectory(lgt_ctx* ctx, int nsteps, double dt, double tol, int max_iter, unsigned long long seed,
                       unsigned trajectory, double* dH, int* accepted, long* cg_iters, double* H_initial);

/* ---- stout smearing of the fermions' links (rho = 0.3; ref. [6] PAPER.md:196) ---- */
/* With n_levels > 0 the Dirac operator everywhere in the library (lgt_dslash*, lgt_cg*, lgt_eo_*, lgt_action's S_F,
 * lgt_fermion_force, the heat bath, lgt_md_*, lgt_hmc_trajectory) is built on the smeared links U^(n):
 *     U^(k+1)_mu(x) = exp(A) U^(k)_mu(x),   A = -rho P_su(3)[ U^(k)_mu(x) V^(k)_mu(x) ],  V = sum of the six staples
 * (ref. [6]'s exp(iQ) U with Omega = C U^dag, C = rho V^dag), U^(0) = the handle's links; the gauge action stays on
 * U^(0).  The fermion force is then the force with respect to U^(0): the force with respect to U^(n) pulled back level
 * by level with the closed Cayley-Hamilton form of d exp.  lgt_fermion_force with given
 * X, Y expects them to belong to D[U^(n)].  n_levels = 0 (default) switches smearing off; at most 8 levels.
 * lgt_get_smeared_links: U^(n) in the canonical layout, [V][4][3][3], device pointer. */
int lgt_set_smearing(lgt_ctx* ctx, int n_levels, double rho);
int lgt_get_smeared_links(lgt_ctx* ctx, void* U);

/* ---- one lattice on several GPUs: time-slab decomposition -------------- */
/* The lattice dims = {Lx,Ly,Lz,Lt} is cut into nranks slabs of Lt / nranks time slices (Lt % nranks == 0 and
 * Lx*Ly*Lz % 32 == 0, else LGT_EINVAL).  A group object holds this process's ranks: in production ONE rank per
 * process (nlocal = 1, local_ranks = {rank}) and the exchange steps of the path -- the halo slices of the stencil
 * kernels' input field before every Dslash / force launch, the link halo after every link change, and the sums of
 * CG and of the actions -- go through NCCL (send/recv of whole time slices, all-reduce of 1-3 doubles) on the group's
 * stream after lgt_dd_nccl_init.  With nlocal = nranks every rank lives in this process on ONE device and the same
 * exchanges are plain device copies: the verification mode used by the tests (no rank ever waits on another).
 * Field arguments are per-rank SLABS in the canonical layout of the slab's own Lt / nranks time slices
 * ([V/nranks][...], global site order restricted to the slab), given as arrays of nlocal device pointers.
 * State goes in and out through the rank handles: lgt_dd_rank(d, i) returns a handle on which ONLY lgt_set_links,
 * lgt_get_links, lgt_set_momenta, lgt_get_momenta, lgt_set_pseudofermion, lgt_get_pseudofermion (+ _host forms),
 * lgt_timing_* and lgt_launch_count may be called (slab arrays); everything else on it returns LGT_ESTATE.
 * Full operator (plain or mixed-precision CG) or even/odd action, stout-smeared fermion links, all three integrators. */
typedef struct lgt_dd lgt_dd;
int lgt_dd_create(lgt_dd** out, const int dims[4], int nranks, int nlocal, const int* local_ranks, double beta, double kappa,
                  const int bc[4], int precision, int device, void* cuda_stream);
/* The same with TWO split directions ("first T, then Z"): grid = {Pt, Pz}, Pt * Pz ranks, rank = pt * Pz + pz
 * owns the time slices [pt Lt/Pt, (pt+1) Lt/Pt) and the z planes [pz Lz/Pz, (pz+1) Lz/Pz); Lt % Pt == 0, Lz % Pz == 0 and
 * Lx*Ly % 32 == 0, else LGT_EINVAL.  A rank's local lattice has two ghost time slices and two ghost z planes; the halo of a
 * field travels first in t (whole local slices) and then in z (the boundary xy planes of every local slice, ghost slices
 * included, which fills the corners the staples need), through the same three transports.  Slab arrays are the rank's
 * block [Lt/Pt][Lz/Pz][Ly][Lx] in lexicographic order.  Full operator with plain or mixed-precision CG, stout smearing,
 * the even/odd action (needs Lx*Ly % 64 == 0 and even Lz/Pz, Lt/Pt), all integrators and the HMC trajectory; LGT_DD_PUSH is for
 * time slabs only (LGT_EINVAL).
 * grid = {nranks, 1} is a time-slab decomposition whose ranks are their own z neighbours. */
int lgt_dd_create_grid(lgt_dd** out, const int dims[4], const int grid[2], int nlocal, const int* local_ranks, double beta,
                       double kappa, const int bc[4], int precision, int device, void* cuda_stream);
int lgt_dd_destroy(lgt_dd* d);
const char* lgt_dd_last_error(const lgt_dd* d);
/* NCCL transport: rank 0 obtains a 128-byte id (HOST buffer), the caller broadcasts it to all processes (e.g. through
 * torch.distributed), every process calls lgt_dd_nccl_init on its one-rank group.  libnccl.so.2 is opened at run time. */
int lgt_dd_nccl_unique_id(void* id128);
int lgt_dd_nccl_init(lgt_dd* d, const void* id128);
/* Host transport (MPI, gloo, ... -- and the two-processes-on-one-GPU test of the inter-process path): instead of NCCL
 * the caller supplies two callbacks that move HOST memory between the processes; the library stages the time slices
 * through pinned buffers and synchronises the group's stream around each call (correct, not fast).
 *   sendrecv(user, send_buf, send_peer, recv_buf, recv_peer, nbytes): post the two sends (send_buf[k], nbytes bytes, to
 *     rank send_peer[k]) and the two receives (recv_buf[k] from rank recv_peer[k]) IN INDEX ORDER and return when all four
 *     have completed; messages between one pair of ranks must be matched in the order they were posted.  A rank may
 *     be its own peer (nranks = 1), and both peers may be the same rank (nranks = 2).
 *   allreduce(user, buf, count): replace buf[0..count) (count <= 8) by its sum over all ranks, the same bits on every rank.
 * Both return 0 on success.  One rank per process; exclusive with lgt_dd_nccl_init (LGT_ESTATE). */
typedef int (*lgt_dd_sendrecv_fn)(void* user, const void* const send_buf[2], const int send_peer[2], void* const recv_buf[2],
                                  const int recv_peer[2], size_t nbytes);
typedef int (*lgt_dd_allreduce_fn)(void* user, double* buf, int count);
int lgt_dd_set_host_transport(lgt_dd* d, lgt_dd_sendrecv_fn sendrecv, lgt_dd_allreduce_fn allreduce, void* user);
/* The halo plan every transport follows (host-only, no device needed): for rank `rank` of `nranks` slabs of lt_local time
 * slices, plan = {send_peer[2], send_slice[2], recv_peer[2], recv_slice[2]} in issue order; slices are local time-slice
 * numbers of the slab's (lt_local + 2)-slice field (0 and lt_local + 1 are the ghost slices).  Rank r's first interior
 * slice goes to the upper ghost slice of rank r - 1, its last interior slice to the lower ghost slice of rank r + 1.
 * A group that holds one of several ranks and has no transport yet returns LGT_ESTATE from every exchanging call. */
int lgt_dd_halo_plan(int nranks, int rank, int lt_local, int plan[8]);
/* How the halo slices of the CG fields travel:
 *   LGT_DD_EXCHANGE (default): a separate exchange (NCCL send/recv, or device copies between local ranks) before
 *     every Dslash;
 *   LGT_DD_PUSH: fused into the producing kernels -- the Dslash kernels of the CG loop store the results of a slab's
 *     first / last interior slice straight into the neighbour's ghost slice (peer memory), the ghost slices of the
 *     search direction follow by local arithmetic, and the all-reduce that follows each Dslash anyway is the barrier:
 *     no separate transfer inside the iteration.  Same iterates bit for bit.  Between processes the neighbours'
 *     buffers are mapped with CUDA IPC: every rank exports 128 bytes (lgt_dd_ipc_export, HOST buffer), the caller
 *     all-gathers them, every rank imports the handles of ranks r-1 and r+1 (lgt_dd_ipc_import), then switches mode.
 *     Ranks that share a process need no import.  LGT_ESTATE if a neighbour's buffers are not reachable. */
/*   LGT_DD_OVERLAP: the exchange of LGT_DD_EXCHANGE, but issued on a second stream while every slab's bulk (the time slices
 *     that touch no ghost slice) is computed; the two boundary slices are launched once the halo has landed (SURVEY.md 8(e):
 *     "interior/boundary kernel split to overlap").  Inside the CG loop, for time slabs of at least three slices that are
 *     whole 128-site chunks; elsewhere it behaves as LGT_DD_EXCHANGE.  Same iterates bit for bit. */
/*   LGT_DD_HALF: the schedule of LGT_DD_OVERLAP with HALF SPINORS on the wire: the boundary sites are projected
 *     before the send -- and for the backward face also multiplied by U_t^dag -- so that 6 instead of 12 complex numbers per face
 *     site travel, and the boundary slices take that t hop from the received face.  Same iterates bit for bit.
 *   With the even/odd action LGT_DD_OVERLAP and LGT_DD_HALF overlap the halo of every hop's input half field with the bulk of
 *     the slab in the same way (ghost slices, respectively projected / multiplied faces of V3/2 half spinors, on the wire;
 *     V3/2 % 128 == 0, slabs of three or more slices, else the plain exchange). */
enum { LGT_DD_EXCHANGE = 0, LGT_DD_PUSH = 1, LGT_DD_OVERLAP = 2, LGT_DD_HALF = 3 };
int lgt_dd_set_halo_mode(lgt_dd* d, int mode);
int lgt_dd_ipc_export(lgt_dd* d, void* handles128);
int lgt_dd_ipc_import(lgt_dd* d, const void* lo_handles128, const void* hi_handles128);
int lgt_dd_local_ranks(const lgt_dd* d);
lgt_ctx* lgt_dd_rank(lgt_dd* d, int local_index);
/* The decomposed forms of lgt_dslash, lgt_cg, lgt_action, lgt_md_kick, lgt_md_drift, lgt_md_trajectory:
 * same mathematics, same kernels on each slab's interior, sums taken over all ranks; scalar outputs are global. */
int lgt_dd_dslash(lgt_dd* d, const void* const* in, void* const* out, int dagger);
int lgt_dd_cg(lgt_dd* d, const void* const* b, void* const* x, double tol, int max_iter, int* iters, double* rel_resid);
int lgt_dd_action(lgt_dd* d, double tol, int max_iter, double* S_g, double* S_F, double* K, int* cg_iters);
/* lgt_set_solver for the solves inside lgt_dd_action / lgt_dd_md_* / lgt_dd_hmc_trajectory: LGT_SOLVER_MIXED_CG runs the
 * decomposed CG in fp32 (fp32 copies of the links incl. ghost slices) inside an fp64 defect correction on the true,
 * all-reduced residual.  lgt_dd_cg itself is always the plain CG. */
int lgt_dd_set_solver(lgt_dd* d, int solver, double inner_tol);
/* lgt_set_fermion_action for the decomposed lattice: LGT_ACTION_EO runs CG on the Schur complement with the half fields'
 * ghost slices exchanged before every hop; with LGT_SOLVER_MIXED_CG the decomposed fp32 CG on the Schur complement runs
 * inside the fp64 defect correction.
 * Needs even extents, an even number of time slices per slab and Lx*Ly*Lz % 64 == 0, else LGT_EINVAL. */
int lgt_dd_set_fermion_action(lgt_dd* d, int action);
/* lgt_set_smearing for the decomposed lattice: every level's links are built on the slabs' interiors and their ghost
 * slices exchanged before the next level; in the force recursion the ghost slices of G are exchanged before each
 * chain kernel. */
int lgt_dd_set_smearing(lgt_dd* d, int n_levels, double rho);
/* lgt_set_integrator for lgt_dd_md_trajectory and lgt_dd_hmc_trajectory (the same kick / drift sequences). */
int lgt_dd_set_integrator(lgt_dd* d, int integrator, int n_inner);
int lgt_dd_md_kick(lgt_dd* d, double eps, double tol, int max_iter, int* cg_iters);
int lgt_dd_md_drift(lgt_dd* d, double eps);
int lgt_dd_md_trajectory(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, double* H_initial, double* H_final,
                         long* cg_iters);
/* lgt_hmc_trajectory on the decomposed lattice: the heat baths draw by GLOBAL element number, so momenta,
 * pseudofermion, dH and the decision are those of the undivided lattice; every rank takes the same decision from the
 * same all-reduced numbers. */
int lgt_dd_hmc_trajectory(lgt_dd* d, int nsteps, double dt, double tol, int max_iter, unsigned long long seed,
                          unsigned trajectory, double* dH, int* accepted, long* cg_iters, double* H_initial);

/* ---- native-layout spinor fields (for callers that keep fields resident between calls) ---- */
/* Bytes of one spinor field in the handle's internal layout and precision. */
long lgt_native_spinor_bytes(const lgt_ctx* ctx);
/* canonical -> native and back; device pointers, src != dst. */
int lgt_spinor_to_native(lgt_ctx* ctx, const void* canonical, void* native);
int lgt_spinor_from_native(lgt_ctx* ctx, const void* native, void* canonical);
/* out = D in / D^dag in on native-layout device buffers (one kernel launch, nothing else). */
int lgt_dslash_native(lgt_ctx* ctx, const void* in, void* out, int dagger);
/* Pi <- Pi - eps F^f from native-layout X, Y (one launch of the fused force kernel). */
int lgt_fermion_force_native(lgt_ctx* ctx, const void* X, const void* Y, double eps);
/* Pi <- Pi - eps F^g (one launch of the staple kernel). */
int lgt_gauge_force_accumulate(lgt_ctx* ctx, double eps);
/* CG on native buffers; b, x native spinors; also leaves Y = D x in `y` if y != NULL. */
int lgt_cg_native(lgt_ctx* ctx, const void* b, void* x, void* y, double tol, int max_iter,
                  int* iters, double* rel_resid);

/* ---- per-kernel timing (CUDA events on the handle's stream, used by bench.py's roofline line) ---- */
enum { LGT_K_DSLASH = 0,        /* out = D in, D^dag in, and CG step "t = D p" (+ |t|^2) */
       LGT_K_CG_BLAS = 1,       /* CG initialisation, the one-block scalar kernels, precision conversion */
       LGT_K_FERMION_FORCE = 2, LGT_K_GAUGE_FORCE = 3, LGT_K_LINK_UPDATE = 4,
       LGT_K_OTHER = 5,         /* layout conversion, actions */
       LGT_K_DSLASH_R = 6,      /* CG step "q = D^dag t, r -= alpha q" (+ |r|^2), q kept on chip */
       LGT_K_CG_UPDATE = 7,     /* CG step "x += alpha p, p = r + beta p" (one pass over x, p, r) */
       LGT_K_COUNT = 8 };
/* While enabled, every kernel launch is bracketed by a pair of CUDA events. */
int lgt_timing_enable(lgt_ctx* ctx, int enable);
/* Forgets the recorded launches (synchronises the stream). */
int lgt_timing_reset(lgt_ctx* ctx);
/* Synchronises, then returns the summed device time (ms) and the number of launches of one kernel class
 * recorded since the last reset.  Either output may be NULL. */
int lgt_timing_read(lgt_ctx* ctx, int kernel_class, double* ms_total, long* launches);

/* ---- measured roofline denominators ---- */
/* Two microbenchmarks on the handle's device and stream, timed with CUDA events, `launches` timed launches each after
 * two untimed ones: (1) the FMA peak of the handle's precision -- 8 independent FMA chains per thread at full occupancy,
 * 2 flops per FMA, in TFLOP/s; (2) a plain copy of the handle's native link field to a scratch buffer, read + write
 * bytes, in GB/s.  `best` = fastest launch (burst), `mean` = average (sustained: under the power cap the clock drops).
 * Any output may be NULL (both of a pair NULL skips that benchmark). */
int lgt_measure_peaks(lgt_ctx* ctx, int launches, double* fma_tflops_best, double* fma_tflops_mean, double* copy_gbs_best,
                      double* copy_gbs_mean);

/* ---- introspection -------------------------------------------------------------------------- */
/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
long lgt_launch_count(const lgt_ctx* ctx);
/* The stream the handle enqueues on (cudaStream_t as void*). */
void* lgt_stream(const lgt_ctx* ctx);
/* Block traversal order of the Dslash, fermion-force and staple kernels (results are bitwise independent of it).  z_planes = 0: lexicographic;
 * z_planes = Z > 0: blocks sweep all time slices of a slab of Z z-planes before the next slab, which keeps the
 * t neighbours of a site in L2 when one time slice of links + spinors no longer fits;
 * z_planes < 0: automatic (the default chosen by lgt_create).  LGT_EINVAL if Z does not divide Lz or Lx*Ly is
 * not a multiple of 128.  Returns the value in effect through *in_effect (may be NULL). */
int lgt_set_block_swizzle(lgt_ctx* ctx, int z_planes, int* in_effect);
/* Implementation variant of one kernel class (LGT_K_*); every variant computes the same operation and
 * the alternatives stay in the library so that each measurement in profiles/ can be repeated.
 *   LGT_K_DSLASH (covers LGT_K_DSLASH_R; D and D^dag bitwise the same in variants 0-5 and 8-11):
 *     0 = one 128-site block per chunk (dslash_kernel; the default and, measured, the fastest in fp64; for the fp32 kernels
 *         on lattices of 297 ... 16384 chunks the default carries variant 8's prefetch, which gains 4-10 % per fp32 CG iteration);
 *     1 = persistent software-pipelined kernel: one wave of blocks loops over the chunks with the next chunk's first
 *         loads in flight during the current chunk's last hops;
 *     2 = persistent, the forward links brought by bulk copy (cp.async.bulk + mbarrier) into per-warp shared-memory
 *         slots one chunk ahead;
 *     3 = 256-thread blocks on 2 x 2 x 2 tiles of 32-site layout blocks (needs Lx*Ly % 64 == 0, even Lz and Lt,
 *         an undivided lattice; other shapes run variant 0; CG sums differ from variant 0 in rounding);
 *     4 = variant 0 plus an L2 prefetch of the forward links and t+1 spinors of the block 2 x SMs further on;
 *     5 = variant 0 with the z and t neighbours loaded past L1 (ld.global.nc.L1::no_allocate);
 *     6 = variant 0 with the hops reordered so that those whose operands come from DRAM go first (t+, z+, y+, x+, then
 *         the backward ones); the eight contributions are summed in another order, so results agree to rounding only;
 *     8 = variant 0 plus the L2 prefetch of variant 4 issued at the END of each block, about one memory latency before the
 *         block that takes its place starts (so the lines do not sit in L2 long enough to push out the t-neighbours' slice);
 *     9 = persistent kernel with the DRAM-bound operands (the four forward links and the t+1 spinor of a site) requested one
 *         chunk ahead by per-thread cp.async into thread-private shared-memory slots (768 B per thread in fp64);
 *     10 = variant 1 with the chunks after a block's first drawn from a global counter (dynamic instead of strided assignment);
 *     11 = two chunks per block as straight-line code (the first site's tail under the second site's first loads);
 *     7 = 12-real links: rows 0 and 1 of every link are read and row 2 = sign * conj(row0 x row1) is
 *         rebuilt in registers (768 instead of 960 compulsory bytes per site).  Exact for special unitary links; links
 *         that have drifted from unitarity by delta change the operator by O(delta).
 *     12 = variant 7 in the fp32 default's build (fp32 handles and the fp32 inner solve; fp64 runs variant 7): compiled for
 *         three blocks per SM, with the end-of-block L2 prefetch restricted to rows 0 and 1.  384 instead of 480 compulsory
 *         bytes per site, and still slower than the default (32^4: 94-97 against 91 us, CG iteration 303-321 against 274-278 us):
 *         the fp32 kernel is not bound by bytes either.  The fp32 even/odd hop kernels ARE (0.95 of the copy bandwidth), and for
 *         them variant 12 selects the same 12-real links (hop_cb_kernel PFL 2: 32^4 hop 67 -> 59 us).  In the fp32 INNER solve
 *         of the mixed-precision even/odd solver on lattices of more than two waves of blocks that is the DEFAULT -- the fp64
 *         defect correction keeps the exact operator, so links that are not special unitary cost iterations, never accuracy
 *         (even/odd mixed-precision MD step at 32^4 27.9 -> 25.4 ms, same iteration count).  On an fp64 handle variant 12 also
 *         puts the fp64 even/odd hops on 12-real links (plain build; 32^4 even/odd CG 645-660 -> 601-626 us per iteration, same
 *         count, solutions equal to 6e-16) -- opt-in only: exact for special unitary links.
 *   LGT_K_GAUGE_FORCE: 0 = one 32-site layout block x 4 directions per 128-thread block (default, fastest);
 *     1 / 2 = two / four layout blocks per 256- / 512-thread block (more sharing through L1; measured slower).  Same sums bit for bit.
 *     3 = one thread per site: the down staples link by link, the up staples plaquette by plaquette (U_mu(s) U_nu(s+mu)
 *         (U_nu(s) U_mu(s+nu))^dag serves the links (s, mu) and (s, nu)): 46 instead of 52 products per site; measured slower.
 *   LGT_K_CG_BLAS: 0 = the CG scalar updates (alpha; beta, count, stop test) as one-block kernels between the stencil
 *     kernels (default); 1 = fused into the stencil kernels: the block that finishes last forms the same fixed-order sum
 *     and applies the update (two launches fewer per iteration, bitwise the same iterates; measured slower: the fence
 *     and ticket at the end of every block cost more than the two short launches);
 *     2 = the whole even/odd CG (lgt_eo_cg, and the inner fp32 solve of the mixed-precision even/odd solver) as ONE cooperative
 *     launch: the four hops and the x / p update of an iteration are phases separated by grid barriers, every block forms the two
 *     sums itself from the same block partials in the same order (bitwise the same iterates and count; undivided lattices;
 *     the full-operator CG is not affected).  Measured slower at every size from 8^4 to 32^4 (a graph-launched kernel
 *     boundary costs about 1 us on this GPU, a grid barrier with its L1 invalidation more);
 *     3 = even/odd CG with the scalar updates FOLDED into the kernels that follow them, without fence or ticket: block 0 of the
 *     third hop forms pAp and alpha, every block of the x / p update forms |r|^2, beta and the stop decision from the same block
 *     partials in the same fixed order and block 0 writes the next iteration's state into the other of two state records (five
 *     launches per iteration instead of seven; bitwise the same iterates and count; undivided lattices of at most 2048 blocks
 *     per half field, otherwise variant 0 runs).  Measured: 8^4 26.2 -> 24.9 us per iteration, but 16^4 fp32 29.9 -> 32.6 and
 *     24^4 fp32 122.8 -> 126.4: the sum at the head of every block of the update costs more than two 2 us launches in a graph.
 * variant < 0 only queries.  The value in effect is returned through *in_effect (may be NULL).
 * LGT_EINVAL for an unknown class or variant. */
int lgt_set_kernel_variant(lgt_ctx* ctx, int kernel_class, int variant, int* in_effect);

/* ---- an entry point that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).
 *
 * The plaquette action (BASELINE.json configs[0]) of a link field the CALLER holds, without a handle:
 *   out[0] = S_g = beta sum_x sum_{mu<nu} (1 - Re tr U_P(x) / 3),   out[1] = (1 / 6V) sum_x sum_{mu<nu} Re tr U_P(x) / 3
 * -- the numbers lgt_action (S_g) and lgt_plaquette return for the same links.
 *   dims, beta : lattice extents (x, y, z, t; each >= 1, periodic links) and coupling.
 *   precision  : LGT_F64 or LGT_F32, the element type of U (the sums are always formed in double).
 *   device     : CUDA device ordinal (0 ... 63) that owns U, out and the stream; made current for the call and restored.
 *   U          : DEVICE pointer, canonical layout [V][4][3][3] complex (re, im), read only; caller-owned.
 *   out        : DEVICE pointer to two doubles, written by the kernel; caller-owned.  Nothing is copied to the host and the
 *                call does not synchronise: read `out` after the stream has reached this point.
 *   cuda_stream: cudaStream_t (or NULL for the default stream); the call enqueues one 256-byte memset and one kernel on it.
 * The scratch of the reduction (one double per block of 128 sites, and the ticket counter) is a file-scope __device__ array
 * of 1 MiB + 256 B inside the library, which every GPU that loads liblgt.so holds until the process exits; its device address
 * is looked up on the first call per device (cudaGetSymbolAddress -- make that first call outside a graph capture), after
 * which the call uses no cudaMalloc, cudaFree or allocating library routine.  Limit: V <= LGT_NOALLOC_MAX_SITES (2^24 sites:
 * every BASELINE.json configuration incl. 48^3 x 96 fits); larger lattices are rejected with LGT_EINVAL.
 * Every call on a device shares the one array: calls that OVERLAP on the GPU (two streams, two threads, two graphs in flight)
 * race on it and return garbage; calls ordered on one stream are safe (the counter is cleared at the start of every call, the
 * partials are overwritten before they are read).  The result is bitwise reproducible from call to call.
 * Errors: LGT_EINVAL (null pointer, bad precision / device / extent, too many sites), LGT_ECUDA; the text is returned by
 * lgt_noalloc_last_error() (per host thread; static storage, never freed by the caller). */
#define LGT_NOALLOC_MAX_SITES 16777216
int lgt_plaquette_action_noalloc(const int dims[4], double beta, int precision, int device, const void* U, double* out,
                                 void* cuda_stream);
const char* lgt_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
