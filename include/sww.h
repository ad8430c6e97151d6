/*
 * sww.h -- C ABI of the B200-native Dirichlet-to-Neumann (DtN) hot path of
 * Wilkening & Yu, "Overdetermined shooting methods for computing standing water waves with spectral accuracy"
 * (arXiv 1210.5672).  Citations are PAPER.md:<line> (+ section / equation); readings R1.. are listed in DESIGN.md section 3.
 *
 * Scope: the spectrally accurate boundary-integral DtN operator of Appendix A / section 2.1-2.2 on a uniform grid
 * alpha_j = 2 pi j / N over a flat bottom, its linearization (Appendix B), and the explicit Runge-Kutta stepper of the
 * free-surface Euler equations (2.1) with the batched variational equation (3.32).
 *
 * Conventions (all entry points)
 *   - Every pointer named DEVICE is a CUDA device pointer valid on the current device; nothing is copied from the host
 *     except by the *_host convenience calls at the bottom, which are explicitly marked HOST.
 *   - A batch of nrhs columns of N reals is column-major N x nrhs: column c starts at element offset c*N.
 *   - prec = SWW_F64: one double per element.
 *     prec = SWW_DD : double-double ("quadruple"), PLANAR layout: an array of L logical elements is 2L doubles,
 *                     hi[0..L) followed by lo[0..L), value = hi + lo with |lo| <= ulp(hi)/2.  (L = N*nrhs for a batch.)
 *   - h, g, dt are plain doubles.  h = INFINITY selects infinite depth (image kernels dropped).
 *   - eta is the elevation about the mean level; the bottom is y = 0 and the surface is y = h + eta_j (R2).
 *   - Work is enqueued on the CUDA stream given at creation; calls return without synchronising unless stated.
 *     Data-dependent failures (SWW_EBOTTOM, SWW_ESINGULAR) are recorded in a device flag and returned by the next
 *     synchronising call (sww_dtn_status, sww_state_read).
 *   - The caller owns every in/out buffer; handles own everything else.  Functions never throw or exit; they return a status.
 *   - N must be a power of two.  Size limits per entry point (checked up front, before anything is allocated; SWW_EINVAL):
 *         sww_dtn_* with SWW_F64 ............ 16 <= N <= 8192
 *         sww_dtn_* with SWW_DD ............. 16 <= N <= 4096   (one N-point complex double-double array per CTA in shared memory)
 *         sww_state_* with SWW_F64 .......... 16 <= N <= 4096   (two N-point complex arrays per CTA)
 *         sww_state_* with SWW_DD ........... 16 <= N <= 2048   (two N-point complex double-double arrays per CTA)
 *     Mesh refinement (2.10)-(2.11) and sizes that are not powers of two are not built.
 */
#ifndef SWW_H
#define SWW_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sww_dtn_s*   sww_dtn_t;   /* one surface: K, G, LU(I/2+K), node tables, base state, workspace (device)  */
typedef struct sww_state_s* sww_state_t; /* time-stepper state: eta, phi, optional variational columns, RK stage storage */
typedef struct sww_shooter_s* sww_shooter_t; /* the shooting map: a stepper with n variational columns + the unknowns c */

enum { SWW_F64 = 0, SWW_DD = 1 };
enum {
    SWW_OK = 0,
    SWW_EINVAL = -1,    /* bad argument (N not a power of two in range, nrhs < 0, null pointer, unknown prec)           */
    SWW_ENOMEM = -2,    /* device or host allocation failed                                                           */
    SWW_ECUDA = -3,     /* a CUDA runtime call failed; sww_last_cuda_error() has the text                             */
    SWW_EBOTTOM = -4,   /* some h + eta_j <= 0: the surface touches the bottom                                         */
    SWW_ESINGULAR = -5, /* a pivot of the unpivoted LU fell below the guard (|U_ii| < 1e-3): I/2+K is not benign here  */
    SWW_ENOBASE = -6,   /* sww_dtn_linearized_apply before sww_dtn_set_base                                            */
    SWW_ETOOBIG = -7    /* a size beyond the fixed scratch of a no-allocation entry point; sww_last_cuda_error() has the text */
};

/* ---- DtN operator of one surface -------------------------------------------------------------------------------
 * sww_dtn_setup: steps S0-S2 of DESIGN.md.
 *   S0  eta', eta'' = D eta, D(D eta) by spectral differentiation carried in double-double (R8);
 *   S1  K_ij, G_ij for all i, j from (2.13) with the image kernels SUBTRACTED (R1: (A.2),(A.3),(A.8),
 *       PAPER.md:637-663), diagonal entries from the limits of PAPER.md:150, 653, 673;
 *   S2  LU factorisation of A = I/2 + K (the matrix of (2.7); "LU-factorization"), unpivoted
 *       (DESIGN.md section 5 justifies: sigma(A) in [0.46, 1.01]) with a |U_ii| guard -> SWW_ESINGULAR.
 * eta: DEVICE, N reals (layout by prec), read during the call's enqueued work; may be reused after the stream reaches it.
 * stream: a cudaStream_t cast to void* (NULL = legacy default stream).  *out receives the handle. */
int sww_dtn_setup(const void* eta, int N, double h, int prec, void* stream, sww_dtn_t* out);

/* Re-run S0-S2 for a new surface of the same N, h, prec in an existing handle (no allocation; what every RK stage does). */
int sww_dtn_refactor(sww_dtn_t d, const void* eta);

/* out_c = G(eta) phi_c, c < nrhs: solve (I/2 + K) mu_c = phi_c (2.7); gamma_c = D mu_c; out_c = H gamma_c / 2 + G gamma_c (2.8)
 * (1/|xi'| = 1 on the uniform grid, R3).  phi, out: DEVICE, N x nrhs; may alias.  Pure: no hidden state.
 * A non-finite input column gives a non-finite output column, spoils the column it shares a complex FFT with (2c and 2c + 1)
 * and leaves all others untouched.  (The triangular solves mark "not computed yet" in their scratch by the all-ones NaN
 * 0xFFFFFFFFFFFFFFFF; an input with exactly that payload is replaced by the canonical quiet NaN on the way in, so it behaves
 * like any other NaN.  Should a task ever wait for data beyond ~0.1 s, it records the sticky status SWW_ECUDA and every other
 * task stops polling at once.) */
int sww_dtn_apply(sww_dtn_t d, const void* phi, int nrhs, void* out);

/* Store the state the linearization is taken about: phi0' = D phi0, W0 = G phi0, and the surface velocities of (2.9)
 * (PAPER.md:116): u = (phi0' - eta' W0)/(1+eta'^2), v = (eta' phi0' + W0)/(1+eta'^2).  phi0: DEVICE, N reals. */
int sww_dtn_set_base(sww_dtn_t d, const void* phi0);

/* out_c = d/de G(eta + e deta_c)[phi0 + e dphi_c] at e = 0 = G[dphi_c - v deta_c] - D(u deta_c)   ((B.1d),(B.2)).
 * deta, dphi, out: DEVICE, N x nrhs.  Needs sww_dtn_set_base first (else SWW_ENOBASE). */
int sww_dtn_linearized_apply(sww_dtn_t d, const void* deta, const void* dphi, int nrhs, void* out);

/* Right-hand side of the adjoint system (B.6) (it serves the adjoint continuation method) at the
 * state the handle holds (surface set up, sww_dtn_set_base done: u = phi_x, v = phi_y on the surface), for nrhs adjoint vectors:
 *     chi_c    = eta~_c + v P phi~_c                                                                               (B.6d)
 *     phi_s,c  = G chi_c + D(u P phi~_c)                                                                           (B.6e)
 *     eta_s,c  = -v G chi_c + u D eta~_c - v D(u) P phi~_c - g P phi~_c + sigma D( D(phi~_c) / (1 + eta'^2)^(3/2) )   (B.6f)
 * (unfiltered, like the identity <DF(q) qdot, q~> = <qdot, DF(q)^* q~> it satisfies).  eta_t, phi_t, eta_s, phi_s: DEVICE, N x nrhs,
 * four distinct buffers (SWW_DD: planar hi block then lo block each, N <= 2048).  Needs sww_dtn_set_base (else SWW_ENOBASE). */
int sww_dtn_adjoint_rhs(sww_dtn_t d, const void* eta_t, const void* phi_t, int nrhs, double g, double sigma, void* eta_s, void* phi_s);

/* Read-only views for tests and diagnostics.  which: 0 = K, 1 = G (column-major N x N: entry (i,j) at i + j*N, i = target
 * alpha_i, j = source alpha_j; DD: planar hi then lo), 2 = eta' , 3 = eta'', 4 = phi0', 5 = W0, 6 = u, 7 = v (N reals each),
 * 8 = the fp64 factors of I/2 + K as lu.cu stores them (N x N doubles for either precision: L_ij = X_ij inv(S_j) below the block
 * diagonal, U_ij above it, the raw diagonal tiles of K on it).
 * dst: DEVICE buffer of the right size; the copy is enqueued on the handle's stream. */
int sww_dtn_get(sww_dtn_t d, int which, void* dst);

int sww_dtn_status(sww_dtn_t d);   /* synchronises the stream; returns the sticky status */
int sww_dtn_destroy(sww_dtn_t d);

/* ---- time stepper (2.1) + variational equation (3.32), PAPER.md:70-72, 294-305, 689-714 ------------------------
 * sww_state_create copies the initial state (DEVICE pointers; deta/dphi may be NULL when ncols = 0).  prec = SWW_DD: every
 * array is double-double planar (eta, phi: 2N doubles; deta, dphi: 2 N ncols doubles, hi block then lo block), and the whole
 * step -- DtN, right-hand sides, FFTs, filter, stage combination with the tableau in double-double -- runs in double-double
 * (the paper's quadruple-precision time stepping).
 * flags bit 0: switch the 36th-order filter (2.14) off (R5).
 * sww_rk_advance: nsteps steps of size dt of the 11-stage order-8 explicit Runge-Kutta scheme (R6), one setup S0-S2 and
 * one batched linearized solve per stage, state filtered after each step; advances (q, Qdot) together, in place.
 * sww_state_read: DEVICE destinations (any may be NULL); synchronises; *t (HOST) receives the elapsed time; returns the
 * sticky status. */
int sww_state_create(int N, double h, double g, int prec, int ncols, const void* eta, const void* phi,
                     const void* deta, const void* dphi, unsigned flags, void* stream, sww_state_t* out);
int sww_rk_advance(sww_state_t s, double dt, int nsteps);
/* The same advance by the 15th-order spectral deferred correction scheme the paper uses in quadruple precision:
 * 8 Radau IIa nodes per step, initial values at the nodes by classical RK4 from node to node, 10 Picard sweeps
 * Y_m <- y_n + dt sum_j S_mj F(Y_j) with the integration matrix of the nodes, then y_{n+1} = y_n + dt sum_j b_j F(Y_j)
 * (R15; 113 right-hand sides per step, each one setup + one batched linearized solve); filter as in sww_rk_advance.
 * Either precision; the first call allocates 22 more state vectors in the handle. */
int sww_sdc_advance(sww_state_t s, double dt, int nsteps);
/* Surface tension sigma / rho >= 0 of (2.1b) (0 by default, 1 in section 4.6): from the next step on
 *   phi_t  += P[ sigma D( eta' / sqrt(1 + eta'^2) ) ],   dphi_t += P[ sigma D( D(deta_c) / (1 + eta'^2)^(3/2) ) ]   (B.4)
 * (filtered like the other terms).  With h = infinity and g = sigma = 1 the linear period is 2 pi / sqrt 2 (4.42). */
int sww_state_set_sigma(sww_state_t s, double sigma);
int sww_state_read(sww_state_t s, void* eta, void* phi, void* deta, void* dphi, double* t);
/* E = (1/2) int (phi G phi + g eta^2) dx = (pi/N) sum_j [phi_j (G phi)_j + g eta_j^2] of the current state;
 * energy_hl: HOST, 2 doubles (hi, lo; lo = 0 for SWW_F64); synchronises.  The handle's internal DtN is re-set-up for the current
 * state (one setup + base state). */
int sww_state_energy(sww_state_t s, double* energy_hl);
int sww_state_destroy(sww_state_t s);

/* ---- mesh refinement in space, section 2.2 (2.10)-(2.11), PAPER.md:122-136 ------------------------------------------------
 * The change of variables x = xi(alpha):  xi' = E = 1 - P[A sin^4(alpha/2)] (where = 0: refine near x = pi) or 1 - P[A cos^4(alpha/2)]
 * (where = 1: refine near x = 0), A = 8 (1 - rho) / (5 + 3 rho), 0 < rho <= 1 the ratio of the smallest to the largest spacing (2.11);
 * rho = 1 is the uniform mesh.  After sww_dtn_set_mesh every array of the handle (eta, phi, the columns, every output) holds values at
 * the points x_j = xi(alpha_j), alpha_j = 2 pi j / N: zeta = xi + i eta o xi in (2.13), the factor 1/|xi'| in (2.8), d/dx =
 * (1/xi') d/dalpha in (2.9), (B.2).  The call invalidates the surface: follow it with sww_dtn_refactor.  Views 2, 3 of sww_dtn_get stay
 * alpha-derivatives of the stored eta; 4..7 (phi0', W0, u, v) are the physical quantities.  Either precision.
 * sww_dtn_adjoint_rhs follows the mesh as well ((B.6) with d/dx and the mean over x); sww_dtn_linearized_host is uniform only.
 * sww_mesh_points: x (HOST, N doubles) <- xi(alpha_j). */
int sww_dtn_set_mesh(sww_dtn_t d, double rho, int where);
int sww_mesh_points(int N, double rho, int where, double* x);
/* The time stepper on a refined mesh (either precision, RK8 or SDC15): the filter (2.14) acts on the stored
 * samples, P removes the mean over x, (1/N) sum_j f_j xi'(alpha_j) (the trapezoidal rule with dx = xi' dalpha), and the
 * energy integral carries the same weight.  Call before advancing; the state's arrays are then values at x_j.
 * sww_state_respace: dst's state (eta, phi and all columns) <- src's, interpolated to dst's mesh: beta_j =
 * xi_src^{-1}(xi_dst(alpha_j)) by Newton's method in double-double, values at beta_j from the trigonometric interpolant of src's samples
 * (one M_dst x M_src matrix applied to all 2 + 2 ncols columns at once; kept in dst for the next call with the same pair of meshes).
 * dst and src: two handles of the same precision with the same ncols and any two sizes and meshes (SWW_DD: the matrix and the
 * product in double-double); dst's elapsed time becomes src's.  Synchronises both streams. */
int sww_state_set_mesh(sww_state_t s, double rho, int where);
int sww_state_respace(sww_state_t dst, sww_state_t src);
/* The same respacing for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): out (M_new x ncol) <- the ncol columns f (M_old x ncol, fp64, column c at c * M) given on the mesh (rho_old, where_old)
 * with M_old points, interpolated to the mesh (rho_new, where_new) with M_new points (the arithmetic of sww_state_respace for SWW_F64
 * states; the interpolation matrix is not stored, its entries are formed where they are used).  f, out: DEVICE, distinct.  No handle.
 * The call makes no cudaMalloc / cudaFree and calls no allocating routine: its scratch (4 M_new doubles) is a fixed device array inside
 * the library, 128 KB held by every GPU that loads it until exit.  Limits: M_new <= SWW_RESPACE_NOALLOC_MAX (beyond: SWW_ETOOBIG, text
 * in sww_last_cuda_error()), M_old even, 4 <= M_old <= 8192; neither size needs to be a power of two.  Two kernels are enqueued on
 * `stream`; nothing synchronises.  The first call on each device looks the array's address up (cudaGetSymbolAddress): make it before a
 * graph capture starts.  ALL calls share the one array, which keeps the last call's contents (every entry a call reads it has written
 * first, nothing needs clearing): calls that overlap on the GPU (different streams, no ordering between them) race on it -- order them. */
#define SWW_RESPACE_NOALLOC_MAX 4096
int sww_respace_noalloc(int M_old, double rho_old, int where_old, int M_new, double rho_new, int where_new, int ncol, const double* f,
                        double* out, void* stream);

/* ---- shooting map of the overdetermined shooting method, uniform mesh (section 3.1 / 3.3) ------------------------
 * Unknowns c (HOST, n + 1 doubles): c[0] = T, the period (3.16); c[k], 1 <= k <= n, the Fourier modes of the initial
 * state (3.15): eta(x, 0) = sum_{k even} 2 c_k cos kx, phi(x, 0) = sum_{k odd} 2 c_k cos kx (eta about the mean level).
 * sww_shoot builds that state and the columns dq0/dc_k on the device, advances (q, Qdot) together by nsteps RK8 steps of size
 * T / (4 nsteps) (3.32; one setup + one batched linearized solve per stage) and returns
 *     r_i  = phi(alpha_i, T/4) / sqrt(N)                                                  (3.17; f = r.r / 2)
 *     J_ik = dr_i/dc_k: k >= 1 the variational solution phidot_k(alpha_i, T/4) / sqrt(N), k = 0 phi_t(alpha_i, T/4) / (4 sqrt(N))
 *                                                                                         (3.31; R13)
 * r: DEVICE, N; J: DEVICE, N x (n + 1) column-major; eta_T4, phi_T4 (optional, DEVICE, N): the state at T/4.  SWW_DD: every
 * output is double-double planar (hi block, lo block); c stays fp64.  Limits: those of sww_state_create, and 2 n < N.
 * The handle keeps the stepper and its DtN between calls (a Levenberg-Marquardt iteration calls sww_shoot repeatedly, App. C);
 * flags as in sww_state_create.  sww_shoot synchronises and returns the sticky status. */
int sww_shooter_create(int N, int n, double h, double g, int prec, unsigned flags, void* stream, sww_shooter_t* out);
int sww_shoot(sww_shooter_t S, const double* c, int nsteps, void* r, void* J, void* eta_T4, void* phi_T4);
int sww_shooter_destroy(sww_shooter_t S);
/* The residual alone (a stepper without variational columns inside the handle: what Levenberg-Marquardt needs for a trial step). */
int sww_shoot_residual(sww_shooter_t S, const double* c, int nsteps, void* r);
int sww_shooter_dims(sww_shooter_t S, int* N, int* n, int* is_dd);
/* The mesh-refinement strategy of section 2.2 for every following shot: nu segments (1 <= nu <= 8; 0 returns to one
 * uniform segment); segment l takes nsteps[l] steps of size theta[l] (T/4) / nsteps[l] on M[l] points of the mesh (rho[l], where[l]) of
 * sww_dtn_set_mesh, and the state with all columns is respaced from l to l + 1 (sww_state_respace).  M[0] = N and rho[0] = 1 (the
 * initial state (3.15) lives on the uniform mesh), sum(theta) = 1.  The residual then has m = M[nu-1] entries,
 *     r_i = phi(xi_nu(alpha_i), T/4) sqrt(E_nu(alpha_i) / M_nu)      (3.17)
 * and J is m x (n + 1); sww_shooter_dims reports m as N; the nsteps argument of sww_shoot, sww_shoot_residual and sww_lm_shoot is
 * ignored.  Either precision (SWW_DD with sww_shooter_set_method(S, 1) is the paper's quadruple-precision configuration of Table 3).
 * All arrays HOST.  Creates the steppers of segments 2..nu (memory: like nu shooters). */
int sww_shooter_set_segments(sww_shooter_t S, int nu, const int* M, const double* theta, const double* rho, const int* where, const int* nsteps);
/* The gradient of f = r.r / 2 with respect to c by ONE backward solve of the adjoint system, section 3.2 (3.21)-(3.30), PAPER.md:228-284:
 * forward solve of (2.1) with the stage states kept, then the transposed Runge-Kutta recursion with DF(Y)^* of (B.6)
 * (sww_dtn_adjoint_rhs) at every stage state, q~(0) = (0, phi(T/4)) (3.26); df/dc_k = <q~(T/4), dq_0/dc_k> (3.30), df/dT by (3.22).
 * Cost: two solves of (2.1) instead of the n variational columns of sww_shoot; grad equals J^T r of sww_shoot up to the (spectrally
 * small) difference between the continuous adjoint (B.6) and the transpose of the discrete linearization.  f (optional) and grad
 * (n + 1 doubles): HOST.  SWW_F64 shooters on one uniform segment with the RK8 stepper; otherwise SWW_EINVAL.  Synchronises. */
int sww_shoot_gradient(sww_shooter_t S, const double* c, int nsteps, double* f, double* grad);
int sww_shooter_set_method(sww_shooter_t S, int method);   /* 0: RK8 (default); 1: SDC15, the paper's quadruple-precision stepper */
int sww_shooter_set_sigma(sww_shooter_t S, double sigma);   /* surface tension of every following shot (see sww_state_set_sigma) */

/* ---- Levenberg-Marquardt with delayed Jacobian updates (Appendix C) ----------------------------
 * min f(c) = r(c).r(c) / 2 over the unknowns that are not held fixed (fixed[k] != 0 keeps c[k]: "holding c_1 constant",
 * PAPER.md:334).  Trust-region step from the thin SVD J = U S V^T (C.3) with the O(m) Newton iteration (C.5) on the Lagrange
 * multiplier; radius update, acceptance, roundoff regime and the rules for re-using J as in rules 1-4 of the appendix
 * (rho_0 = 1/4, rho_1 = 0.85, alpha_0 = 3/8, alpha_1 = 1.875, alpha_2 = 0.2).  HOST algebra in fp64 (long-double sums) on an
 * M x m matrix; every r and J comes from the callback.  sww_lm_shoot runs it on the device shooting map (M = N, unknowns c of
 * sww_shoot; residual-only trial steps through sww_shoot_residual).  c: HOST, in/out. */
typedef int (*sww_lm_fun)(void* ctx, const double* c, int want_J, double* r, double* J);   /* J: M x ntot column-major */
typedef struct {
    double f_tol, g_tol, df_tol;   /* rule 1 (the paper: 1e-26, 1e-13, 1e-5) */
    double delta0;                 /* initial trust-region radius (<= 0: 1) */
    double lambda_tol;             /* tolerance of (C.5) (<= 0: 1e-12) */
    int max_stepsJ, max_iter;      /* rule 1 (the paper: 10); iteration limit (<= 0: 10, 100) */
} sww_lm_options;
typedef struct {
    double f, delta;
    int iterations, residual_evals, jacobian_evals;
    int status;                    /* 0 iteration limit, 1 f = 0, 2 c unchanged, 3 roundoff regime ended */
} sww_lm_report;
int sww_lm_minimize(sww_lm_fun fun, void* ctx, int M, int ntot, double* c, const int* fixed, const sww_lm_options* opt, sww_lm_report* rep);
int sww_lm_shoot(sww_shooter_t S, double* c, const int* fixed, int nsteps, const sww_lm_options* opt, sww_lm_report* rep);

/* ---- diagnostics ---------------------------------------------------------------------------------------------- */
const char* sww_strerror(int status);
const char* sww_last_cuda_error(void);
/* Number of kernels this library has launched since it was loaded (bench.py reports the count per step). */
unsigned long long sww_launch_count(void);
/* Per-kernel-class device timing for bench.py's roofline block.  sww_timing_enable(1): from now on every kernel launch of
 * this library is bracketed by a CUDA event pair on its stream (diagnostic mode: costs two event records per launch; not
 * thread-safe).  sww_timing_read synchronises those events, adds up elapsed milliseconds and launch counts per class since
 * the previous read and clears the list.  ms, launches: HOST arrays of nclass >= 8 entries; classes: 0 = K/G assembly (S1),
 * 1 = LU factorisation (persistent DMMA dataflow kernel, S2), 2 = FP64 DMMA GEMM (G product, S6),
 * 3 = FFT / spectral (S5, S7), 4 = double-double matrix products (EFT kernels), 5 = everything else (streaming),
 * 6 = multi-right-hand-side triangular solves (persistent DMMA dataflow kernel, 16- and 32-column slabs, S4),
 * 7 = the same kernel's 8-column instantiation (batches of <= 64 columns: the single-vector solves of the base state). */
int sww_timing_enable(int on);
int sww_timing_read(double* ms, unsigned long long* launches, int nclass);
/* Microbenchmarks used to measure the roofline denominators on the box: returns achieved FLOP/s of a
 * register-resident DFMA loop (which = 0) or DMMA.8x8x4 loop (which = 1) over the whole chip, timed with CUDA events. */
int sww_probe_fp64_peak(int which, double* flops_per_s);

/* ---- HOST-buffer convenience path (what bench.py's "e2e" leg times) -------------------------------------------
 * Same computation as setup + set_base + linearized_apply, but every array is a HOST pointer (pinned or pageable);
 * the call copies inputs to the device, runs the device path, copies the result back and synchronises.  The library keeps ONE
 * cached context (handle + device staging buffers) between calls, reused while N and prec stay the same (a caller stepping a
 * surface calls this once per stage); it runs on the default stream (the batch columns are uploaded on an internal second
 * stream while setup and base state run, so pinned host buffers make the upload free) and is not thread-safe.  sww_host_cache_clear() frees the
 * cached context (it is also dropped after any failing call). */
int sww_dtn_linearized_host(const void* eta, const void* phi0, const void* deta, const void* dphi, void* out,
                            int N, double h, int prec, int nrhs);
int sww_host_cache_clear(void);

#ifdef __cplusplus
}
#endif
#endif /* SWW_H */
