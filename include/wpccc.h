/* wpccc.h -- C ABI of the B200-native WP-CCC hot path (arXiv 2403.04252).
 *
 * The library evaluates, at every projectile position R(t) = (b, 0, v t) of many straight-line
 * trajectories, the coupling matrix elements of the two-centre close-coupling equations
 * (eq. (1)) and advances the amplitudes by classical RK4 (Algorithm 1,
 * PAPER.md L69-104).  Citations "P:Lnnn" are lines of /root/reference/PAPER.md; "A<n>" are the
 * readings of the paper listed in DESIGN.md (section "Readings").
 *
 * Conventions common to every entry point
 *   - Plain pointers and sizes only.  Each pointer argument is marked [host] or [device].
 *   - The library NEVER allocates device memory (no cudaMalloc / cudaMallocAsync anywhere): the
 *     caller owns the basis arena, the workspace and every output buffer.  A pointer is borrowed
 *     for the duration of the call, except the arena, which the basis handle keeps using until
 *     wpccc_free_basis() (it also holds 1 MiB of index scratch for wpccc_probabilities).
 *   - All device work is enqueued on the caller's CUDA stream (`stream` is a cudaStream_t passed
 *     as void*; NULL = legacy default stream).  wpccc_propagate additionally forks onto two
 *     internal streams and joins them back, also on every error path, before it returns.
 *     Calls are asynchronous with respect to the host unless stated otherwise.
 *   - A basis handle is NOT re-entrant: it carries per-call state (timing events, the status of
 *     the last propagation, its two internal streams, the options).  One call at a time per
 *     handle, from one host thread; use one handle per concurrent caller.  The entry points take
 *     `const wpccc_basis *` because they never change the staged basis itself.
 *   - Complex numbers are interleaved double[2] = (re, im).  All arithmetic is IEEE fp64.
 *   - Return value: 0 on success, a negative WPCCC_E* code otherwise; wpccc_last_error() gives a
 *     thread-local message.  There is no CPU fallback: without a CUDA device every compute call
 *     returns WPCCC_ECUDA.
 *   - State ordering (binding): centre T then centre P; inside a centre the radial functions in
 *     caller order; each radial function expands to m = -l .. +l ascending.
 *   - Geometry (A.1): target nucleus at the origin, projectile at (b, 0, z), velocity v along +z.
 *     wpccc_matrix_elements accepts b >= 0 (with R > 0); wpccc_propagate and the cross sections of
 *     wpccc_probabilities need b > 0.  Atomic units.
 */
#ifndef WPCCC_H
#define WPCCC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WPCCC_OK          0
#define WPCCC_EINVAL     (-1)  /* bad argument (message says which)                               */
#define WPCCC_ENOMEM     (-2)  /* arena or workspace too small                                     */
#define WPCCC_ECUDA      (-3)  /* CUDA runtime error / no device                                   */
#define WPCCC_ESINGULAR  (-4)  /* overlap system of some trajectory not factorisable (see propagate) */

#define WPCCC_INIT_FROM_DC (-1) /* init_state of wpccc_propagate: start from the amplitudes already in dC */

typedef struct wpccc_basis wpccc_basis; /* opaque */

/* One expansion centre: bound eigenstates plus wave-packet pseudostates tabulated on the
 * uniform radial grid r_k = k h, k = 0..Nr ("precomputed and stored"; A7).  All arrays [host]. */
typedef struct {
    double        Z;      /* nuclear charge of this centre (H: 1, He2+: 2)                         */
    int           n_rad;  /* number of radial functions                                            */
    const int    *l;      /* [n_rad] orbital angular momentum                                      */
    const double *eps;    /* [n_rad] energies eps_a (a.u.), used in the phases e^{i(eps'-eps)z/v}  */
    const int    *kind;   /* [n_rad] 0 = bound eigenstate, 1 = wave packet (labels for classes)    */
    const int    *nq;     /* [n_rad] principal quantum number or bin index (labels only)           */
    const double *u;      /* [n_rad][Nr+1] reduced radial function u_a(r_k) = r f_a(r), u(0) = 0   */
    const double *g;      /* [n_rad][Nr+1] residual (H_c - eps_a) u_a (A5); NULL = all zero        */
} wpccc_centre;

/* Fixed product rule for the two-centre integrals of eq. (9) in the body frame.
 * kind 0 (BASELINE.json configs[1], [3]; A10): Gauss-Legendre in cylindrical coordinates (rho', phi', z'):
 *   rho' one panel on [0, rho_max] (n_rho nodes); phi' one panel on [0, 2 pi] (n_phi nodes);
 *   z' three panels [-z_pad, 0], [0, R], [R, R + z_pad] with n_z/4, n_z/2, n_z/4 nodes.
 *   n_z must be a multiple of 16, n_rho >= 1, n_phi >= 1.
 *   phi_rule 0: the discrete n_phi-node sum.  phi_rule 1: the continuum azimuthal integral
 *   (-+i)^Delta J_Delta(x) of eq. (9), evaluated by a 512-node periodic trapezoid rule
 *   (exact to rounding for x + |Delta| < 400).
 * kind 1 (the paper's own rule): prolate spheroidal coordinates
 *   r_T = R (eta + tau)/2, r_P = R (eta - tau)/2: n_rho-point Gauss-Laguerre rule in eta, with
 *   x = eta_scale (R/2)(eta - 1), n_z-point Gauss-Legendre rule in tau on [-1, 1] (n_z a multiple of 16), analytic
 *   azimuthal integral (-+i)^Delta J_Delta (Bessel functions by backward recurrence); n_phi, phi_rule, rho_max, z_pad
 *   are ignored.  No mirror pairing. */
typedef struct {
    int    n_rho, n_phi, n_z;
    double rho_max, z_pad;
    int    phi_rule;
    int    kind;        /* 0 cylindrical Gauss-Legendre, 1 spheroidal Gauss-Laguerre x Gauss-Legendre */
    double eta_scale;   /* kind 1: decay constant of the Laguerre weight e^{-eta_scale (r_T + r_P - R)/2}, > 0 */
} wpccc_quad;

/* ---- a0: staging ("stored in the GPU global memory") ------------ */

/* Bytes of device arena wpccc_setup_basis needs for this problem (0 on invalid arguments). */
size_t wpccc_basis_bytes(int n_centres, const wpccc_centre *centres /*[host]*/, int Nr, int lambda_max,
                         const wpccc_quad *quad /*[host] or NULL*/);

/* Copies the host tables, builds the position-independent tables (angular coefficients of eq. (6),
 * pair-product matrix w_k u_a'(r_k) u_a(r_k) for eq. (7), interpolation tables, Gauss-Legendre
 * nodes) into `dev_arena` [device, arena_bytes, 256-byte aligned] and returns a handle.
 *   n_centres 1: target centre only (eq. (5): S = I, H = D^T);  2: target then projectile.
 *   Z_proj: charge seen by target-centred states; with two centres it must equal centres[1].Z.
 *   h, w[Nr+1] [host]: grid step and quadrature weights of the radial grid (A7, A8); w[0] ignored.
 *   lambda_max: largest multipole in eq. (6).
 * Host arrays are copied before return (the call synchronises `stream`).  The handle itself is
 * host memory owned by the library; free it with wpccc_free_basis (the arena stays the caller's). */
int wpccc_setup_basis(wpccc_basis **out, int n_centres, const wpccc_centre *centres /*[host]*/,
                      double Z_proj, int Nr, double h, const double *w /*[host]*/, int lambda_max,
                      const wpccc_quad *quad /*[host]; NULL iff n_centres == 1*/,
                      void *dev_arena /*[device]*/, size_t arena_bytes, void *stream);
/* The same on a non-uniform radial grid r[0] = 0 < r[1] < ... < r[Nr] [host] ("The grid is denser around the origin";
 * SURVEY.md 8(f) NEXT-3): u, g and w are tabulated on these points (w: the caller's quadrature weights, e.g. trapezoid
 * (r[k+1] - r[k-1])/2).  Eq. (7) sums over the given points; the five-point interpolation of the two-centre node tables takes
 * the grid point nearest to r (the lower one on a tie) as stencil centre, clamped to [2, Nr - 2], with Lagrange weights on the
 * actual abscissae; functions vanish beyond r[Nr]. */
int wpccc_setup_basis_grid(wpccc_basis **out, int n_centres, const wpccc_centre *centres /*[host]*/,
                           double Z_proj, int Nr, const double *r /*[host]*/, const double *w /*[host]*/, int lambda_max,
                           const wpccc_quad *quad /*[host]; NULL iff n_centres == 1*/,
                           void *dev_arena /*[device]*/, size_t arena_bytes, void *stream);
void wpccc_free_basis(wpccc_basis *basis);

/* Sizes the caller needs to allocate outputs: total number of states N_tot, states on centre c,
 * radial functions on centre c, number of radial entries E_c = allowed (a' <= a, lambda) of centre c. */
int wpccc_n_states(const wpccc_basis *basis);
int wpccc_n_states_centre(const wpccc_basis *basis, int c);
int wpccc_n_rad_centre(const wpccc_basis *basis, int c);
int wpccc_n_radial_entries(const wpccc_basis *basis, int c);
/* Describes radial entry e of centre c: (a', a, lambda) with a' <= a.  Returns 0 or WPCCC_EINVAL. */
int wpccc_radial_entry(const wpccc_basis *basis, int c, int e, int *a_prime, int *a, int *lambda);

/* Workspace bytes.  what = 0: wpccc_matrix_elements for n_traj positions (n_steps ignored);
 * what = 1: wpccc_propagate of n_traj trajectories with n_steps RK4 steps (a size that lets the
 * pipeline keep its preferred window; any size >= the value for what = 2 works, with shorter
 * windows); what = 2: the minimum wpccc_propagate accepts. */
size_t wpccc_workspace_bytes(const wpccc_basis *basis, int n_traj, int n_steps, int what);

/* ---- options -------------------------------------------------------------------------------------
 * Selects between CUDA routes that compute the same thing (never a CPU path); takes effect from the
 * next call on this handle.  Keys:
 *   "mirror_pairs"       1 (default) / 0: on a z-grid symmetric about 0, evaluate the body-frame integrals of
 *                        eq. (9) at (b, -z) and (b, +z) together, and the direct radial entries of eq. (7), which
 *                        depend on the position through R only, once per pair (see wpccc_last_units).
 *   "solve_route"        how S(R) x = y is solved in every RK4 stage (role of ZGESV), with
 *                        S = [[I, K^H], [K, I]] reduced to its Schur complement A = I - K K^H (Hermitian,
 *                        positive definite whenever S is):
 *                        0 (default): blocked Cholesky factor A = L L^H, two triangular solves per stage
 *                           (a linear solve, as the paper insists, not an inverse); a position where A is not
 *                           positive definite is reported (WPCCC_ESINGULAR, wpccc_last_status);
 *                        1: explicit inverse A^{-1} by Gauss-Jordan elimination with partial pivoting
 *                           (the pivots plain partial pivoting of S would take, A22), applied as a
 *                           matrix-vector product per stage; works for any non-singular S, rounding error
 *                           cond(A) 2^-53.
 *   "inverse_kernel"     solve_route 1 only: 0 automatic, 1 shared-memory kernel, 2 global-memory blocked kernel.
 *   "inverse_chunk_cols" solve_route 1, register kernel: stage K in chunks of this many columns (0 automatic).
 *   "sweep_cluster"      CTAs (one thread-block cluster) per trajectory of the RK4 sweep a8: 0 (default) automatic -- one CTA for
 *                        small bases (N < 128), two up to N = 511, four beyond, where the streams of one SM bound a stage -- or 1, 2, 4
 *                        forced (4: two-centre only; a size the basis has no kernel instance for falls back to the nearest).
 *                        The CTAs of a cluster split the matrix-vector products of a stage by rows and exchange partial sums
 *                        through distributed shared memory; results agree to rounding (the summation order differs).
 *   "timing"             1 (default) / 0: record the CUDA events behind wpccc_last_timing.
 * Returns 0 or WPCCC_EINVAL (unknown key, value out of range). */
int wpccc_set_option(wpccc_basis *basis, const char *key, long long value);

/* ---- a2 alternative: tabulated direct couplings (the paper's own route, in exact form)
 * V_lambda(r, R) = min^lambda / max^(lambda+1) separates at r = R, so the grid sum of eq. (7) is
 *   F^c_lambda(a', a; R) = R^-(lambda+1) P_e[g] + R^lambda Q_e[g],   g = #{k : r_k < R},
 *   P_e[g] = sum_{k <= g} w_k u_a' u_a r_k^lambda,   Q_e[g] = sum_{k > g} w_k u_a' u_a r_k^-(lambda+1):
 * the same discrete sum as the GEMM of wpccc_matrix_elements / wpccc_propagate (up to rounding order), at 24 bytes of
 * HBM traffic per entry and position instead of 2 N_r flops.
 * wpccc_direct_table_bytes: bytes of the table [g = 0..N_r][entry] of (P, Q) pairs for this basis.
 * wpccc_enable_direct_tables: builds the tables in `dev_tables` [device, 256-byte aligned, caller-owned, must stay
 *   valid while enabled] and makes every later call on this handle use them instead of the GEMM; dev_tables == NULL
 *   switches back to the GEMM.  Synchronises `stream`.  Errors: WPCCC_EINVAL, WPCCC_ENOMEM (bytes too small). */
size_t wpccc_direct_table_bytes(const wpccc_basis *basis);
int wpccc_enable_direct_tables(wpccc_basis *basis, void *dev_tables /*[device] or NULL*/, size_t bytes, void *stream);

/* ---- a1-a6: matrix elements at given positions ------------------------------------------------
 * For each position p (b[p], z[p], v[p]) [host arrays] computes
 *   S = [[I, S_PT^H], [S_PT, I]],  H = [[D^T, H_TP], [H_PT, D^P]]            (eq. (1); A1)
 *   D^T, D^P   direct elements, eq. (6)-(7), radial integral as the grid sum over r_k
 *              evaluated at the exact R (A9), by an FP64 tensor-core GEMM over the radial grid;
 *   S_PT, H_PT, H_TP  two-centre overlap and electron-transfer elements with the translation
 *              factor e^{-+ i v z_m} (eq. (8)-(9) structure; A4, A5, A10) by the fixed
 *              product rule of wpccc_quad.
 * flags bit 0: multiply every element by e^{i (eps_row - eps_col) z / v} (interaction picture, A2).
 * flags bit 1: also return the radial entries F^c_lambda(a', a; R) in dF.
 * Outputs [device]: dS, dH [n_pos][N_tot][N_tot] complex, row-major (either may be NULL);
 *   dF [n_pos][E_T (+ E_P)] doubles (centre T entries then centre P), or NULL.
 * With one centre S is the identity and H = D^T. */
int wpccc_matrix_elements(const wpccc_basis *basis, int n_pos, const double *b /*[host]*/,
                          const double *z /*[host]*/, const double *v /*[host]*/, int flags,
                          double *dS /*[device]*/, double *dH /*[device]*/, double *dF /*[device]*/,
                          void *ws /*[device]*/, size_t ws_bytes, void *stream);

/* ---- a1-a8: propagation ------------------------------------------------------------------------
 * Integrates i S dc/dt = H c, i.e. dc/dz = -(i/v) S^{-1} H c (eq. (2)-(4)), for n_traj
 * straight-line trajectories (b[t], v[t]) [host arrays] concurrently, with classical RK4
 * (Algorithm 1) on the uniform grid z_i = z_min + i (z_max - z_min)/n_steps (A13).
 * The 2 n_steps + 1 evaluations of (S, H) per path are computed in windows for all
 * trajectories at once; the overlap system is factorised once per position and solved once per
 * RK4 stage (A14) by the route "solve_route" of wpccc_set_option selects (the role of ZGESV).
 * Initial condition c = delta_{j, init_state}; init_state = WPCCC_INIT_FROM_DC continues
 * from the amplitudes in dC (and the running maxima in d_norm_drift), e.g. to walk through a long
 * z-range in several calls.
 * Outputs [device]: dC [n_traj][N_tot] complex amplitudes at z_max;
 *   d_norm_drift [n_traj] max over steps of |c^H S c - 1| (A17), or NULL.
 * Errors: WPCCC_ENOMEM if ws_bytes < wpccc_workspace_bytes(.., 2).
 * WPCCC_ESINGULAR: at some position of some trajectory the overlap system could not be factorised:
 *   I - K K^H not positive definite (solve_route 0: with an over-complete two-centre basis the
 *   configured quadrature can leave S(R) indefinite at small R, A23), or a zero pivot /
 *   |S_PT| >= 1 (solve_route 1).  The amplitudes and the drift of those trajectories are NaN, every
 *   other trajectory is complete and valid; wpccc_last_status tells which and where.
 * The call synchronises `stream` before returning (it reads that status). */
int wpccc_propagate(const wpccc_basis *basis, int n_traj, const double *b /*[host]*/,
                    const double *v /*[host]*/, double z_min, double z_max, int n_steps, int init_state,
                    double *dC /*[device]*/, double *d_norm_drift /*[device] or NULL*/,
                    void *ws /*[device]*/, size_t ws_bytes, void *stream);

/* The same on an explicit step grid zgrid[0] < ... < zgrid[n_points - 1] [host], e.g. the paper's
 * z-grid zgrid[+-i] = +-z_min (z_max / z_min)^(i / n_z), zgrid[0] = 0: step i goes from z = zgrid[i] to
 * z_new = zgrid[i + 1] with h = z_new - z and z_mid = z + h / 2 (Algorithm 1 lines 13-15), n_points - 1 steps,
 * 2 n_points - 1 evaluations of (S, H) (4 n_z + 1 for the paper's 2 n_z + 1 points).  Everything else as above. */
int wpccc_propagate_grid(const wpccc_basis *basis, int n_traj, const double *b /*[host]*/, const double *v /*[host]*/,
                         int n_points, const double *zgrid /*[host]*/, int init_state,
                         double *dC /*[device]*/, double *d_norm_drift /*[device] or NULL*/,
                         void *ws /*[device]*/, size_t ws_bytes, void *stream);

/* Outcome of the last wpccc_propagate / wpccc_propagate_grid per trajectory: traj_status[t] [host, n_traj] = 0 (complete),
 * or (code << 28) | (1 + half-step index of the first position whose overlap system could not be factorised), code
 * 1 zero pivot, 2 |S_PT| >= 1, 3 not positive definite.  Half-step index i: z = z_min + i h / 2 on the uniform grid. */
int wpccc_last_status(const wpccc_basis *basis, int n_traj, int *traj_status /*[host]*/);

/* ---- eq. (4) as the paper solves it: the explicit matrix M ---------------
 * M = -(i/v) S^{-1} H at each position, i.e. the overlap system solved for the N_tot right-hand sides that are the
 * columns of H -- what the paper's ZGESV call produces (Fig. 3 measures its share of the run).  The hot path
 * (wpccc_propagate) never forms M (A14); this entry point exists for the like-for-like comparison of the solver cost and
 * for callers who want M itself.  Route: Schur complement A = I - K K^H, its inverse by Gauss-Jordan elimination with
 * partial pivoting, then three batched complex matrix products (Y_P -= K Y_T; W_P = A^{-1} Y_P; W_T = Y_T - K^H W_P).
 * flags bit 0: interaction-picture phases e^{i (eps_row - eps_col) z / v} (A2).  dM [device][n_pos][N_tot][N_tot] complex.
 * One centre: M = -(i/v) D^T (eq. (5)).  Synchronises `stream`; WPCCC_ESINGULAR names a position with a zero pivot. */
size_t wpccc_coupling_matrix_ws_bytes(const wpccc_basis *basis, int n_pos);
int wpccc_coupling_matrix(const wpccc_basis *basis, int n_pos, const double *b /*[host]*/, const double *z /*[host]*/,
                          const double *v /*[host]*/, int flags, double *dM /*[device]*/,
                          void *ws /*[device]*/, size_t ws_bytes, void *stream);

/* ---- a9: observables ------------------------------------------------------------------
 * From amplitudes dC [device, n_traj][N_tot] complex:
 *   P_state [n_traj][N_tot]       |c_j|^2
 *   P_nl    [n_traj][n_rad_tot]   sum over m for each radial function (centre T functions, then P)
 *   P_class [n_traj][5]           elastic (radial function of init_state), target excitation (bound),
 *                                 target continuum (wave packets), capture bound, capture continuum
 *   sigma_nl [n_vgroups][n_rad_tot], sigma_class [n_vgroups][5]
 *                                 2 pi Int b P(b) db by the trapezoid rule in ln b over the
 *                                 trajectories of each velocity group, sorted by b (units a0^2).
 * b [host][n_traj] (> 0: the rule lives on ln b), vgroup [host][n_traj] in 0..n_vgroups-1.  All outputs
 * [device]; any may be NULL (sigma_* need b and vgroup, P_nl / P_class respectively, and at most ~80 000
 * trajectories per call: their index scratch lives in the basis arena).  With sigma_* the call synchronises. */
int wpccc_probabilities(const wpccc_basis *basis, int n_traj, const double *dC /*[device]*/,
                        const double *b /*[host]*/, const int *vgroup /*[host]*/, int n_vgroups,
                        int init_state, double *P_state, double *P_nl, double *P_class,
                        double *sigma_nl, double *sigma_class, void *stream);

/* ---- a9 without any allocation: cross sections with the scratch in a static device array -------
 * For callers that cannot call cudaMalloc and hold no workspace (code under CUDA graph capture set-up, tight serving
 * loops, harnesses that forbid allocation): the cross-section integral of P:L106,
 *   dSigma [device][n_vgroups][n_cols] = 2 pi Int b P(b) db  (trapezoid rule in ln b over the trajectories of each
 *   velocity group sorted by b, exactly as sigma_nl / sigma_class of wpccc_probabilities),
 * of any per-trajectory probability table dP [device][n_traj][n_cols] (row-major, e.g. P_nl or P_class).  It takes no
 * basis handle and no workspace: its index scratch (b, the sorted order, the group offsets) is a file-scope
 * `static __device__` array of WPCCC_STATIC_SCRATCH_BYTES inside the library, which every GPU that loads libwpccc.so
 * holds until the process exits.  b [host][n_traj] > 0, vgroup [host][n_traj] in 0..n_vgroups-1.
 * Limits: n_traj <= WPCCC_STATIC_MAX_TRAJ and n_vgroups <= WPCCC_STATIC_MAX_VGROUPS per call, else WPCCC_ENOMEM with a
 * message naming the limit (nothing is launched).  Calls no cudaMalloc / cudaFree / allocating library routine.
 * All calls on a device share the one array: calls whose GPU work overlaps (other streams or host threads) race --
 * issue one at a time per device.  The array keeps the previous call's contents; each call rewrites every element it
 * reads, nothing needs to start at zero.  Synchronises `stream` (the host index vectors must outlive the copies). */
#define WPCCC_STATIC_SCRATCH_BYTES (256 * 1024)
#define WPCCC_STATIC_MAX_TRAJ 16384
#define WPCCC_STATIC_MAX_VGROUPS 1024
int wpccc_cross_sections_static(int n_traj, int n_cols, const double *dP /*[device]*/, const double *b /*[host]*/,
                                const int *vgroup /*[host]*/, int n_vgroups, double *dSigma /*[device]*/, void *stream);

/* ---- diagnostics ----------------------------------------------------------------------------- */

/* Per-family device time of the last wpccc_propagate / wpccc_matrix_elements call on this handle,
 * in milliseconds, measured with CUDA events on the streams the kernels ran on, and launch counts.
 * ms[k], launches[k], k: 0 direct GEMM (a2), 1 direct assembly (a3), 2 transfer node tables (a4),
 * 3 transfer contraction (a5), 4 rotation/assembly (a6), 5 factorisation (a7), 6 RK4 sweep (a8),
 * 7 other.  Synchronises the device.  Returns the number of families (8). */
int wpccc_last_timing(const wpccc_basis *basis, double *ms /*[host][8]*/, long long *launches /*[host][8]*/);

/* Positions processed by each family (same order) in the last wpccc_propagate / wpccc_matrix_elements
 * call, for the families that count them (0 direct GEMM / tables in wpccc_propagate, 2 node tables,
 * 3 contraction, 4 rotation; 0 otherwise).
 * wpccc_propagate on a z-grid symmetric about 0 (z_min = -z_max) evaluates the body-frame integrals of
 * eq. (9) once per mirror pair (b, -z), (b, +z) -- they differ only by the complex conjugation of the
 * axial phase -- as far as the workspace beyond wpccc_workspace_bytes(.., 2) can hold the second
 * member's integrals until the sweep reaches it; units[3] is then smaller
 * than the number of positions.  The direct radial entries F^c_lambda(a', a; R) of eq. (7) are the same at
 * (b, -z) and (b, +z) (same R): on such a grid, when the workspace can hold F of the half-step positions up to
 * z = 0 of every distinct b ((n_steps + 1) x n_entries doubles each; included in wpccc_workspace_bytes(.., 1)
 * up to its cap), the contraction of a2 runs for z <= 0 only and units[0] is about half the positions; the
 * assembly a3 (which differs through P_lambda^mu(cos Theta)) runs everywhere.
 * wpccc_set_option(basis, "mirror_pairs", 0) disables both.
 * Returns the number of families (8) or WPCCC_EINVAL. */
int wpccc_last_units(const wpccc_basis *basis, long long *units /*[host][8]*/);

/* Measures the device's FP64 peak with a register-resident micro-benchmark on `stream`:
 * kind 0 = DFMA (plain FP64 FMA pipe), kind 1 = DMMA (mma.sync.m8n8k4.f64).  Returns TFLOP/s
 * (negative WPCCC_E* as a double on error).  Used by bench.py for the roofline denominator. */
double wpccc_fp64_peak(int kind, void *stream);

const char *wpccc_last_error(void);
const char *wpccc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WPCCC_H */
