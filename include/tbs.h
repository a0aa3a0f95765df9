/*
 * tbs.h -- C ABI of libtbs: traditional Born series (TBS) solve of the inhomogeneous Helmholtz
 * equation on one B200 (sm_100a).  Paper: arxiv 2507.13754 (citations: PAPER.md line numbers).
 *
 *   psi = G V psi + G S                      (Eq. 17)
 *   psi = [1 + GV + GVGV + ...] G S          (Eq. 18)  -- summed term by term:
 *   u_0 = A.(G S), u_{n+1} = A.G(V.u_n), p = sum_n u_n
 *   G = crop . IDFT_2N . ghat(p) . DFT_2N . zero-pad,  ghat = 1/(|p|^2 - k0^2 - i eps)
 *   V(r) = ktilde(r)^2 - k0^2 - i eps, eps = damping k0^2
 *
 * Conventions
 *  - Every array is row-major with x fastest: index = (z*Ny + y)*Nx + x.
 *  - complex64 = interleaved float (re, im).  "dev" = CUDA device pointer, "host" = host pointer.
 *  - The caller owns every buffer it passes in.  V, S, p of every frequency and the FFT intermediates live in
 *    one device range, the workspace: the caller's (tbs_plan_set_workspace, e.g. a torch allocation) or, when
 *    none was given by the first call that needs it, the plan's own.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *  - No exception crosses the ABI: every call returns a tbs_status; tbs_last_error() gives text.
 *  - A plan is not thread-safe; distinct plans are independent.
 *  - Grid sizes: every n[i] a power of two, 32 <= n[i] <= 4096 (2-D), 32 <= n[i] <= 512 (3-D),
 *    else TBS_ERR_UNSUPPORTED_SIZE.  The padded length is 2 n[i] per axis and is never
 *    materialised in more than one axis beyond what a pass needs.
 *  - There is no CPU fallback: without a CUDA device every compute call returns TBS_ERR_CUDA.
 */
#ifndef TBS_H_
#define TBS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tbs_plan tbs_plan;

typedef enum {
    TBS_OK = 0,
    TBS_NOT_CONVERGED = 1,       /* max_terms reached: field and history are valid */
    TBS_ERR_INVALID_ARG = -1,
    TBS_ERR_UNSUPPORTED_SIZE = -2,
    TBS_ERR_NOT_READY = -3,      /* medium or source not set */
    TBS_ERR_CUDA = -4,
    TBS_ERR_DIVERGED = -5,       /* the series diverges (||GV|| >= 1): see tbs_solve */
    TBS_ERR_ALLOC = -6
} tbs_status;

/* Library version string (static storage). */
const char *tbs_version(void);

/* Create a plan for one grid and nfreq frequencies (Alg. 1 Input).
 *   ndim: 2 or 3.  n: grid points per axis in x, y, z order (n[2] ignored for ndim = 2).
 *   dx_m: grid spacing (m), equal on all axes.  f_hz[nfreq]: frequencies (host).
 *   c0: reference sound speed (m/s), k0 = 2 pi f/c0.
 *   damping: eps/k0^2, the paper uses 0.8.
 * Builds the per-axis |p|^2 tables and twiddles (Green's-spectrum precompute)
 * and allocates device workspaces.  *out is NULL on failure. */
tbs_status tbs_plan_create(tbs_plan **out, int ndim, const int32_t n[3], double dx_m, int nfreq,
                           const double *f_hz, double c0, double damping);
void tbs_plan_destroy(tbs_plan *plan);

/* Workspace (inputs of Alg. 1, held on the device).  tbs_plan_workspace_bytes: the size the
 * plan needs -- V, S and p [n] complex64 per frequency, the x-transformed rows W1 [nz ny][2 nx] and, in 3-D, the
 * y/z-transformed W2 [nz][2 ny][2 nx], the latter two once per series in flight (one, or two for nfreq > 1),
 * every region rounded up to 256 bytes -- known as soon as the plan exists.  tbs_plan_set_workspace: run in
 * caller-owned device memory (dev_ptr 256-byte aligned, bytes >= the size above; it must outlive the plan or the
 * next call of this function).  Contents are undefined afterwards: set medium and source (again).  Without this
 * call the plan allocates the same range itself at the first call that needs it.
 * tbs_plan_device_bytes: device bytes the plan itself has allocated (tables, control, and its own workspace). */
size_t tbs_plan_workspace_bytes(const tbs_plan *plan);
tbs_status tbs_plan_set_workspace(tbs_plan *plan, void *dev_ptr, size_t bytes);
size_t tbs_plan_device_bytes(const tbs_plan *plan);

/* The m-th frequency a periodic n-point grid of spacing dx_m carries exactly, m c0/(n dx) -- the paper picks its
 * frequency this way (f = 55 v_f/(4096 dx) = 1 007 080 Hz).  0 for non-positive arguments. */
double tbs_grid_harmonic_frequency(int m, double c0, int n, double dx_m);

/* Frequency batch (nfreq > 1): how many members are solved at once, 1 ... 4 (default 2).  The members in flight
 * run on streams of the plan's own, so that the HBM-bound passes of one overlap the FP32-bound convolution pass of
 * another as SM resources free up; a member that has stopped hands its place to the next frequency.  The transform
 * intermediates of the first two members are part of the workspace; for a third and fourth the plan allocates its
 * own (W1, and W2 in 3-D, each).  Pays on grids that do not fill the GPU (3-D 64^3 x 16 frequencies: 126 ms one after
 * the other, 93 / 83 / 76 ms with 2 / 3 / 4 in flight); at 256^3 two members gain 4 % and more add nothing.  The paper's
 * harmonic loop is sequential. */
tbs_status tbs_set_concurrency(tbs_plan *plan, int members);

/* Text of the last error on this plan (plan-owned storage, valid until the next call). */
const char *tbs_last_error(const tbs_plan *plan);

/* Homogeneous absorbing(-dispersive) medium in the paper's own form, Eq. 24: the potential
 * acts in k-space, VV(k) = -i tau w k^nu + eta k^(nu+1) - i eps with tau = -2 alpha0 v_f^(nu-1),
 * eta = 2 alpha0 v_f^nu tan(pi nu/2), v_f = the plan's c0, alpha0_si in Np (rad/s)^-nu m^-1;
 * dispersive = 0 drops the eta term (the "absorbing" row of Table 3).  The term update becomes
 * u_{n+1} = A F^-1[ghat(p) VV(|p|) F[u_n]]: the spatial potential is ignored (tbs_set_medium not needed)
 * and the multiplier is applied inside the fused Green's-spectrum stage.  alpha0_si = 0 switches back to the
 * spatial potential, which then has to be set again; so does a later tbs_set_medium / tbs_set_potential (the two
 * forms are not combined).  With TBS_SCHEME_CBS selected (or selecting it afterwards): TBS_ERR_INVALID_ARG. */
tbs_status tbs_set_kspace_absorption(tbs_plan *plan, double alpha0_si, double nu, int dispersive);

/* A scatterer inside the absorbing(-dispersive) medium of tbs_set_kspace_absorption: the potential operator is the
 * sum of the k-space multiplier of Eq. 23 and the spatial term U_s(r) = (w/c(r))^2 - k0^2 of Eq. 25
 * (its -i eps is the multiplier's), so that
 *   u_{n+1} = A F^-1[ghat(p) (VV(|p|) F[u_n] + F[U_s u_n])].
 * The paper runs the two potentials in separate experiments (Eq. 24, Eq. 26); both are terms of the one operator V of
 * Eq. 17.  c [n] dev float: sound-speed map (c == the plan's c0 outside the scatterer).  Needs the
 * periodic boundary in 2-D (the paper's form: the unpadded kernels carry U_s u_n and u_n as the two lanes of every
 * packed value and transform them together) and an active multiplier; else TBS_ERR_INVALID_ARG / TBS_ERR_NOT_READY.
 * Undone by tbs_set_kspace_absorption, tbs_set_medium, tbs_set_potential or leaving the periodic boundary. */
tbs_status tbs_set_kspace_scatterer(tbs_plan *plan, const float *c, void *stream);

/* Boundary treatment (default TBS_BOUNDARY_PAD: zero-pad to 2N per axis, linear convolution, crop --
 * BASELINE north_star).  TBS_BOUNDARY_PERIODIC is the paper's own: the FFTs act on the N-grid itself
 * (Eq. 19, Alg. 1 l.36-38) and wrap-around is left to the absorbing layer of tbs_set_abl
 * (PAPER.md:251-256).  It runs through the same kernels: only the even padded frequencies, which are the
 * frequencies of the N-grid, keep a non-zero Green's spectrum.  Rebuilds the axis tables. */
enum { TBS_BOUNDARY_PAD = 0, TBS_BOUNDARY_PERIODIC = 1 };
tbs_status tbs_set_boundary(tbs_plan *plan, int boundary);

/* Convergence measure r_n (history[n], compared with tol).  TBS_CRIT_L2_GRID (default, reading A8):
 * ||u_n||_2 / ||p_n||_2 over the whole grid.  TBS_CRIT_L1_ROW: the paper's Eq. 30,
 * sum_m |psi_{l+1}(row, m) - psi_l(row, m)| / sum_m |psi_l(row, m)| = sum |u_n| / sum |p_{n-1}| on grid row
 * `row` (index y in 2-D, z*ny + y in 3-D); history[0] = 1. */
enum { TBS_CRIT_L2_GRID = 0, TBS_CRIT_L1_ROW = 1 };
tbs_status tbs_set_criterion(tbs_plan *plan, int criterion, int row);

/* Iteration scheme of tbs_solve* (default TBS_SCHEME_BORN, the paper's traditional Born series,
 * PAPER.md:156-160 Eqs. 18-19).  TBS_SCHEME_CBS is the convergent Born series the paper names as the way
 * past strong / extended scatterers (formula from its ref. [16]): with the
 * preconditioner gamma = i V / eps,  psi <- psi + gamma (G(V psi + S) - psi);  in term form
 * u_0 = gamma A G S, u_{n+1} = u_n + gamma (A G(V u_n) - u_n), p = sum u_n.  Same kernels, same stopping
 * rule; one more field of n complex64 per frequency.  Converges when eps >= max |k^2 - k0^2|. */
enum { TBS_SCHEME_BORN = 0, TBS_SCHEME_CBS = 1 };
tbs_status tbs_set_scheme(tbs_plan *plan, int scheme);

/* Absorbing layer of Eq. 29 on all faces, `cells` wide, window
 * 1/(1+exp(-zeta (x - mu/2))) with zeta*mu/2 = zeta_half_mu (paper: 9.666).  cells = 0 (default)
 * is the pure zero-pad/crop boundary.  Folded into the crop kernel as per-axis factors. */
tbs_status tbs_set_abl(tbs_plan *plan, int cells, double zeta_half_mu);

/* Medium -> potential, for every frequency of the plan (absorption from
 * Eq. 3 and Eq. 7):
 *   ktilde = w/c(r) + alpha (tan(pi y/2) + i), alpha = alpha0 w^y, V = ktilde^2 - k0^2 - i eps.
 *   c [n] dev float: sound speed map.  rho [n] dev float or NULL: density map; accepted and not read -- density
 *   does not enter V (rho_s ~ rho_f).  rho0 > 0: the ambient density of xi = beta/(rho0 c0^4),
 *   the constant of the harmonic sources; unused by a linear solve.
 *   alpha0_map [n] dev float or NULL (then the scalar alpha0_db_mhz_cm is used), dB/(MHz^y cm).
 *   y: power-law exponent, y != 1 unless alpha0 == 0.  beta = 1 + B/2A.
 * tbs_set_medium_host takes the same maps as HOST pointers and copies them itself. */
tbs_status tbs_set_medium(tbs_plan *plan, const float *c, const float *rho, const float *alpha0_map,
                          double alpha0_db_mhz_cm, double y, double beta, double rho0, void *stream);
tbs_status tbs_set_medium_host(tbs_plan *plan, const float *c, const float *rho,
                               const float *alpha0_map, double alpha0_db_mhz_cm, double y,
                               double beta, double rho0, void *stream);

/* Raw potential for frequency ifreq (test hook and user-supplied V): V [n][2] dev, in 1/m^2,
 * must already include the -i eps term. */
tbs_status tbs_set_potential(tbs_plan *plan, int ifreq, const float *V, void *stream);

/* Point sources (transducer elements): pos_m [n_src][ndim] host doubles in
 * (x, y[, z]) order, centre of cell (0,0,0) at r = 0; amp [nfreq][n_src][2] host floats (re, im).
 * Off-grid points are deposited with multilinear weights; a point on a node is the paper's
 * single-pixel source.  A point outside the grid gives TBS_ERR_INVALID_ARG. */
tbs_status tbs_set_source(tbs_plan *plan, int n_src, const double *pos_m, const float *amp,
                          void *stream);
/* Dense source density for frequency ifreq: S [n][2] dev. */
tbs_status tbs_set_source_field(tbs_plan *plan, int ifreq, const float *S, void *stream);

/* Run the series for every frequency until history < tol, max_terms, or divergence.
 *   p_out [nfreq][n][2]: dev (tbs_solve) or host (tbs_solve_host) complex64 field.
 *   history [nfreq][max_terms+1] host doubles: history[k] = ||u_k||_2/||p_k||_2, history[0] = 1;
 *     entries after n_terms are 0.   n_terms [nfreq] host: index of the last term added.
 * Synchronises `stream` before returning.  Returns the worst status over frequencies.
 * TBS_ERR_DIVERGED (field and history up to that term are still written): the measure became non-finite, or
 * ||u_n|| exceeded 10^6 ||u_0||, or history[n] stayed above ten times its running minimum for 32 terms in a row
 * (the paper only caps the iterations; convergence needs ||GV|| < 1).
 * Range: fields and norms are complex64 / fp32 partial sums; |u_n|^2 must stay inside the fp32 range, i.e.
 * term magnitudes between about 1e-19 and 1e19.  A series whose terms fall below that (harmonics 3-5 of a
 * source of arbitrary small strength) reports TBS_ERR_DIVERGED (0/0); scale the source, or use the
 * surface-pressure rescaling of tbs_solve_harmonics.  The Eq. 30 row criterion pre-scales by 2^20 and
 * covers 1e-25 < |u_n| < 1e13. */
tbs_status tbs_solve(tbs_plan *plan, int max_terms, double tol, float *p_out, double *history,
                     int32_t *n_terms, void *stream);
tbs_status tbs_solve_host(tbs_plan *plan, int max_terms, double tol, float *p_out_host,
                          double *history, int32_t *n_terms, void *stream);

/* Continue a series that stopped at its cap (the natural call after TBS_NOT_CONVERGED; the paper caps at 2000
 * iterations): single-frequency plans only, and only directly after the tbs_solve* that returned
 * TBS_NOT_CONVERGED -- any call that changes the medium, source, options, workspace or the running field in between
 * gives TBS_ERR_NOT_READY.  max_terms is the new cap on the TOTAL number of terms (> the terms already summed);
 * history [max_terms+1] receives the whole history, n_terms the total.  The partial sum, the transformed V u_n of the
 * next term and the norms are still on the device, so the result equals one uninterrupted tbs_solve(max_terms, tol)
 * term for term. */
tbs_status tbs_solve_resume(tbs_plan *plan, int max_terms, double tol, float *p_out, double *history,
                            int32_t *n_terms, void *stream);

/* Nonlinear case (Eq. 27b, 229 Eq. 28b, 266): solve `p1` (fundamental, nfreq = 1),
 * optionally rescale it so that max|p1| over the row/plane `ref_row` equals surface_pressure_pa
 * (<= 0: no rescale), form S2 = -xi (2w)^2 p1^2/2 with xi = beta/(rho0 c0^4), and solve `p2`
 * (a plan created at 2 f on the same grid, medium already set).  Outputs as tbs_solve, once for
 * each plan; p1_out / p2_out [n][2] dev. */
tbs_status tbs_solve_second_harmonic(tbs_plan *p1, tbs_plan *p2, int max_terms, double tol,
                                     int ref_row, double surface_pressure_pa, float *p1_out,
                                     float *p2_out, double *history1, double *history2,
                                     int32_t *n_terms1, int32_t *n_terms2, void *stream);

/* Harmonics 1..n_harm (n_harm <= 5) of a nonlinear medium, one after the other (Eqs. 27-28,
 * PAPER.md:266): plans[h-1] is a plan with nfreq = 1 created at h*f1 on the same grid with its medium set
 * (so k0 -> h k0, eps_h = damping (h k0)^2, absorption at h w).  The fundamental is solved from its own
 * source, optionally rescaled as in tbs_solve_second_harmonic, and harmonic h >= 2 from
 *   S_h = -xi (h w1)^2 C_h,  C_2 = psi1^2/2, C_3 = psi1 psi2, C_4 = psi2^2/2 + psi1 psi3,
 *   C_5 = psi2 psi3 + psi1 psi4   (sum-frequency terms only), xi = beta/(rho0 c0^4) of plans[0].
 * p_out[h-1] dev [n][2]; history[h-1] host [max_terms+1]; n_terms host [n_harm].  Host arrays of pointers.
 * Returns the worst status; a negative status of one harmonic stops the chain. */
tbs_status tbs_solve_harmonics(tbs_plan *const *plans, int n_harm, int max_terms, double tol, int ref_row,
                               double surface_pressure_pa, float *const *p_out, double *const *history,
                               int32_t *n_terms, void *stream);

/* Introspection for tests and the bench. */
/* One application of G to x (dev [n][2]) for frequency ifreq: out = crop IDFT ghat DFT pad x. */
tbs_status tbs_apply_green(tbs_plan *plan, int ifreq, const float *x, float *out, void *stream);
/* Copy the plan's V or S for frequency ifreq to dev buffer out [n][2]. */
tbs_status tbs_get_potential(tbs_plan *plan, int ifreq, float *out, void *stream);
tbs_status tbs_get_source(tbs_plan *plan, int ifreq, float *out, void *stream);
/* Full Green's spectrum ghat on the padded grid in natural FFT order, dev [prod(2 n[i])][2]
 * (the tabulated form of the precompute kernel; the hot path recomputes ghat from axis tables). */
tbs_status tbs_green_spectrum(tbs_plan *plan, int ifreq, float *out, void *stream);
/* Kernel launches issued by the last tbs_solve* on this plan, and device time (ms) of its term
 * loop measured with CUDA events on `stream`. */
int64_t tbs_last_launch_count(const tbs_plan *plan);
double tbs_last_loop_ms(const tbs_plan *plan);
/* Per-kernel device time of ONE term (ms) for frequency ifreq: after a live series of term 0 and three
 * warm-up terms, each kernel of the term is launched `reps` <= 256 times back to back between two CUDA events
 * on `stream` (no event between launches), and the average is returned: out_ms[0] = row kernel K31,
 * out_ms[1] = K2 (2-D) or out_ms[1..3] = y-forward, z-convolution, y-inverse passes (3-D).  Requires medium
 * and source; leaves the plan's running field and intermediates undefined. */
tbs_status tbs_profile_term(tbs_plan *plan, int ifreq, int reps, double out_ms[4], void *stream);
/* Launch overlap (default off; measured 2 % slower at 2-D 2048^2 on B200): the kernels of the term loop are launched with programmatic stream serialization,
 * so the CTAs of a kernel become resident while the previous one drains; every kernel orders its memory accesses
 * behind the previous kernel with griddepcontrol.wait.  0 = plain stream order. */
tbs_status tbs_set_launch_overlap(tbs_plan *plan, int on);
/* Terms per graph launch (default 16); 0 disables CUDA graphs (plain launches). */
tbs_status tbs_set_graph_batch(tbs_plan *plan, int terms_per_graph);

#ifdef __cplusplus
}
#endif
#endif /* TBS_H_ */
