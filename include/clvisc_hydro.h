/* clvisc_hydro.h -- C ABI of the B200-native CLVisc evolution step.
 *
 * One call of hydro_step(ctx, 1) advances second-order viscous hydrodynamics on a
 * (tau, x, y, eta_s) Milne grid by one RK2 (Heun) step, arXiv:1802.04449:
 *   - KT central finite-volume update of T^{tau mu} and pi^{mu nu}   PAPER.md:193-213 (Eq.40-44)
 *   - Israel-Stewart relaxation source of pi^{mu nu}                 PAPER.md:165-183 (Eq.33-38)
 *   - geometric (Milne) source of T^{tau mu}                         PAPER.md:161     (Eq.31)
 *   - root-find T^{tau mu} - pi^{tau mu} -> e, P, u^mu through the EoS  PAPER.md:229,235 (Eq.51,54)
 *   - predictor/corrector with u* = 2u^n - u^{n-1}                   PAPER.md:225-239 (Eq.49-54)
 * The readings of every garbled / silent passage are listed in DESIGN.md ("Readings", A1..A26).
 *
 * Conventions
 *   - "tilde" (tetrad) components, g~ = diag(1,-1,-1,-1): u~ = gamma (1, v_x, v_y, v_eta),
 *     pi~ per PAPER.md:129 (Eq.20); T_f^{tau mu} = (T^{tau tau}, T^{tau x}, T^{tau y}, tau T^{tau eta_s})
 *     WITHOUT the paper's extra overall factor tau (Eq.18: T~ = tau * T_f).
 *   - pi component order: 0 tt, 1 tx, 2 ty, 3 tn, 4 xx, 5 xy, 6 xn, 7 yy, 8 yn, 9 nn  (n = eta_s).
 *   - user arrays are UNPADDED component-major SoA [comp][nz][ny][nx], x fastest, element type
 *     double (precision 64) or float (precision 32) as chosen at create.
 *   - every field pointer carries a memory-space tag (HYDRO_MEM_DEVICE / HYDRO_MEM_HOST).  Device
 *     pointers are used in place, stream-ordered on opts->stream.  Host pointers are copied
 *     through the workspace with cudaMemcpyAsync on the same stream; the call synchronises the
 *     stream before it returns so the host buffer may be reused (pinned memory makes it fast).
 *   - the caller owns every buffer it passes, including the workspace; the library never frees
 *     them and keeps no pointer to field arguments after the call returns.  The workspace must
 *     stay alive (and untouched) until hydro_destroy.
 *   - return value: 0 success; negative = error (below); hydro_diag returns a non-negative warning bit mask
 *     (hydro_step never synchronises, so warnings are reported by hydro_diag only).  No exceptions, no global state; a context is not thread-safe.
 *   - the whole path runs in CUDA kernels for sm_100a; there is no CPU fallback: without a usable
 *     device every compute entry point returns HYDRO_ECUDA.
 */
#ifndef CLVISC_HYDRO_H
#define CLVISC_HYDRO_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hydro_ctx hydro_ctx; /* opaque, owned by the library (host memory only) */

enum { HYDRO_OK = 0, HYDRO_EINVAL = -1, HYDRO_ENOMEM = -2, HYDRO_ECUDA = -3, HYDRO_ESTATE = -4 };
enum { HYDRO_WARN_CFL = 1, HYDRO_WARN_NAN = 2, HYDRO_WARN_ROOT = 4 };
enum { HYDRO_MEM_DEVICE = 0, HYDRO_MEM_HOST = 1 };

/* Grid: nx,ny,nz cells along x, y, eta_s; cell sizes in fm, fm, (unitless).
 * bc[a]: 0 = zero-gradient outflow (neighbour index clamped; "constant extrapolation for boundary
 * cells"), 1 = periodic.  geometry: 0 = Milne, 1 = Cartesian (all Christoffel terms
 * off and all tau factors 1, the paper's own test mode). */
typedef struct {
  int nx, ny, nz;
  double dx, dy, deta;
  int bc[3];
  int geometry;
} hydro_grid;

/* Equation of state.  kind 0: EOSI, P = e/3, T = hbarc (e/(c_sb hbarc))^{1/4}.
 * kind 1: table with n log-spaced nodes e_k = e_min (e_max/e_min)^{k/(n-1)}; P and T (GeV) are HOST
 * arrays of n doubles, copied at create; linear interpolation in e inside a bracket, c_s^2 = the
 * slope of the bracket; below e_min P = P_0 e/e_min, T = T_0 (e/e_min)^{1/4}; above e_max
 * P = P_{n-1} + (e-e_max)/3, T = T_{n-1} (e/e_max)^{1/4}  (A16). */
typedef struct {
  int kind;
  int n;
  double e_min, e_max;
  const double *P, *T;
  double c_sb;
} hydro_eos;

/* Options.  precision 64 or 32 (storage AND arithmetic).  minmod_theta in [1,2] (A4); e_floor: dynamic
 * floor on e (A8); pi_limit_xi <= 0 switches the pi limiter off (A14); v_max: clamp of |M|/M0 (A7),
 * <= 0 selects the default 0.999 (gamma <= 22.4; A7 gives the evidence); root_iters: fixed Newton iteration
 * count of the table root-find (<= 0: default 6); stream: a cudaStream_t (NULL = legacy default
 * stream); workspace: DEVICE memory of the current device, at least hydro_workspace_bytes(), 256-byte aligned (a host
 * pointer or memory of another GPU is refused with HYDRO_EINVAL).
 * kernel: 0 = default (the fastest one as measured on B200: 4 from 5e5 cells on, 2 for smaller grids, both precisions);
 * 4 = marching per-cell kernel (hydro_stage_march.cuh): kernel 2's store and x / y flux code, but a block walks along
 * eta_s and forms every eta_s slope and face once, with the per-column pipeline state in tensor memory;
 * 2 = per-cell fused kernel on the extended 19-word state (hydro_stage_fused.cuh); 3 = tile kernel
 * (hydro_stage_tile.cuh): TMA-staged 32x8 tiles marching along eta_s, every slope and face flux computed once, 14-word
 * ghosted SoA state; 1 = per-cell reference kernel (re-derives P, u^tau, c_a at every stencil point).  All four give
 * the same results to rounding and are covered by the parity tests. */
typedef struct {
  int precision;
  double minmod_theta, e_floor, pi_limit_xi, v_max;
  int root_iters;
  int kernel;
  void *stream;
  void *workspace;
  size_t workspace_bytes;
  /* SURVEY 8(f)-2 (PAPER.md:58-60 Eq.4, :169 Eq.33, :412-437): the lambda_1 term  -(lambda_1/tau_pi) pi^{<mu}_l pi^{nu>l}
   * with lambda_1 = lambda1_hat / e, 0 = off (the paper's production setting); and the coefficient of
   * the relaxation time tau_pi = tau_pi_coeff eta_v/(T s), <= 0 selects the paper's 5.  The paper's
   * closed-form Gubser test uses lambda1_hat = -10 and tau_pi_coeff = 4 lambda1_hat^2 / 9. */
  double lambda1_hat, tau_pi_coeff;
  /* SURVEY 8(f)-4 (Eq.53 as printed; A12): 1 = the stage-2 right-hand side of T^{tau mu} is
   * evaluated with pi^{n+1} (the result of Eq.52) instead of pi': stage 2 becomes three launches (4 per RK2 step).
   * Kernels 2 and 4 only (HYDRO_EINVAL otherwise); ignored for eta_over_s = 0.  0 = standard Heun (default). */
  int strict_eq53;
  /* SURVEY 8(f)-3 (PAPER.md:46-56 Eq.1-3; :153-171 Eq.28, 30, 32, 34; :614 the 16-word cell): bulk_baryon = 1 evolves the
   * bulk pressure Pi and the net-baryon density n next to T^{tau mu} and pi^{mu nu} (readings A28-A32):
   *   T_f^{mu nu} = (e + P + Pi) u u - (P + Pi) g + pi;   d_mu(u^mu Pi) = -(Pi + zeta theta)/tau_Pi - Pi theta/3 with
   *   tau_Pi = tau_pi and zeta = zeta_over_s * s;   d~_mu(tau n u~^mu) = 0;   root-find with P + Pi;   |Pi| <= xi P.
   * Viscous runs only, kernels 2 and 4 (opts->kernel 0, 2 or 4), not with strict_eq53; needs
   * hydro_workspace_bytes_ext(); state loaded / read with hydro_load_ext / hydro_read_ext.  0 = off (the paper's setting,
   * "bulk viscosity and net baryon density are set to 0 in the current version"). */
  int bulk_baryon;
  double zeta_over_s;
} hydro_opts;

/* Diagnostics (PAPER.md:640 for e_max).  cfl[a] = max over cells of
 * c_a h / Delta_a in stage 1 of the last step; counters are cumulative since hydro_load. */
typedef struct {
  double tau;
  long long step;
  double cfl[3];
  double e_max;
  long long n_floor, n_clamp, n_pi_limited, n_nan, n_root_unconverged;
} hydro_diag_t;

/* Bytes of device workspace a context for this grid/precision/viscosity needs (0 on bad input). */
size_t hydro_workspace_bytes(const hydro_grid *grid, int precision, double eta_over_s);

/* As hydro_workspace_bytes, for a context created with opts->bulk_baryon (16 evolved words per cell). */
size_t hydro_workspace_bytes_ext(const hydro_grid *grid, int precision, double eta_over_s, int bulk_baryon);

/* Create a context.  tau0: initial proper time (fm/c), dtau: fixed step h; eta_over_s = 0 selects
 * the ideal-fluid path (no pi array is touched, A15).  Errors: HYDRO_EINVAL (bad sizes, precision,
 * theta, table), HYDRO_ENOMEM (workspace too small or misaligned), HYDRO_ECUDA. */
int hydro_create(hydro_ctx **out, const hydro_grid *grid, double dtau, double tau0,
                 const hydro_eos *eos, double eta_over_s, const hydro_opts *opts);

/* Load initial data: T_tau_mu = T_f^{tau mu} [4][nz][ny][nx]; pi_mu_nu = pi~ [10][nz][ny][nx] or NULL
 * (= 0).  Root-finds the primitives (Eq.51), bootstraps u^{-1} with one ideal-fluid predictor
 * (A23), resets tau, step and counters.  mem: HYDRO_MEM_DEVICE / HYDRO_MEM_HOST. */
int hydro_load(hydro_ctx *ctx, const void *T_tau_mu, const void *pi_mu_nu, int mem);

/* SURVEY 8(f)-3, contexts created with opts->bulk_baryon: hydro_load with two more fields, Pi [nz][ny][nx] and the
 * net-baryon density n [nz][ny][nx] (either may be NULL = 0).  T_tau_mu is the FULL tensor including the bulk pressure.
 * hydro_read_ext returns Pi and n of the current state (either may be NULL).  HYDRO_ESTATE on other contexts. */
int hydro_load_ext(hydro_ctx *ctx, const void *T_tau_mu, const void *pi_mu_nu, const void *Pi, const void *n_b, int mem);
int hydro_read_ext(hydro_ctx *ctx, void *Pi, void *n_b, int mem);

/* Overwrite / read the history u~^i at step n-1, [3][nz][ny][nx] (analytic tests, bitwise resume). */
int hydro_set_history(hydro_ctx *ctx, const void *u_prev, int mem);
int hydro_read_history(hydro_ctx *ctx, void *u_prev, int mem);

/* Advance n RK2 steps (2 kernel launches per step on opts->stream, no host synchronisation).
 * Errors: HYDRO_ESTATE before hydro_load; HYDRO_ECUDA on a launch error. */
int hydro_step(hydro_ctx *ctx, int n);

/* ---- eta_s-slab decomposition --------------------------------------------------------------
 * One event can be split into slabs of eta_s planes, one context per slab (one GPU each), each slab carrying two ghost
 * planes per interior side and a zero-gradient boundary in its own eta_s: the stencil reaches two planes, so the results
 * of a slab's interior planes are exactly those of the undivided grid as long as the ghost planes hold the neighbours'
 * data when a stage reads them.  That takes one exchange after EACH stage, hence:
 * hydro_stage: run ONE stage of the current RK2 step (1: state n -> state '; 2: -> state n+1, completes the step).
 *   hydro_step(ctx, 1) == hydro_stage(ctx, 1); hydro_stage(ctx, 2).  HYDRO_ESTATE out of order; HYDRO_EINVAL for
 *   kernel 3 or strict_eq53.
 * hydro_plane_bytes: bytes of one eta_s plane of a state buffer (all fields, internal layout; 0 for kernel 3).
 * hydro_planes: copy nk whole planes [k0, k0 + nk) of a state buffer out of (dir 0) or into (dir 1) the context.
 *   which 0: the current state (state n; after a completed step state n+1); which 1: the stage-1 state '.
 *   The layout is opaque: the bytes are only meant for the same planes of another context with the same nx, ny,
 *   precision and viscosity (paper_1802_04449_b200/slabs.py).  Stream-ordered; host buffers synchronise. */
int hydro_stage(hydro_ctx *ctx, int stage);
size_t hydro_plane_bytes(const hydro_ctx *ctx);
int hydro_planes(hydro_ctx *ctx, int which, int k0, int nk, void *buf, int dir, int mem);

/* Read the state: e [nz][ny][nx], u = u~^mu [4][nz][ny][nx], pi = pi~ [10][nz][ny][nx]; any may be
 * NULL.  Synchronises the stream when mem == HYDRO_MEM_HOST. */
int hydro_read(hydro_ctx *ctx, void *e, void *u, void *pi, int mem);

/* ---- Freeze-out hypersurface ------------------------------------------------------------------
 * PAPER.md:268 (text under Eq.55): d Sigma_mu is the surface element of the hypersurface of constant freeze-out energy
 * density e_frz; it is found on the GPU during the evolution, next to the e_max reduction that stops the
 * run, so the full field never leaves the device.  The paper does not print the finder; reading A27: the
 * cuboidal surface between two stored time levels a and b (faces between hot, e >= e_frz, and cold 4-D cells; crossing
 * point and fluid state by linear interpolation in e).
 *
 * hydro_freezeout_bytes: size of the DEVICE workspace (two stored levels of 15 words per cell + counters).
 * hydro_freezeout_begin: stores the current state as level a, resets the element counter and the slab index.  The
 *   workspace is caller-owned, 256-byte aligned, and must stay alive while the finder is in use.
 * hydro_freezeout_slab: takes the current state as level b, APPENDS the elements between a and b to keys / rows
 *   (DEVICE arrays of `capacity` int64 keys and capacity x 22 doubles; unordered), then b becomes the new a.
 *     key  = (slab * 4 + dir) * N + cell      dir 0: time-like face of the cell; 1,2,3: face towards +x, +y, +eta_s
 *                                             cell = (k * ny + j) * nx + i; N = nx ny nz
 *     row  = [0:4] tau, x, y, eta_s of the crossing point   [4:8] d Sigma~_mu (covariant tilde components, normal
 *            pointing to the cold side)   [8:11] u~^i   [11] u~^tau   [12:22] pi~ (order of the header)
 *   fp64 arithmetic in both precisions.  *n_total = elements since begin (also those that did not fit), *n_hot = hot
 *   cells of level b (0 <=> e_max < e_frz, the paper's stop criterion).  Synchronises the stream (16 bytes come back).
 *   Returns HYDRO_ENOMEM when n_total exceeds capacity (the elements that did not fit are dropped), HYDRO_ESTATE before
 *   hydro_freezeout_begin.
 * hydro_freezeout_run: repeats { hydro_step(steps_per_slab); hydro_freezeout_slab } until no hot cell is left or
 *   max_slabs slabs are done; *n_slabs = slabs done.
 *
 * hydro_eos_e_of_temperature: the energy density at which the EoS (rule A16: linear in e inside a bracket) has temperature T (GeV),
 *   so that a constant-T_f surface is the constant-e_frz surface at e_frz = e(T_f).  Host arithmetic, no device needed.
 *   HYDRO_EINVAL for a bad table or a table whose T does not increase with e. */
int hydro_eos_e_of_temperature(const hydro_eos *eos, double T, double *e_out);
size_t hydro_freezeout_bytes(const hydro_grid *grid, int precision);
int hydro_freezeout_begin(hydro_ctx *ctx, void *workspace, size_t workspace_bytes, double e_frz);
int hydro_freezeout_slab(hydro_ctx *ctx, long long *keys, double *rows, long long capacity,
                         long long *n_total, long long *n_hot);
int hydro_freezeout_run(hydro_ctx *ctx, int steps_per_slab, int max_slabs, long long *keys, double *rows,
                        long long capacity, long long *n_total, int *n_slabs);

/* Copy the diagnostics to the host (synchronises the stream).  Returns a warning mask. */
int hydro_diag(hydro_ctx *ctx, hydro_diag_t *out);

/* Number of kernel launches issued by this context since create (host counter). */
long long hydro_launch_count(const hydro_ctx *ctx);

/* The stage kernel this context runs (1, 2, 3 or 4): opts->kernel, or what 0 resolved to. */
int hydro_kernel(const hydro_ctx *ctx);

void hydro_destroy(hydro_ctx *ctx);
const char *hydro_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* CLVISC_HYDRO_H */
