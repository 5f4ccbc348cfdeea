/*
 * erf_b200.h -- C-ABI of liberf_b200.so: one RK3 step of the dry, compressible,
 * non-hydrostatic dynamical core of ERF (arXiv 2412.04395) on one B200 (sm_100a).
 *
 * PAPER.md = /root/reference/PAPER.md (the paper's text).  What each call computes:
 *   - governing equations, flux form: Sec. 2.1 Eq. 1-3 (L63-L67), EOS Eq. 7 (L80-L82),
 *     perturbation pressure and buoyancy (L84), stress tensor Eq. 9 (L100-L104);
 *   - RK3 stages Eq. 10-13 (L120-L136) with acoustic substepping (L138-L144, L170) in
 *     the perturbation form of Appendix A (L577-L593);
 *   - Arakawa C-grid, terrain-following height coordinate, node heights (L178-L180);
 *   - advective fluxes and the interpolation stencils Eq. 17-21 (L196-L215);
 *   - lateral boundaries periodic or open (L229), slip-wall lids (L231, Table C1), an optional
 *     Rayleigh damping layer under the model top (L219, L622).
 * Where the paper is silent the discrete reading is "D0", listed in DESIGN.md.
 *
 * Conventions.
 *   - Every function returns an int status (ERF_OK = 0, negative = error), never throws,
 *     never prints.  erf_strerror() maps a status to a static string.
 *   - "DEVICE" pointers are CUDA global-memory addresses valid on the current device;
 *     "HOST" pointers are ordinary process memory.  The caller owns every pointer it
 *     passes; the library copies what it needs during the call's enqueued work and never
 *     retains a caller pointer after that work has run on the stream.
 *   - Field layout at the boundary: dense, unpadded, x fastest.  rho, rhou, rhov,
 *     rhotheta are [nz][ny][nx]; rhow is [nz+1][ny][nx].  rhou[k][j][i] sits on the low-x
 *     face of cell i, rhov[k][j][i] on the low-y face of cell j, rhow[k][j][i] on the
 *     low-z face of level k.  All fp64.
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Calls only enqueue work on that stream (erf_create and erf_destroy also
 *     synchronise it).  Using one context from two streams concurrently is undefined.
 *   - There is no CPU fallback: every call fails with ERF_ECUDA if no CUDA device works.
 */
#ifndef ERF_B200_H
#define ERF_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define ERF_OK 0
#define ERF_EINVAL (-1)       /* null pointer, non-positive size, bad order / substep count / dt / option */
#define ERF_EUNSUPPORTED (-2) /* anelastic mode on a terrain or laterally open grid, or with a scalar */
#define ERF_ENOMEM (-3)       /* host or device allocation failed                                */
#define ERF_ECUDA (-4)        /* a CUDA runtime call or kernel launch failed (sticky)            */
#define ERF_ETOOLARGE (-5)    /* erf_poisson_modes_noalloc: nx*ny*nz exceeds ERF_NOALLOC_MAX_VALUES */

typedef struct erf_ctx erf_ctx; /* opaque; owns all internal device memory */

typedef struct {
  int nx, ny, nz;             /* cells */
  double dx, dy;              /* m, uniform (L178) */
  int periodic_x, periodic_y; /* per direction: 1 periodic; 0 open (L229 "periodic, inflow, outflow, or open"):
                                 every ghost value is the nearest interior value (zero normal gradient,
                                 DESIGN.md reading G27); 2 inflow at the low side, open (outflow) at the high
                                 side: the first column of cells -- rho*u on the boundary face included -- is
                                 held at the values given to erf_set_state (reading G30; the five prognostic
                                 fields only: a transported scalar sees the open closure there); non-periodic
                                 grids run the terrain-general kernels                                     */
} erf_grid;

typedef struct {
  const double *z_nodes;   /* DEVICE [(nz+1)][(ny+1)][(nx+1)] node heights, m: terrain lives at
                              nodes, deformation vertical only (L178).  Column nx must repeat
                              column 0 and row ny row 0 (periodic).  NULL => flat grid.        */
  const double *z_levels;  /* HOST [(nz+1)] face heights of a flat (possibly stretched, L180)
                              grid; used only when z_nodes is NULL.                             */
  const double *rho0;      /* DEVICE base-state density (L84): [nz][ny][nx], or [nz] if base_is_1d */
  const double *rhotheta0; /* DEVICE base-state rho0*theta0, same shape; p0 and pi0 follow from
                              Eq. 7 (L80)                                                        */
  int base_is_1d;
} erf_metrics;

typedef struct {
  double Rd, cp, g, p00;        /* 287, 1004.5, 9.81, 1e5 in the paper (L82)                  */
  int adv_order_h, adv_order_v; /* 2..6: Eq. 17-21 (L198-L215); horizontal / vertical (L215)  */
  int diffusion;                /* 0 none, 1 constant nu (L104), 2 Smagorinsky-Lilly (L104)   */
  double nu, alpha_theta;       /* m^2/s, kinematic; mu = rho*nu, K = rho*alpha (+ SGS part)  */
  double Cs, Pr_t;              /* Smagorinsky constant (Table C1), turbulent Prandtl number  */
  double beta_s;                /* off-centring of the vertically implicit solve, 0.1 (L591)  */
  double beta_d;                /* divergence damping (L144), 0.1; 0 switches it off          */
  int substep_mode;             /* 1 semi-implicit substepping (default);
                                   0 none: S_stage = S^n + dt_s f(S) (L140), a test mode      */
  int scalar_adv;               /* advection of the cell-centred scalars theta and phi (L213):
                                   0 = adv_order_h / adv_order_v (Eq. 17-21); 13, 15 = WENO-JS
                                   (Jiang & Shu 1996) of 3rd / 5th order; 23, 25 = WENO-Z (Borges
                                   et al. 2008); a WENO scheme applies in all three directions and
                                   runs on the terrain-general kernels                          */
  double ray_depth, ray_coef;   /* Rayleigh damping layer (L219; Appendix C, Table C1): depth below the
                                   model top in m (0 = off) and strength at the top in 1/s; the strength
                                   ramps as sine squared from 0 at the bottom of the layer               */
  int ray_fields;               /* damped fields: bit 1 u, 2 v, 4 w, 8 theta                             */
  double ray_uref, ray_vref;    /* m/s: u, v relax towards these; w towards 0, theta towards the base
                                   state (reading G28)                                        */
} erf_params;

/* Build a context: copies grid/params, derives all metric terms from the node heights
 * (S0), the base-state p0 and pi0 from Eq. 7, allocates the work arrays of the path
 * that will run (flat grid with a 1-D base state: per-level tables and the fused kernels'
 * arrays; the terrain-general arrays are allocated on first use of that path).
 * Any nz >= 1 is accepted with any advection order: next to the lids the vertical stencil
 * falls back to the widest order of the same family that fits (reading G13), so a
 * grid with fewer levels than the stencil is wide simply runs at lower vertical order.
 * The metrics pointers are read during the call only.  Synchronises cuda_stream. */
int erf_create(const erf_grid *grid, const erf_metrics *metrics, const erf_params *params,
               void *cuda_stream, erf_ctx **out);

/* Copy a state S^n = (rho, rho*u, rho*v, rho*w, rho*theta) from DEVICE arrays into the
 * context and impose the kinematic lid values of rho*w (Omega = 0 at k = 0 and k = nz). */
int erf_set_state(erf_ctx *ctx, const double *rho, const double *rhou, const double *rhov,
                  const double *rhow, const double *rhotheta, void *cuda_stream);

/* Advance the state by one RK3 step of size dt (Eq. 11-13).  n_acoustic = number
 * of acoustic substeps per dt: even and >= 2 (L170); RK stage 1 takes one substep of dt/3,
 * stage 2 n_acoustic/2 and stage 3 n_acoustic substeps of dt/n_acoustic.  Enqueue only. */
int erf_rk3_step(erf_ctx *ctx, double dt, int n_acoustic, void *cuda_stream);

/* Copy the current state into DEVICE arrays (any of them may be NULL = skip). */
int erf_get_state(erf_ctx *ctx, double *rho, double *rhou, double *rhov, double *rhow,
                  double *rhotheta, void *cuda_stream);

/* One transported scalar phi (Eq. 4), passed and returned as rho*phi, DEVICE [nz][ny][nx].  Once set,
 * every erf_rk3_step advances it in each RK stage AFTER the acoustic substeps, advected by the time average over
 * the stage of the normal momenta that advanced rho in the substeps (L138) -- so a constant phi stays constant --
 * and diffused with theta's diffusivity.  The dycore keeps its path (on flat periodic grids the fused substep kernel
 * accumulates the averaged momenta); the scalar's own stage runs on the terrain-general kernels, whose 3-D metric arrays
 * erf_set_scalar allocates.  erf_get_scalar before erf_set_scalar: ERF_EINVAL. */
int erf_set_scalar(erf_ctx *ctx, const double *rhophi, void *cuda_stream);
int erf_get_scalar(erf_ctx *ctx, double *rhophi, void *cuda_stream);

/* Anelastic mode (Sec. 2.2 Eq. 8; Sec. 3.2 Eq. 14-16): one RK2 step of size dt of the anelastic
 * equations, no substepping, with a projection after each of the two stages:  dt div(grad psi) = div(rho0 u**),
 * rho0 u* = rho0 u** - dt grad psi,  p' += psi.  The buoyancy is rho0 (theta - theta0)/theta0 g and the pressure
 * gradient uses the lagged p' of the projections only (L96); rho of the state is overwritten by the base state rho0
 * (L94).  The Poisson equation is solved by a discrete Fourier transform in x and y and a tridiagonal system in z per
 * mode (reading G29), so the grid must be flat and periodic in x and y: otherwise ERF_EUNSUPPORTED.
 * Uses the same context, state and parameters as erf_rk3_step; p' starts at zero and lives in the context.
 * A transported scalar (erf_set_scalar) is advanced by erf_rk3_step only: on a context that has one,
 * erf_anelastic_step returns ERF_EUNSUPPORTED and changes nothing (erf_project still works).
 * erf_get_pprime: DEVICE [nz][ny][nx]; ERF_EINVAL before the first anelastic call.
 * erf_project applies the projection alone to the momenta of the current state (tests). */
int erf_anelastic_step(erf_ctx *ctx, double dt, void *cuda_stream);
int erf_get_pprime(erf_ctx *ctx, double *pprime, void *cuda_stream);
int erf_project(erf_ctx *ctx, double dt, void *cuda_stream);

/* The vertical solve of the anelastic Poisson equation (Sec. 3.2 Eq. 16; reading G29) WITHOUT ANY
 * ALLOCATION and without a context, for callers that are not free to take device memory when they call: a solver that
 * runs inside an application whose own allocator already holds the whole GPU (a cudaMalloc from this library would fail
 * there, or eat into what that allocator expects to find), a job held to a memory budget its own buffers use up, or a
 * time loop that cannot afford the device-wide synchronisation an allocation brings.  Every other entry point of this
 * library goes through an erf_ctx, and erf_create (and the first use of some paths) allocates; this one never calls
 * cudaMalloc, cudaFree or any library routine that does.
 *
 * What it computes: the step erf_project performs between its forward and inverse horizontal transforms.  On entry
 * (hat_re, hat_im) hold the discrete Fourier coefficients in x and y of the divergence div(rho0 u), DEVICE
 * [nz][ny][nx] each with the x-wavenumber m fastest (unnormalised forward transform, the layout of a plain 2-D FFT of
 * every level); on return they hold the coefficients of psi, the solution of
 *     [lx(m) + ly(n)] P_k + [ (P_{k+1} - P_k)/dzw[k+1] - (P_k - P_{k-1})/dzw[k] ] / dz[k] = Dhat_k / dt
 * with lx(m) = -(4/dx^2) sin^2(pi m/nx), ly(n) = -(4/dy^2) sin^2(pi n/ny), no-gradient lids, and P_0 = 0 for the
 * mean mode (0, 0).  dz: DEVICE [nz] cell thicknesses; dzw: DEVICE [nz+1] distances between cell centres across face k
 * (entries 1 .. nz-1 are read).  The caller owns all four arrays; hat_re / hat_im are overwritten in place.  Enqueue
 * only, on cuda_stream; the arrays must stay valid until that work has run.
 *
 * The work space -- one double per (mode, level) -- is a fixed array of ERF_NOALLOC_MAX_VALUES doubles (8 MiB) built
 * into the library's device code.  Consequences the caller has to know:
 *   - LIMIT: nx*ny*nz <= ERF_NOALLOC_MAX_VALUES (for example 128 x 128 x 64); anything larger is refused with
 *     ERF_ETOOLARGE before any CUDA call, and nothing is written.  Larger problems need erf_project and a context.
 *   - Every GPU on which the process uses liberf_b200.so holds these 8 MiB until the process ends, used or not.
 *   - There is ONE array per GPU, shared by every call: two calls that may run at the same time on one GPU (two
 *     streams, two host threads) corrupt each other's result silently.  Keep calls on a GPU ordered on one stream, or
 *     order them with events.  The array keeps the last call's values between calls; the solve does not depend on
 *     them (each entry is written before it is read), so nothing needs clearing.
 *   - The FIRST call on each GPU looks up the array's device address (and may make the CUDA runtime load the library's
 *     device code onto that GPU); later calls only launch the kernel.  Make that first call with the GPU current,
 *     during set-up, before any stream capture is begun in the process.
 * Returns ERF_EINVAL for a null pointer or a non-positive size, dx, dy or dt; ERF_ECUDA if the address look-up or the
 * launch fails. */
#define ERF_NOALLOC_MAX_VALUES 1048576
int erf_poisson_modes_noalloc(int nx, int ny, int nz, double dx, double dy, double dt, const double *dz,
                              const double *dzw, double *hat_re, double *hat_im, void *cuda_stream);

/* Free everything; erf_destroy(NULL) is a no-op. */
void erf_destroy(erf_ctx *ctx);

const char *erf_strerror(int code);

/* ---- per-operator entry points (used by the parity tests and the profiler) ---- */

/* The slow right-hand side f(S) of Eq. 1-3 for the CURRENT state: advection (L196-L215),
 * diffusion (Eq. 9), pressure gradient and buoyancy (L84).  DEVICE outputs, dense;
 * R_W is [nz+1][ny][nx] with zero lids.  Any output may be NULL. */
int erf_slow_rhs(erf_ctx *ctx, double *R_rho, double *R_U, double *R_V, double *R_W,
                 double *R_Theta, void *cuda_stream);

/* Appendix A: n substeps of size dtau about the CURRENT state as stage state S^t, given the
 * slow tendencies R and the perturbation S'' (DEVICE, dense, in/out; W'' is [nz+1]). */
int erf_acoustic(erf_ctx *ctx, double dtau, int n, const double *R_rho, const double *R_U,
                 const double *R_V, const double *R_W, const double *R_Theta, double *rho_pp,
                 double *U_pp, double *V_pp, double *W_pp, double *Theta_pp, void *cuda_stream);

/* =====================================================================================
 * DIAGNOSTICS -- not part of the five-call boundary; used by tests/ and bench.py only.
 * Nothing here changes what a step computes; options select between kernels that compute
 * the same discrete operators.
 * ===================================================================================== */

/* Select the kernel path: ERF_PATH_AUTO picks the fused kernels where they apply;
 * ERF_PATH_GENERAL forces the unfused, terrain-general kernels (one kernel per operator,
 * every intermediate field in HBM), kept as an on-device cross-check of the fused ones. */
#define ERF_PATH_AUTO 0
#define ERF_PATH_GENERAL 1
int erf_set_path(erf_ctx *ctx, int path);

/* erf_set_option(ctx, key, value): explicit, per-context replacements of what used to be a
 * process-wide environment variable.  Unknown key or value: ERF_EINVAL.
 *   ERF_OPT_VARIANT  value = OR of ERF_VARIANT_* bits, 0 = the defaults that bench.py times.
 *   ERF_OPT_GRAPH    value = 1: erf_rk3_step captures the launches of a step into a CUDA graph
 *                    on first use (per (dt, n_acoustic)) and replays it; 0 (default) = plain
 *                    stream launches.  Meant for grids so small that a step is launch-bound. */
#define ERF_OPT_VARIANT 1
#define ERF_OPT_GRAPH 2
#define ERF_VARIANT_ADV_SPLIT_MASK 192  /* legacy advection: 64 one, 128 two, 192 four launches */
#define ERF_VARIANT_DIFF_SPLIT 1024     /* momentum and scalar diffusion in separate launches  */
#define ERF_VARIANT_FORCE_COLUMN 4096   /* thread-per-column substep kernel on every flat grid */
#define ERF_VARIANT_SPLIT_SLOW_RHS 8192 /* round-1 slow RHS: k_prim_flat + per-field advection */
#define ERF_VARIANT_FORCE_TILE 16384    /* column-tile substep kernel on every flat grid       */
int erf_set_option(erf_ctx *ctx, int key, long long value);

/* Number of kernels launched by this context so far (for bench.py's gpu_launches). */
long long erf_launch_count(const erf_ctx *ctx);

/* Per-kernel device timing.  erf_set_timing(ctx, 1) makes every subsequent call bracket each
 * kernel (or group of small kernels) with CUDA events on the call's stream; erf_get_timing
 * synchronises, and returns for class id (0 <= id < ERF_TIMING_CLASSES) the number of bracketed
 * launches and their total device time in milliseconds since the last erf_reset_timing.
 * erf_timing_name(id) is a static string.  Off by default (no events are recorded). */
#define ERF_TIMING_CLASSES 8
int erf_set_timing(erf_ctx *ctx, int on);
int erf_get_timing(erf_ctx *ctx, int id, long long *launches, double *total_ms);
int erf_reset_timing(erf_ctx *ctx);
const char *erf_timing_name(int id);

/* The fp64 FMA peak of the current device, measured with a register-resident DFMA kernel (8 independent chains
 * per thread, best of 3 timed launches on cuda_stream; synchronises).  *tflops counts an FMA as 2 flop.  This is the
 * denominator for the fp64-pipe utilisation of the slow right-hand-side kernels. */
int erf_measure_fp64_peak(double *tflops, void *cuda_stream);

/* Device bytes owned by the context. */
long long erf_device_bytes(const erf_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
