/*
 * erf_oracle.h -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded fp64 restatement of one RK3 step of the dry
 * compressible dynamical core described in /root/reference/PAPER.md
 * (ERF, arXiv 2412.04395): Sec. 2.1 Eq. 1-3, 7 (L63-L84), Sec. 2.3 Eq. 9
 * (L100-L104), Sec. 3.1 Eq. 10-13 (L120-L144), Sec. 3.3 (L170), Sec. 3.4
 * (L178-L180), Sec. 3.6 Eq. 17-21 (L196-L215), Appendix A (L577-L593).
 * Where the paper is silent the readings are those listed in DESIGN.md
 * ("D0"); every function in erf_oracle.c cites the passage it follows.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use this library.  It shares no code, header,
 * table or helper with the CUDA path under paper_2412_04395_b200/.
 *
 * All pointers are HOST pointers.  Field layout at this interface is dense,
 * x fastest: rho, rhou, rhov, rhotheta are [nz][ny][nx]; rhow is
 * [nz+1][ny][nx].  rhou[k][j][i] sits on the low-x face of cell i, rhov on
 * the low-y face of cell j, rhow[k] on the low-z face of level k.
 */
#ifndef ERF_ORACLE_H
#define ERF_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct erfo_ctx erfo_ctx;

typedef struct {
  int nx, ny, nz;
  double dx, dy;
  int periodic_x, periodic_y; /* per direction: 1 periodic (L229); 0 open = zero normal gradient [R:G27];
                                 2 inflow at the low side (a Dirichlet column of cells [R:G30]), open at the high side */
} erfo_grid;

typedef struct {
  const double *z_nodes;   /* [(nz+1)][(ny+1)][(nx+1)] node heights or NULL  */
  const double *z_levels;  /* [(nz+1)] face heights (flat grids) or NULL     */
  const double *rho0;      /* [nz][ny][nx] (or [nz] if base_is_1d)           */
  const double *rhotheta0; /* same shape                                      */
  int base_is_1d;
} erfo_metrics;

typedef struct {
  double Rd, cp, g, p00;
  int adv_order_h, adv_order_v; /* 2..6 */
  int diffusion;                /* 0 none, 1 constant, 2 Smagorinsky */
  double nu, alpha_theta;
  double Cs, Pr_t;
  double beta_s;
  double beta_d;
  int substep_mode; /* 1 semi-implicit, 0 none */
  int scalar_adv;   /* advection of the cell-centred scalars theta, phi (L213): 0 = adv_order_h/v (Eq. 17-21);
                       13, 15 = WENO-JS 3rd/5th; 23, 25 = WENO-Z 3rd/5th, the same scheme in all directions */
  /* Rayleigh damping layer (L219; Appendix C, Table C1): depth below the model top (m; 0 = off), strength at
   * the top (1/s), sine-squared ramp; damped fields: bit 1 u, 2 v, 4 w, 8 theta; references u_ref, v_ref (m/s),
   * 0 for w, the base state for theta [R:G28] */
  double ray_depth, ray_coef;
  int ray_fields;
  double ray_uref, ray_vref;
} erfo_params;

/* return 0 on success, negative on error */
int erfo_create(const erfo_grid *, const erfo_metrics *, const erfo_params *, erfo_ctx **out);
int erfo_set_state(erfo_ctx *, const double *rho, const double *rhou, const double *rhov,
                   const double *rhow, const double *rhotheta);
int erfo_rk3_step(erfo_ctx *, double dt, int n_acoustic);
int erfo_get_state(erfo_ctx *, double *rho, double *rhou, double *rhov, double *rhow,
                   double *rhotheta);
void erfo_destroy(erfo_ctx *);

/* One transported scalar rho*phi [nz][ny][nx] (Eq. 4).  Once set, erfo_rk3_step advances it in every
 * RK stage AFTER the acoustic substeps, with the stage-time-averaged normal momenta (L138). */
int erfo_set_scalar(erfo_ctx *, const double *rhophi);
int erfo_get_scalar(erfo_ctx *, double *rhophi);

/* Anelastic mode (Sec. 2.2 Eq. 8, Sec. 3.2 Eq. 14-16): one RK2 step of size dt with a projection after each
 * stage; flat, laterally periodic grids only (else -1).  rho of the state is held at the base state rho0; the lagged
 * perturbation pressure p' (zero at first) lives in the context. */
int erfo_anelastic_step(erfo_ctx *, double dt);
int erfo_get_pprime(erfo_ctx *, double *pprime);     /* [nz][ny][nx] */
int erfo_project(erfo_ctx *, double dt);             /* Eq. 16 applied to the current momenta */
int erfo_divergence(erfo_ctx *, double *D);          /* dU/dx + dV/dy + dW/dz of the current momenta, [nz][ny][nx] */

/* ---- per-operator entry points used by the pinning tests ---- */

/* Eq. 17-21 interpolant at the flux point between q[2]=q_{m-1} and q[3]=q_m;
 * q[0..5] = q_{m-3} .. q_{m+2}; sgn = +1/-1 (sign of the advecting flux).
 * order 2..6, or a WENO code 13, 15, 23, 25 (see erfo_params.scalar_adv). */
double erfo_interp(int order, double sgn, const double *q);

/* effective vertical order next to the lids (reading G13) */
int erfo_vertical_order(int requested, int r);

/* Eq. 7 in perturbation form: p' and Exner pi from rho*theta and base rho0*theta0 */
void erfo_eos(double Rd, double cp, double p00, double Theta, double Theta0,
              double *pprime, double *pi);

/* slow right-hand side f(S) (Eq. 1-3) of the CURRENT state; dense outputs,
 * R_W is [nz+1][ny][nx] with zero lids. */
int erfo_slow_rhs(erfo_ctx *, double *R_rho, double *R_U, double *R_V, double *R_W,
                  double *R_Theta);

/* Smagorinsky/constant dynamic viscosity mu [nz][ny][nx] of the current state */
int erfo_viscosity(erfo_ctx *, double *mu);

/* geometry: name in {"hc","zc","hw","hx","hy","hu","hv","sxw","syw","sxu","syv","zw"}.
 * dense [nz+1][ny][nx]; levels a quantity does not have are zero. */
int erfo_get_geometry(erfo_ctx *, const char *name, double *out);

/* Appendix A: run n substeps of size dtau with the CURRENT state as the
 * stage state S^t, given slow tendencies R (dense, R_W [nz+1]) and the
 * perturbation S'' (dense, in/out; W'' is [nz+1]).  */
int erfo_acoustic(erfo_ctx *, double dtau, int n, const double *R_rho, const double *R_U,
                  const double *R_V, const double *R_W, const double *R_Theta, double *rho_pp,
                  double *U_pp, double *V_pp, double *W_pp, double *Theta_pp);

/* rows of the column tridiagonal system (A sub-, D main, C super-diagonal),
 * k = 1..nz-1 stored at index k (index 0 unused), with the CURRENT state as S^t */
int erfo_tridiag_rows(erfo_ctx *, double dtau, int i, int j, double *A, double *D, double *C);

/* substep schedule of stage s in {1,2,3}: count and size */
void erfo_schedule(int stage, double dt, int n_acoustic, int *nsub, double *dtau, double *dts);

#ifdef __cplusplus
}
#endif
#endif
