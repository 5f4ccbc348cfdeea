/*
 * erf_oracle.c -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * One RK3 step of ERF's dry compressible dynamical core, written out step by
 * step in the paper's order and notation (PAPER.md = /root/reference/PAPER.md,
 * arXiv 2412.04395).  fp64, single thread, every intermediate field is a full
 * 3-D array, no blocking / fusion / reordering.  Build with
 *     gcc -O2 -ffp-contract=off -fPIC -shared
 * Readings of passages where the paper is silent or garbled are tagged
 * [R:Gn] and listed under the same tag in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_*.py): stencil weights / polynomial
 * exactness (Eq. 17-21), EOS closed form (Eq. 7), RK3 amplification factor
 * (Eq. 11-13), rest state, mass / rho*theta conservation, free-stream
 * preservation over terrain, discrete acoustic dispersion (horizontal and
 * vertical), gravity-wave frequency, column solve against a dense coupled
 * solve of Appendix A, Smagorinsky closed forms, substep schedule;
 * tests/test_oracle_pins_r2.py: sign and factor of every stress component
 * and of the scalar diffusion flux on single Fourier / cosine modes (Eq. 2-3,
 * Eq. 9), mu = rho*nu with edge means, K = mu_t/Pr_t, the divergence-damping
 * recurrence (L144), kinematic lids over terrain, chain-rule metric terms of
 * the strain and of the scalar flux on Cartesian-linear fields;
 * test_oracle_scalar.py (Eq. 4 with the averaged momenta), test_oracle_weno.py
 * (WENO-JS / WENO-Z from their definitions), test_oracle_open_rayleigh.py
 * (open and inflow boundaries, Rayleigh layer), test_oracle_anelastic.py
 * (Eq. 8, 14-16: dense brute-force projection, invariants, RK2 polynomial);
 * test_oracle_symmetry.py (round 3): slow_rhs, acoustic and a full step
 * commute with the reflections of x and y and the exchange of x and y (flat
 * and over an unsymmetric periodic terrain, orders 2-6) and, on a uniform
 * column, with the reflection of z together with g -> -g: pins every two-
 * and four-point mean and metric factor whose one-sided replacement is not
 * symmetric (face density, face pi, edge viscosity, flux means, hu, hy, the
 * metric pressure gradient); test_oracle_appendix_a_terrain.py (round 3):
 * the rho'' and Theta'' equations of a substep over terrain as residuals
 * rebuilt with numpy from the node heights (pins the size and averaging of
 * omega, hx / hy, the beta weights).  Still unpinned: hw against hc in R_W
 * over terrain and the chain-rule terms of the stress divergence.
 * The full nonlinear step on the benchmark configurations has no value
 * printed in the paper: "parity unpinned" beyond those invariants.
 *
 * Notation.  Cells (i,j,k), x fastest.  State S = (rho, U, V, W, Theta),
 * Theta = rho*theta.  U on x-faces (i-1/2,j,k), V on y-faces, W on z-faces
 * k = 0..nz.  Laterally periodic, open or inflow/outflow per direction; rigid
 * free-slip lids at k = 0 and k = nz.  Work arrays carry NG ghost cells in x
 * and y, filled by the lateral boundary rule after every field is computed.
 */
#include "erf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define NG 4

enum { RHO = 0, UU = 1, VV = 2, WW = 3, TH = 4 };

struct erfo_ctx {
  int nx, ny, nz;
  int perx, pery; /* lateral boundary per direction: 1 periodic, 0 open */
  int inx, iny;   /* inflow: the first column (row) of cells is held at the values given to erfo_set_state [R:G30] */
  double *inflow[5];
  int flat;       /* z_nodes == NULL: level heights depend on k only */
  double dx, dy;
  erfo_params p;
  double gam, cv, rdocv; /* gamma = cp/(cp-Rd) (L82); cv = cp-Rd; Rd/cv */
  size_t sj, sk, n;      /* strides of the ghosted arrays, and their length */
  /* geometry, S0 [R:G14] */
  double *zxf, *zyf, *zw;          /* levels 0..nz   */
  double *hx, *hy, *hc, *zc;       /* levels 0..nz-1 */
  double *hw;                      /* levels 1..nz-1 */
  double *hu, *hv;                 /* levels 0..nz-1 */
  double *sxw, *syw;               /* levels 0..nz   */
  double *sxu, *syv;               /* levels 0..nz-1 */
  /* base state */
  double *rho0, *Th0, *p0, *pi0;
  /* state at time level n */
  double *S[5];
  /* one transported scalar rho*phi (Eq. 4); NULL until erfo_set_scalar */
  double *Q;
  /* anelastic mode (Sec. 2.2, 3.2): the lagged perturbation pressure p' of the projection; NULL until first used */
  double *pan;
};

/* ------------------------------------------------------------------ */
/* array helpers                                                       */
/* ------------------------------------------------------------------ */

static size_t IX(const erfo_ctx *c, int i, int j, int k) {
  return (size_t)k * c->sk + (size_t)(j + NG) * c->sj + (size_t)(i + NG);
}

static double *fnew(const erfo_ctx *c) { return (double *)calloc(c->n, sizeof(double)); }

static int wrapi(int a, int n) {
  int r = a % n;
  return r < 0 ? r + n : r;
}

static int clampi(int a, int n) { return a < 0 ? 0 : (a >= n ? n - 1 : a); }

/* lateral boundary ("periodic, inflow, outflow, or open"), one choice per direction:
 * periodic: ghost = image of the interior; open: ghost = the nearest interior value (zero normal gradient) for
 * EVERY field, including the normal momentum, whose first face beyond the last stored one (U at i = nx, V at
 * j = ny) is such a ghost [R:G27] */
static void fill_lateral(const erfo_ctx *c, double *f) {
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= c->nz; k++)
    for (int j = -NG; j < c->ny + NG; j++)
      for (int i = -NG; i < c->nx + NG; i++)
        if (i < 0 || i >= c->nx || j < 0 || j >= c->ny) {
          int is = c->perx ? wrapi(i, c->nx) : clampi(i, c->nx);
          int js = c->pery ? wrapi(j, c->ny) : clampi(j, c->ny);
          f[IX(c, i, j, k)] = f[IX(c, is, js, k)];
        }
}

static void put_dense(const erfo_ctx *c, double *f, const double *dense, int nlev) {
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nlev; k++)
    for (int j = 0; j < c->ny; j++)
      for (int i = 0; i < c->nx; i++)
        f[IX(c, i, j, k)] = dense[((size_t)k * c->ny + j) * c->nx + i];
  fill_lateral(c, f);
}

static void get_dense(const erfo_ctx *c, const double *f, double *dense, int nlev) {
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nlev; k++)
    for (int j = 0; j < c->ny; j++)
      for (int i = 0; i < c->nx; i++)
        dense[((size_t)k * c->ny + j) * c->nx + i] = f[IX(c, i, j, k)];
}

/* ------------------------------------------------------------------ */
/* Eq. 17-21: interpolation to a flux point                            */
/* ------------------------------------------------------------------ */

/* PAPER.md L200-L211.  q[0..5] = q_{m-3}, q_{m-2}, q_{m-1}, q_m, q_{m+1}, q_{m+2};
 * the flux point is m-1/2.  Eq. 17 (2nd), the unnumbered 4th-order line,
 * Eq. 19 (6th), Eq. 20 (3rd) as printed; Eq. 21 (5th) with the sign and the
 * index of its first bracket corrected [R:G1]: as printed it is neither
 * upwind nor 5th order. */
/* WENO reconstruction of cell-centred scalars ("third-, fifth-... order WENO ... the classic WENO-JS
 * (Jiang & Shu, 1996), WENO-Z (Borges et al., 2008)"; the paper gives no formulas -- these are the cited schemes
 * as published [R:G26]).  kind 1 = JS, 2 = Z; ord 3 or 5.  v = the upwind-ordered cell values: for ord 5
 * v[0..4] = cells i-2 .. i+2 around the upwind cell i, value at its downwind face i+1/2; for ord 3 v[1..3].
 *   JS:  omega_k ~ d_k / (eps + beta_k)^2,            eps = 1e-6
 *   Z :  omega_k ~ d_k (1 + tau / (beta_k + eps)),    tau = |beta_0 - beta_last|, eps = 1e-40
 * with the ideal weights d = (1/10, 6/10, 3/10) resp. (1/3, 2/3) and the Jiang-Shu smoothness indicators. */
static double weno_face(int kind, int ord, const double *v) {
  if (ord == 3) {
    double p0 = 0.5 * (3.0 * v[2] - v[1]), p1 = 0.5 * (v[2] + v[3]);
    double b0 = (v[2] - v[1]) * (v[2] - v[1]), b1 = (v[3] - v[2]) * (v[3] - v[2]);
    double a0, a1;
    if (kind == 1) {
      a0 = (1.0 / 3.0) / ((1e-6 + b0) * (1e-6 + b0));
      a1 = (2.0 / 3.0) / ((1e-6 + b1) * (1e-6 + b1));
    } else {
      double tau = fabs(b0 - b1);
      a0 = (1.0 / 3.0) * (1.0 + tau / (b0 + 1e-40));
      a1 = (2.0 / 3.0) * (1.0 + tau / (b1 + 1e-40));
    }
    return (a0 * p0 + a1 * p1) / (a0 + a1);
  }
  double p0 = (2.0 * v[0] - 7.0 * v[1] + 11.0 * v[2]) / 6.0;
  double p1 = (-v[1] + 5.0 * v[2] + 2.0 * v[3]) / 6.0;
  double p2 = (2.0 * v[2] + 5.0 * v[3] - v[4]) / 6.0;
  double t0 = v[0] - 2.0 * v[1] + v[2], u0 = v[0] - 4.0 * v[1] + 3.0 * v[2];
  double t1 = v[1] - 2.0 * v[2] + v[3], u1 = v[1] - v[3];
  double t2 = v[2] - 2.0 * v[3] + v[4], u2 = 3.0 * v[2] - 4.0 * v[3] + v[4];
  double b0 = 13.0 / 12.0 * t0 * t0 + 0.25 * u0 * u0;
  double b1 = 13.0 / 12.0 * t1 * t1 + 0.25 * u1 * u1;
  double b2 = 13.0 / 12.0 * t2 * t2 + 0.25 * u2 * u2;
  double a0, a1, a2;
  if (kind == 1) {
    a0 = 0.1 / ((1e-6 + b0) * (1e-6 + b0));
    a1 = 0.6 / ((1e-6 + b1) * (1e-6 + b1));
    a2 = 0.3 / ((1e-6 + b2) * (1e-6 + b2));
  } else {
    double tau = fabs(b0 - b2);
    a0 = 0.1 * (1.0 + tau / (b0 + 1e-40));
    a1 = 0.6 * (1.0 + tau / (b1 + 1e-40));
    a2 = 0.3 * (1.0 + tau / (b2 + 1e-40));
  }
  return (a0 * p0 + a1 * p1 + a2 * p2) / (a0 + a1 + a2);
}

/* order codes: 2..6 = Eq. 17-21; 10*kind + ord = WENO (13, 15 = JS3, JS5; 23, 25 = Z3, Z5) */
double erfo_interp(int order, double sgn, const double *q) {
  if (order >= 10) { /* upwind-ordered values: the flux point lies between q[2] and q[3] */
    double v[5];
    if (sgn > 0.0) { v[0] = q[0]; v[1] = q[1]; v[2] = q[2]; v[3] = q[3]; v[4] = q[4]; }
    else           { v[0] = q[5]; v[1] = q[4]; v[2] = q[3]; v[3] = q[2]; v[4] = q[1]; }
    return weno_face(order / 10, order % 10, v);
  }
  double q2 = 0.5 * (q[3] + q[2]);
  if (order == 2) return q2;
  double q4 = 7.0 / 12.0 * (q[3] + q[2]) - 1.0 / 12.0 * (q[4] + q[1]);
  if (order == 4) return q4;
  if (order == 3) return q4 + sgn / 12.0 * ((q[4] - q[1]) - 3.0 * (q[3] - q[2]));
  double q6 = 37.0 / 60.0 * (q[3] + q[2]) - 2.0 / 15.0 * (q[4] + q[1]) + 1.0 / 60.0 * (q[5] + q[0]);
  if (order == 6) return q6;
  /* order == 5 */
  return q6 - sgn / 60.0 * ((q[5] - q[0]) - 5.0 * (q[4] - q[1]) + 10.0 * (q[3] - q[2]));
}

/* [R:G13] order reduction next to the lids.  r = min(#valid points below,
 * #valid points above) the flux point. */
int erfo_vertical_order(int requested, int r) {
  if (requested >= 10) { /* WENO: the 5-cell stencil needs 3 valid cells on either side, the 3-cell one 2 */
    if (r >= (requested % 10 + 1) / 2) return requested;
    return r >= 2 ? 10 * (requested / 10) + 3 : 2;
  }
  int need = (requested + 1) / 2;
  if (r >= need) return requested;
  if (r >= 2 && requested >= 3) return (requested & 1) ? 3 : 4;
  return 2;
}

static double sgn_of(double m) { return m < 0.0 ? -1.0 : 1.0; } /* sign(0)=+1 [R:G19] */

/* interpolate f along x to the point between (m-1,j,k) and (m,j,k) */
static double interp_x(const erfo_ctx *c, const double *f, int m, int j, int k, int order,
                       double M) {
  double q[6];
  for (int n = 0; n < 6; n++) q[n] = f[IX(c, m - 3 + n, j, k)];
  return erfo_interp(order, sgn_of(M), q);
}

static double interp_y(const erfo_ctx *c, const double *f, int i, int m, int k, int order,
                       double M) {
  double q[6];
  for (int n = 0; n < 6; n++) q[n] = f[IX(c, i, m - 3 + n, k)];
  return erfo_interp(order, sgn_of(M), q);
}

/* interpolate f along z to the point between levels m-1 and m; valid levels
 * of f are lo..hi (cells 0..nz-1, or faces 0..nz for w) */
static double interp_z(const erfo_ctx *c, const double *f, int i, int j, int m, int lo, int hi,
                       int order_req, double M) {
  int below = m - lo;     /* points m-1, m-2, ... lo */
  int above = hi - m + 1; /* points m, m+1, ... hi   */
  int r = below < above ? below : above;
  int order = erfo_vertical_order(order_req, r);
  int half = (order % 10 + 1) / 2;
  double q[6] = {0, 0, 0, 0, 0, 0};
  for (int n = 3 - half; n < 3 + half; n++) q[n] = f[IX(c, i, j, m - 3 + n)];
  return erfo_interp(order, sgn_of(M), q);
}

/* ------------------------------------------------------------------ */
/* Eq. 7: equation of state in perturbation form                       */
/* ------------------------------------------------------------------ */

/* PAPER.md L80-L84.  p = P00 (Rd Theta / P00)^gamma, p' = p - p0 with p0
 * defined by the same formula from Theta0, hence p' = p0 [(Theta/Theta0)^gamma - 1],
 * evaluated as p0 * expm1(gamma * log1p((Theta-Theta0)/Theta0)) [R:S1] so that
 * the subtraction of two 1e5 Pa numbers never happens.  Exner function
 * pi = (p/P00)^(Rd/cp) = (Rd Theta/P00)^(Rd/cv)  (L84, L587). */
void erfo_eos(double Rd, double cp, double p00, double Theta, double Theta0, double *pprime,
              double *pi) {
  double cv = cp - Rd;
  double gam = cp / cv;
  double p0 = p00 * pow(Rd * Theta0 / p00, gam);
  *pprime = p0 * expm1(gam * log1p((Theta - Theta0) / Theta0));
  *pi = pow(Rd * Theta / p00, Rd / cv);
}

/* ------------------------------------------------------------------ */
/* S0: geometry from node heights                                      */
/* ------------------------------------------------------------------ */

/* terrain given at nodes, deformation vertical only.  All
 * metric quantities are differences of node heights [R:G14]. */
static void build_geometry(erfo_ctx *c, const double *zn) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
#define ZN(i, j, k) zn[((size_t)(k) * (ny + 1) + (j)) * (nx + 1) + (i)]
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        c->zxf[IX(c, i, j, k)] = 0.5 * (ZN(i, j, k) + ZN(i, j + 1, k));
        c->zyf[IX(c, i, j, k)] = 0.5 * (ZN(i, j, k) + ZN(i + 1, j, k));
        c->zw[IX(c, i, j, k)] =
            0.25 * (ZN(i, j, k) + ZN(i + 1, j, k) + ZN(i, j + 1, k) + ZN(i + 1, j + 1, k));
      }
#undef ZN
  fill_lateral(c, c->zxf);
  fill_lateral(c, c->zyf);
  fill_lateral(c, c->zw);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        c->hx[IX(c, i, j, k)] = c->zxf[IX(c, i, j, k + 1)] - c->zxf[IX(c, i, j, k)];
        c->hy[IX(c, i, j, k)] = c->zyf[IX(c, i, j, k + 1)] - c->zyf[IX(c, i, j, k)];
        c->hc[IX(c, i, j, k)] = c->zw[IX(c, i, j, k + 1)] - c->zw[IX(c, i, j, k)];
        c->zc[IX(c, i, j, k)] = 0.5 * (c->zw[IX(c, i, j, k)] + c->zw[IX(c, i, j, k + 1)]);
      }
  fill_lateral(c, c->hx);
  fill_lateral(c, c->hy);
  fill_lateral(c, c->hc);
  fill_lateral(c, c->zc);
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++)
        c->hw[IX(c, i, j, k)] = c->zc[IX(c, i, j, k)] - c->zc[IX(c, i, j, k - 1)];
  fill_lateral(c, c->hw);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        c->hu[IX(c, i, j, k)] = 0.5 * (c->hc[IX(c, i - 1, j, k)] + c->hc[IX(c, i, j, k)]);
        c->hv[IX(c, i, j, k)] = 0.5 * (c->hc[IX(c, i, j - 1, k)] + c->hc[IX(c, i, j, k)]);
        c->sxu[IX(c, i, j, k)] = (c->zc[IX(c, i, j, k)] - c->zc[IX(c, i - 1, j, k)]) / c->dx;
        c->syv[IX(c, i, j, k)] = (c->zc[IX(c, i, j, k)] - c->zc[IX(c, i, j - 1, k)]) / c->dy;
      }
  fill_lateral(c, c->hu);
  fill_lateral(c, c->hv);
  fill_lateral(c, c->sxu);
  fill_lateral(c, c->syv);
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        c->sxw[IX(c, i, j, k)] = (c->zxf[IX(c, i + 1, j, k)] - c->zxf[IX(c, i, j, k)]) / c->dx;
        c->syw[IX(c, i, j, k)] = (c->zyf[IX(c, i, j + 1, k)] - c->zyf[IX(c, i, j, k)]) / c->dy;
      }
  fill_lateral(c, c->sxw);
  fill_lateral(c, c->syw);
}

/* Inflow boundary ("inflow", Table C1 "Inflow, Outflow"; no discrete form in the paper) [R:G30]: the
 * first column of cells at the low-x side -- rho, rho*theta, rho*v, rho*w of cell i = 0 and rho*u on its low face,
 * which is the boundary face -- is held at the values the state was given (erfo_set_state): a Dirichlet column.  Beyond
 * it the open closure applies (ghost = nearest interior value = the inflow value); the far side is open (outflow).
 * Imposed on every stage result; likewise in y. */
static void impose_inflow(const erfo_ctx *c, double *const S[5]) {
  if (c->inx)
    for (int m = 0; m < 5; m++)
      for (int k = 0; k <= c->nz; k++)
        for (int j = 0; j < c->ny; j++) S[m][IX(c, 0, j, k)] = c->inflow[m][IX(c, 0, j, k)];
  if (c->iny)
    for (int m = 0; m < 5; m++)
      for (int k = 0; k <= c->nz; k++)
        for (int i = 0; i < c->nx; i++) S[m][IX(c, i, 0, k)] = c->inflow[m][IX(c, i, 0, k)];
}

/* ------------------------------------------------------------------ */
/* lids: kinematic boundary condition on W  [R:G15]                    */
/* ------------------------------------------------------------------ */

/* Rigid lids: the contravariant flux Omega vanishes at k=0 and k=nz, i.e.
 * W = sxw*u-average + syw*v-average taken from the adjacent level
 * (zero on flat lids). Needs U,V ghosts filled. */
static void impose_lids(const erfo_ctx *c, const double *U, const double *V, double *W) {
  int nz = c->nz;
  for (int j = 0; j < c->ny; j++)
    for (int i = 0; i < c->nx; i++) {
      W[IX(c, i, j, 0)] =
          c->sxw[IX(c, i, j, 0)] * 0.5 * (U[IX(c, i, j, 0)] + U[IX(c, i + 1, j, 0)]) +
          c->syw[IX(c, i, j, 0)] * 0.5 * (V[IX(c, i, j, 0)] + V[IX(c, i, j + 1, 0)]);
      W[IX(c, i, j, nz)] =
          c->sxw[IX(c, i, j, nz)] * 0.5 * (U[IX(c, i, j, nz - 1)] + U[IX(c, i + 1, j, nz - 1)]) +
          c->syw[IX(c, i, j, nz)] * 0.5 * (V[IX(c, i, j, nz - 1)] + V[IX(c, i, j + 1, nz - 1)]);
    }
  fill_lateral(c, W);
}

/* contravariant vertical mass flux, PAPER.md L196 ("rho*Omega ... normal to
 * the face"), discrete form [R:G14]: Omega = W - sxw*avg4(U) - syw*avg4(V)
 * on interior faces, 0 on the lids. */
static void contravariant_flux(const erfo_ctx *c, const double *U, const double *V,
                               const double *W, double *Om) {
  int nz = c->nz;
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= nz; k++)
    for (int j = 0; j < c->ny; j++)
      for (int i = 0; i < c->nx; i++) {
        double om = 0.0;
        if (k >= 1 && k <= nz - 1) {
          double ubar = 0.25 * (U[IX(c, i, j, k - 1)] + U[IX(c, i + 1, j, k - 1)] +
                                U[IX(c, i, j, k)] + U[IX(c, i + 1, j, k)]);
          double vbar = 0.25 * (V[IX(c, i, j, k - 1)] + V[IX(c, i, j + 1, k - 1)] +
                                V[IX(c, i, j, k)] + V[IX(c, i, j + 1, k)]);
          om = W[IX(c, i, j, k)] - c->sxw[IX(c, i, j, k)] * ubar - c->syw[IX(c, i, j, k)] * vbar;
        }
        Om[IX(c, i, j, k)] = om;
      }
  fill_lateral(c, Om);
}

/* ------------------------------------------------------------------ */
/* primitive fields of a state                                         */
/* ------------------------------------------------------------------ */

typedef struct {
  double *theta, *pp, *pi; /* cells */
  double *u, *v, *w;       /* faces; advected "primitive variable" (L196) */
} prim_t;

/* S1 + face velocities.  theta = Theta/rho; p', pi from Eq. 7; velocity =
 * momentum / face density, face density = arithmetic mean of the two
 * adjacent cells [R:G11]; at the lids rho_w = adjacent cell. */
static void primitives(const erfo_ctx *c, double *const S[5], prim_t *q) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        q->theta[a] = S[TH][a] / S[RHO][a];
        q->pp[a] = c->p0[a] * expm1(c->gam * log1p((S[TH][a] - c->Th0[a]) / c->Th0[a]));
        q->pi[a] = pow(c->p.Rd * S[TH][a] / c->p.p00, c->rdocv);
        q->u[a] = S[UU][a] / (0.5 * (S[RHO][IX(c, i - 1, j, k)] + S[RHO][a]));
        q->v[a] = S[VV][a] / (0.5 * (S[RHO][IX(c, i, j - 1, k)] + S[RHO][a]));
      }
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        double rw;
        if (k == 0) rw = S[RHO][a];
        else if (k == nz) rw = S[RHO][IX(c, i, j, nz - 1)];
        else rw = 0.5 * (S[RHO][IX(c, i, j, k - 1)] + S[RHO][a]);
        q->w[a] = S[WW][a] / rw;
      }
  fill_lateral(c, q->theta);
  fill_lateral(c, q->pp);
  fill_lateral(c, q->pi);
  fill_lateral(c, q->u);
  fill_lateral(c, q->v);
  fill_lateral(c, q->w);
}

/* ------------------------------------------------------------------ */
/* S2: advection  (Eq. 1-3 first terms)            */
/* ------------------------------------------------------------------ */

static void advection(const erfo_ctx *c, double *const S[5], const prim_t *q, double *R[5]) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  int oh = c->p.adv_order_h, ov = c->p.adv_order_v;
  /* cell-centred scalars may use a WENO scheme instead, the same in all directions (L213) */
  int ohs = c->p.scalar_adv ? c->p.scalar_adv : oh, ovs = c->p.scalar_adv ? c->p.scalar_adv : ov;
  double dx = c->dx, dy = c->dy;
  /* mass fluxes through cell faces: Fx = hx U, Fy = hy V (face-height
   * weighted, finite-volume form [R:G14]) and Omega */
  double *Fx = fnew(c), *Fy = fnew(c), *Om = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        Fx[a] = c->hx[a] * S[UU][a];
        Fy[a] = c->hy[a] * S[VV][a];
      }
  fill_lateral(c, Fx);
  fill_lateral(c, Fy);
  contravariant_flux(c, S[UU], S[VV], S[WW], Om);

#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        /* ---- continuity, Eq. 1 (L63) ---- */
        double fxm = Fx[IX(c, i, j, k)], fxp = Fx[IX(c, i + 1, j, k)];
        double fym = Fy[IX(c, i, j, k)], fyp = Fy[IX(c, i, j + 1, k)];
        double omm = Om[IX(c, i, j, k)], omp = Om[IX(c, i, j, k + 1)];
        R[RHO][a] = -((fxp - fxm) / dx + (fyp - fym) / dy + (omp - omm)) / c->hc[a];
        /* ---- rho*theta, Eq. 3 first term (L67): flux = normal momentum at
         * the face times theta interpolated to the face (L196) ---- */
        double txm = fxm * interp_x(c, q->theta, i, j, k, ohs, fxm);
        double txp = fxp * interp_x(c, q->theta, i + 1, j, k, ohs, fxp);
        double tym = fym * interp_y(c, q->theta, i, j, k, ohs, fym);
        double typ = fyp * interp_y(c, q->theta, i, j + 1, k, ohs, fyp);
        double tzm = (k >= 1) ? omm * interp_z(c, q->theta, i, j, k, 0, nz - 1, ovs, omm) : 0.0;
        double tzp =
            (k + 1 <= nz - 1) ? omp * interp_z(c, q->theta, i, j, k + 1, 0, nz - 1, ovs, omp) : 0.0;
        R[TH][a] = -((txp - txm) / dx + (typ - tym) / dy + (tzp - tzm)) / c->hc[a];

        /* ---- U momentum, Eq. 2 first term (L65).  "Spatial averaging is
         * utilized to obtain the normal momentum at the flux location"
         * (L196): two-point arithmetic means [R:G11]. ---- */
        {
          double Mxm = 0.5 * (Fx[IX(c, i - 1, j, k)] + Fx[IX(c, i, j, k)]);     /* centre i-1 */
          double Mxp = 0.5 * (Fx[IX(c, i, j, k)] + Fx[IX(c, i + 1, j, k)]);     /* centre i   */
          double Mym = 0.5 * (Fy[IX(c, i - 1, j, k)] + Fy[IX(c, i, j, k)]);     /* edge j-1/2 */
          double Myp = 0.5 * (Fy[IX(c, i - 1, j + 1, k)] + Fy[IX(c, i, j + 1, k)]);
          double Mzm = 0.5 * (Om[IX(c, i - 1, j, k)] + Om[IX(c, i, j, k)]);     /* edge k-1/2 */
          double Mzp = 0.5 * (Om[IX(c, i - 1, j, k + 1)] + Om[IX(c, i, j, k + 1)]);
          double gxm = Mxm * interp_x(c, q->u, i, j, k, oh, Mxm);     /* between u(i-1), u(i) */
          double gxp = Mxp * interp_x(c, q->u, i + 1, j, k, oh, Mxp); /* between u(i), u(i+1) */
          double gym = Mym * interp_y(c, q->u, i, j, k, oh, Mym);
          double gyp = Myp * interp_y(c, q->u, i, j + 1, k, oh, Myp);
          double gzm = (k >= 1) ? Mzm * interp_z(c, q->u, i, j, k, 0, nz - 1, ov, Mzm) : 0.0;
          double gzp =
              (k + 1 <= nz - 1) ? Mzp * interp_z(c, q->u, i, j, k + 1, 0, nz - 1, ov, Mzp) : 0.0;
          R[UU][a] = -((gxp - gxm) / dx + (gyp - gym) / dy + (gzp - gzm)) / c->hu[a];
        }
        /* ---- V momentum ---- */
        {
          double Mxm = 0.5 * (Fx[IX(c, i, j - 1, k)] + Fx[IX(c, i, j, k)]);     /* edge i-1/2 */
          double Mxp = 0.5 * (Fx[IX(c, i + 1, j - 1, k)] + Fx[IX(c, i + 1, j, k)]);
          double Mym = 0.5 * (Fy[IX(c, i, j - 1, k)] + Fy[IX(c, i, j, k)]);     /* centre j-1 */
          double Myp = 0.5 * (Fy[IX(c, i, j, k)] + Fy[IX(c, i, j + 1, k)]);     /* centre j   */
          double Mzm = 0.5 * (Om[IX(c, i, j - 1, k)] + Om[IX(c, i, j, k)]);
          double Mzp = 0.5 * (Om[IX(c, i, j - 1, k + 1)] + Om[IX(c, i, j, k + 1)]);
          double gxm = Mxm * interp_x(c, q->v, i, j, k, oh, Mxm);
          double gxp = Mxp * interp_x(c, q->v, i + 1, j, k, oh, Mxp);
          double gym = Mym * interp_y(c, q->v, i, j, k, oh, Mym);
          double gyp = Myp * interp_y(c, q->v, i, j + 1, k, oh, Myp);
          double gzm = (k >= 1) ? Mzm * interp_z(c, q->v, i, j, k, 0, nz - 1, ov, Mzm) : 0.0;
          double gzp =
              (k + 1 <= nz - 1) ? Mzp * interp_z(c, q->v, i, j, k + 1, 0, nz - 1, ov, Mzp) : 0.0;
          R[VV][a] = -((gxp - gxm) / dx + (gyp - gym) / dy + (gzp - gzm)) / c->hv[a];
        }
      }
  /* ---- W momentum on interior faces k = 1..nz-1; R_W = 0 on the lids ---- */
#pragma omp parallel for schedule(static)
  for (int k = 0; k <= nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        if (k == 0 || k == nz) {
          R[WW][a] = 0.0;
          continue;
        }
        double Mxm = 0.5 * (Fx[IX(c, i, j, k - 1)] + Fx[IX(c, i, j, k)]);         /* edge i-1/2 */
        double Mxp = 0.5 * (Fx[IX(c, i + 1, j, k - 1)] + Fx[IX(c, i + 1, j, k)]);
        double Mym = 0.5 * (Fy[IX(c, i, j, k - 1)] + Fy[IX(c, i, j, k)]);
        double Myp = 0.5 * (Fy[IX(c, i, j + 1, k - 1)] + Fy[IX(c, i, j + 1, k)]);
        double Mzm = 0.5 * (Om[IX(c, i, j, k - 1)] + Om[IX(c, i, j, k)]);         /* centre k-1 */
        double Mzp = 0.5 * (Om[IX(c, i, j, k)] + Om[IX(c, i, j, k + 1)]);         /* centre k   */
        double gxm = Mxm * interp_x(c, q->w, i, j, k, oh, Mxm);
        double gxp = Mxp * interp_x(c, q->w, i + 1, j, k, oh, Mxp);
        double gym = Mym * interp_y(c, q->w, i, j, k, oh, Mym);
        double gyp = Myp * interp_y(c, q->w, i, j + 1, k, oh, Myp);
        /* between w-faces k-1 and k (flux point = centre k-1), valid faces 0..nz */
        double gzm = Mzm * interp_z(c, q->w, i, j, k, 0, nz, ov, Mzm);
        double gzp = Mzp * interp_z(c, q->w, i, j, k + 1, 0, nz, ov, Mzp);
        R[WW][a] = -((gxp - gxm) / dx + (gyp - gym) / dy + (gzp - gzm)) / c->hw[a];
      }
  free(Fx);
  free(Fy);
  free(Om);
}

/* ------------------------------------------------------------------ */
/* S3: diffusion  (Eq. 2 "-div tau", Eq. 3 "div(rho alpha grad theta)", */
/*                 Eq. 9)                                    */
/* ------------------------------------------------------------------ */

/* mean of the (up to) four two-point vertical difference quotients
 * qv(.,k'), k' in {k, k+1}, at two horizontal positions a0,a1 (given as
 * flat offsets at level 0), for a quantity whose quotients exist on
 * k' = 1..nz-1 only: two values at the lids [R:G14]. */
static double avg_q_valid(const erfo_ctx *c, const double *qv, size_t a0, size_t a1, int k) {
  double s = 0.0;
  int n = 0;
  for (int kk = k; kk <= k + 1; kk++)
    if (kk >= 1 && kk <= c->nz - 1) {
      s += qv[a0 + (size_t)kk * c->sk] + qv[a1 + (size_t)kk * c->sk];
      n += 2;
    }
  return n ? s / n : 0.0;
}

typedef struct {
  double *mu, *K;                         /* cell centres */
  double *S11, *S22, *S33, *S12, *S13, *S23;
  double *qu, *qv;                        /* du/dz, dv/dz two-point quotients at edges */
} diff_t;

/* strain-rate tensor on the C-grid and the viscosity.  S = 1/2(grad u +
 * grad u^T) (L104).  Placement [R:G11]: S11,S22,S33 at centres, S12 at
 * xy-edges (i-1/2,j-1/2,k), S13 at xz-edges (i-1/2,j,k-1/2), S23 at yz-edges.
 * Terrain [R:G14]: d/dx|_z = delta_x - slope * mean(vertical quotients).
 * Free-slip lids (Table C1 "Slip Wall"): du/dz = dv/dz = 0 and S13=S23=0
 * at k=0 and k=nz. */
static void strain_and_viscosity(const erfo_ctx *c, double *const S[5], const prim_t *q,
                                 diff_t *d) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  double dx = c->dx, dy = c->dy;
  /* vertical quotients of u and v at (i-1/2,j,k-1/2), (i,j-1/2,k-1/2); 0 on lids */
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k), b = IX(c, i, j, k - 1);
        double hwx = 0.5 * (c->hw[IX(c, i - 1, j, k)] + c->hw[a]);
        double hwy = 0.5 * (c->hw[IX(c, i, j - 1, k)] + c->hw[a]);
        d->qu[a] = (q->u[a] - q->u[b]) / hwx;
        d->qv[a] = (q->v[a] - q->v[b]) / hwy;
      }
  fill_lateral(c, d->qu);
  fill_lateral(c, d->qv);
  /* S33 first: it is also the vertical quotient of w at centres */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        d->S33[a] = (q->w[IX(c, i, j, k + 1)] - q->w[a]) / c->hc[a];
      }
  fill_lateral(c, d->S33);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t up = c->sk;
        /* heights of the u- and v-points: mean of the adjacent cell centres */
#define ZCU(ii, jj) (0.5 * (c->zc[IX(c, (ii)-1, jj, k)] + c->zc[IX(c, ii, jj, k)]))
#define ZCV(ii, jj) (0.5 * (c->zc[IX(c, ii, (jj)-1, k)] + c->zc[IX(c, ii, jj, k)]))
        {
          double s = (ZCU(i + 1, j) - ZCU(i, j)) / dx;
          size_t e0 = IX(c, i, j, k), e1 = IX(c, i + 1, j, k);
          double m = 0.25 * (d->qu[e0] + d->qu[e1] + d->qu[e0 + up] + d->qu[e1 + up]);
          d->S11[a] = (q->u[e1] - q->u[e0]) / dx - s * m;
        }
        {
          double s = (ZCV(i, j + 1) - ZCV(i, j)) / dy;
          size_t e0 = IX(c, i, j, k), e1 = IX(c, i, j + 1, k);
          double m = 0.25 * (d->qv[e0] + d->qv[e1] + d->qv[e0 + up] + d->qv[e1 + up]);
          d->S22[a] = (q->v[e1] - q->v[e0]) / dy - s * m;
        }
        { /* S12 at (i-1/2, j-1/2, k) */
          double sa = (ZCU(i, j) - ZCU(i, j - 1)) / dy;
          size_t e0 = IX(c, i, j - 1, k), e1 = IX(c, i, j, k);
          double ma = 0.25 * (d->qu[e0] + d->qu[e1] + d->qu[e0 + up] + d->qu[e1 + up]);
          double dudy = (q->u[e1] - q->u[e0]) / dy - sa * ma;
          double sb = (ZCV(i, j) - ZCV(i - 1, j)) / dx;
          size_t f0 = IX(c, i - 1, j, k), f1 = IX(c, i, j, k);
          double mb = 0.25 * (d->qv[f0] + d->qv[f1] + d->qv[f0 + up] + d->qv[f1 + up]);
          double dvdx = (q->v[f1] - q->v[f0]) / dx - sb * mb;
          d->S12[a] = 0.5 * (dudy + dvdx);
        }
#undef ZCU
#undef ZCV
      }
  /* S13 at (i-1/2, j, k-1/2), S23 at (i, j-1/2, k-1/2); zero on the lids */
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        {
          double s = (c->zw[a] - c->zw[IX(c, i - 1, j, k)]) / dx;
          double m = 0.25 * (d->S33[IX(c, i - 1, j, k - 1)] + d->S33[IX(c, i, j, k - 1)] +
                             d->S33[IX(c, i - 1, j, k)] + d->S33[IX(c, i, j, k)]);
          double dwdx = (q->w[a] - q->w[IX(c, i - 1, j, k)]) / dx - s * m;
          d->S13[a] = 0.5 * (d->qu[a] + dwdx);
        }
        {
          double s = (c->zw[a] - c->zw[IX(c, i, j - 1, k)]) / dy;
          double m = 0.25 * (d->S33[IX(c, i, j - 1, k - 1)] + d->S33[IX(c, i, j, k - 1)] +
                             d->S33[IX(c, i, j - 1, k)] + d->S33[IX(c, i, j, k)]);
          double dwdy = (q->w[a] - q->w[IX(c, i, j - 1, k)]) / dy - s * m;
          d->S23[a] = 0.5 * (d->qv[a] + dwdy);
        }
      }
  fill_lateral(c, d->S11);
  fill_lateral(c, d->S22);
  fill_lateral(c, d->S12);
  fill_lateral(c, d->S13);
  fill_lateral(c, d->S23);
  /* viscosity mu = mu_m + mu_t (L100) and scalar diffusivity K = rho*alpha */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t up = c->sk;
        double rho = S[RHO][a];
        double mu = rho * c->p.nu;           /* mu_m = rho*nu [R:G10] */
        double K = rho * c->p.alpha_theta;
        if (c->p.diffusion == 2) {
          /* Smagorinsky-Lilly (cited only, L104) [R:G9]:
           * mu_t = rho (Cs Delta)^2 |S|, |S| = sqrt(2 Sij Sij), edge strains
           * brought to the centre by 4-point means, Delta = (dx dy hc)^(1/3) */
          size_t a10 = IX(c, i + 1, j, k), a01 = IX(c, i, j + 1, k), a11 = IX(c, i + 1, j + 1, k);
          double s12 = 0.25 * (d->S12[a] + d->S12[a10] + d->S12[a01] + d->S12[a11]);
          double s13 = 0.25 * (d->S13[a] + d->S13[a10] + d->S13[a + up] + d->S13[a10 + up]);
          double s23 = 0.25 * (d->S23[a] + d->S23[a01] + d->S23[a + up] + d->S23[a01 + up]);
          double ss = 2.0 * (d->S11[a] * d->S11[a] + d->S22[a] * d->S22[a] + d->S33[a] * d->S33[a]) +
                      4.0 * (s12 * s12 + s13 * s13 + s23 * s23);
          double delta = cbrt(c->dx * c->dy * c->hc[a]);
          double mut = rho * (c->p.Cs * delta) * (c->p.Cs * delta) * sqrt(ss);
          mu += mut;
          K += mut / c->p.Pr_t;
        }
        d->mu[a] = mu;
        d->K[a] = K;
      }
  fill_lateral(c, d->mu);
  fill_lateral(c, d->K);
}

static void diffusion(const erfo_ctx *c, double *const S[5], const prim_t *q, double *R[5]) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  double dx = c->dx, dy = c->dy;
  diff_t d;
  d.mu = fnew(c); d.K = fnew(c);
  d.S11 = fnew(c); d.S22 = fnew(c); d.S33 = fnew(c);
  d.S12 = fnew(c); d.S13 = fnew(c); d.S23 = fnew(c);
  d.qu = fnew(c); d.qv = fnew(c);
  strain_and_viscosity(c, S, q, &d);

  /* Eq. 9 (L102): tau = -2 mu sigma, sigma = S - 1/3 (div u) I. Edge
   * viscosity = 4-point mean of the centre values [R:G11]. */
  double *t11 = fnew(c), *t22 = fnew(c), *t33 = fnew(c);
  double *t12 = fnew(c), *t13 = fnew(c), *t23 = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        double div3 = (d.S11[a] + d.S22[a] + d.S33[a]) / 3.0;
        t11[a] = -2.0 * d.mu[a] * (d.S11[a] - div3);
        t22[a] = -2.0 * d.mu[a] * (d.S22[a] - div3);
        t33[a] = -2.0 * d.mu[a] * (d.S33[a] - div3);
        double mu12 = 0.25 * (d.mu[IX(c, i - 1, j - 1, k)] + d.mu[IX(c, i, j - 1, k)] +
                              d.mu[IX(c, i - 1, j, k)] + d.mu[a]);
        t12[a] = -2.0 * mu12 * d.S12[a];
        if (k >= 1) {
          double mu13 = 0.25 * (d.mu[IX(c, i - 1, j, k - 1)] + d.mu[IX(c, i, j, k - 1)] +
                                d.mu[IX(c, i - 1, j, k)] + d.mu[a]);
          double mu23 = 0.25 * (d.mu[IX(c, i, j - 1, k - 1)] + d.mu[IX(c, i, j, k - 1)] +
                                d.mu[IX(c, i, j - 1, k)] + d.mu[a]);
          t13[a] = -2.0 * mu13 * d.S13[a];
          t23[a] = -2.0 * mu23 * d.S23[a];
        } /* k = 0 and k = nz stay 0: free slip */
      }
  fill_lateral(c, t11); fill_lateral(c, t22); fill_lateral(c, t33);
  fill_lateral(c, t12); fill_lateral(c, t13); fill_lateral(c, t23);

  /* vertical two-point quotients of the stresses (for the chain rule) and of theta */
  double *q11 = fnew(c), *q22 = fnew(c), *q12 = fnew(c), *q13 = fnew(c), *q23 = fnew(c);
  double *qth = fnew(c);
  double *ze12 = fnew(c); /* height of the xy-edge: mean of the 4 cell centres */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++)
        ze12[IX(c, i, j, k)] = 0.25 * (c->zc[IX(c, i - 1, j - 1, k)] + c->zc[IX(c, i, j - 1, k)] +
                                       c->zc[IX(c, i - 1, j, k)] + c->zc[IX(c, i, j, k)]);
  fill_lateral(c, ze12);
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k), b = IX(c, i, j, k - 1);
        q11[a] = (t11[a] - t11[b]) / c->hw[a];
        q22[a] = (t22[a] - t22[b]) / c->hw[a];
        qth[a] = (q->theta[a] - q->theta[b]) / c->hw[a];
        q12[a] = (t12[a] - t12[b]) / (ze12[a] - ze12[b]);
      }
  /* tau13, tau23 live on k-1/2 edges; their quotients live at level centres 0..nz-1 */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k), t = IX(c, i, j, k + 1);
        double ze13a = 0.5 * (c->zw[IX(c, i - 1, j, k)] + c->zw[a]);
        double ze13t = 0.5 * (c->zw[IX(c, i - 1, j, k + 1)] + c->zw[t]);
        double ze23a = 0.5 * (c->zw[IX(c, i, j - 1, k)] + c->zw[a]);
        double ze23t = 0.5 * (c->zw[IX(c, i, j - 1, k + 1)] + c->zw[t]);
        q13[a] = (t13[t] - t13[a]) / (ze13t - ze13a);
        q23[a] = (t23[t] - t23[a]) / (ze23t - ze23a);
      }
  fill_lateral(c, q11); fill_lateral(c, q22); fill_lateral(c, q12);
  fill_lateral(c, q13); fill_lateral(c, q23); fill_lateral(c, qth);

  /* ---- momentum: R -= div tau (non-conservative chain-rule form over terrain) ---- */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t z0 = IX(c, i, j, 0), zim = IX(c, i - 1, j, 0), zjm = IX(c, i, j - 1, 0);
        size_t zip = IX(c, i + 1, j, 0), zjp = IX(c, i, j + 1, 0);
        { /* U at (i-1/2, j, k) */
          double d11 = (t11[a] - t11[IX(c, i - 1, j, k)]) / dx -
                       c->sxu[a] * avg_q_valid(c, q11, zim, z0, k);
          double s12 = (ze12[IX(c, i, j + 1, k)] - ze12[a]) / dy;
          double d12 = (t12[IX(c, i, j + 1, k)] - t12[a]) / dy -
                       s12 * avg_q_valid(c, q12, z0, zjp, k);
          double d13 = (t13[IX(c, i, j, k + 1)] - t13[a]) / c->hu[a];
          R[UU][a] -= d11 + d12 + d13;
        }
        { /* V at (i, j-1/2, k) */
          double s12 = (ze12[IX(c, i + 1, j, k)] - ze12[a]) / dx;
          double d12 = (t12[IX(c, i + 1, j, k)] - t12[a]) / dx -
                       s12 * avg_q_valid(c, q12, z0, zip, k);
          double d22 = (t22[a] - t22[IX(c, i, j - 1, k)]) / dy -
                       c->syv[a] * avg_q_valid(c, q22, zjm, z0, k);
          double d23 = (t23[IX(c, i, j, k + 1)] - t23[a]) / c->hv[a];
          R[VV][a] -= d12 + d22 + d23;
        }
        if (k >= 1) { /* W at (i, j, k-1/2) */
          double ze_i = 0.5 * (c->zw[IX(c, i - 1, j, k)] + c->zw[a]);
          double ze_ip = 0.5 * (c->zw[a] + c->zw[IX(c, i + 1, j, k)]);
          double ze_j = 0.5 * (c->zw[IX(c, i, j - 1, k)] + c->zw[a]);
          double ze_jp = 0.5 * (c->zw[a] + c->zw[IX(c, i, j + 1, k)]);
          double m13 = 0.25 * (q13[IX(c, i, j, k - 1)] + q13[IX(c, i + 1, j, k - 1)] +
                               q13[a] + q13[IX(c, i + 1, j, k)]);
          double m23 = 0.25 * (q23[IX(c, i, j, k - 1)] + q23[IX(c, i, j + 1, k - 1)] +
                               q23[a] + q23[IX(c, i, j + 1, k)]);
          double d13 = (t13[IX(c, i + 1, j, k)] - t13[a]) / dx - (ze_ip - ze_i) / dx * m13;
          double d23 = (t23[IX(c, i, j + 1, k)] - t23[a]) / dy - (ze_jp - ze_j) / dy * m23;
          double d33 = (t33[a] - t33[IX(c, i, j, k - 1)]) / c->hw[a];
          R[WW][a] -= d13 + d23 + d33;
        }
      }

  /* ---- scalar: conservative form (needed for conservation of rho*theta) ----
   * Fx = -Kx Dx(theta) at x-faces, Fy likewise, Fz = -Kw dtheta/dz at w-faces,
   * contravariant Fzeta = Fz - sxw avg4(Fx) - syw avg4(Fy), zero on the lids.
   * Diffusion acts on the full theta (Eq. 3) [R:G17]. */
  double *Fx = fnew(c), *Fy = fnew(c), *Fz = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t z0 = IX(c, i, j, 0), zim = IX(c, i - 1, j, 0), zjm = IX(c, i, j - 1, 0);
        double Kx = 0.5 * (d.K[IX(c, i - 1, j, k)] + d.K[a]);
        double Ky = 0.5 * (d.K[IX(c, i, j - 1, k)] + d.K[a]);
        double dthx = (q->theta[a] - q->theta[IX(c, i - 1, j, k)]) / dx -
                      c->sxu[a] * avg_q_valid(c, qth, zim, z0, k);
        double dthy = (q->theta[a] - q->theta[IX(c, i, j - 1, k)]) / dy -
                      c->syv[a] * avg_q_valid(c, qth, zjm, z0, k);
        Fx[a] = -Kx * dthx;
        Fy[a] = -Ky * dthy;
      }
  fill_lateral(c, Fx);
  fill_lateral(c, Fy);
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        double Kw = 0.5 * (d.K[IX(c, i, j, k - 1)] + d.K[a]);
        double fz = -Kw * qth[a];
        double fxb = 0.25 * (Fx[IX(c, i, j, k - 1)] + Fx[IX(c, i + 1, j, k - 1)] + Fx[a] +
                             Fx[IX(c, i + 1, j, k)]);
        double fyb = 0.25 * (Fy[IX(c, i, j, k - 1)] + Fy[IX(c, i, j + 1, k - 1)] + Fy[a] +
                             Fy[IX(c, i, j + 1, k)]);
        Fz[a] = fz - c->sxw[a] * fxb - c->syw[a] * fyb;
      } /* Fz = 0 on k = 0 and k = nz */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t ip = IX(c, i + 1, j, k), jp = IX(c, i, j + 1, k), kp = IX(c, i, j, k + 1);
        R[TH][a] -= ((c->hx[ip] * Fx[ip] - c->hx[a] * Fx[a]) / dx +
                     (c->hy[jp] * Fy[jp] - c->hy[a] * Fy[a]) / dy + (Fz[kp] - Fz[a])) /
                    c->hc[a];
      }
  free(Fx); free(Fy); free(Fz);
  free(q11); free(q22); free(q12); free(q13); free(q23); free(qth); free(ze12);
  free(t11); free(t22); free(t33); free(t12); free(t13); free(t23);
  free(d.mu); free(d.K); free(d.S11); free(d.S22); free(d.S33);
  free(d.S12); free(d.S13); free(d.S23); free(d.qu); free(d.qv);
}

/* ------------------------------------------------------------------ */
/* S4: pressure gradient and buoyancy (Eq. 2; B = -(rho-rho0) g, L84) */
/* ------------------------------------------------------------------ */

/* vertical derivative at a cell centre: centred over the two neighbouring
 * centres, one-sided two-point at k=0 and k=nz-1 [R:G14] */
static double dz_centre(const erfo_ctx *c, const double *f, int i, int j, int k) {
  int kb = k > 0 ? k - 1 : 0;
  int kt = k < c->nz - 1 ? k + 1 : c->nz - 1;
  return (f[IX(c, i, j, kt)] - f[IX(c, i, j, kb)]) / (c->zc[IX(c, i, j, kt)] - c->zc[IX(c, i, j, kb)]);
}

/* horizontal gradient at constant height of a cell-centred field, at the
 * u-point: difference along the coordinate surface minus slope times the
 * mean vertical derivative of the two cells [R:G14] */
static double grad_x(const erfo_ctx *c, const double *f, int i, int j, int k) {
  double along = (f[IX(c, i, j, k)] - f[IX(c, i - 1, j, k)]) / c->dx;
  if (c->nz == 1) return along;
  return along - c->sxu[IX(c, i, j, k)] * 0.5 * (dz_centre(c, f, i - 1, j, k) + dz_centre(c, f, i, j, k));
}
static double grad_y(const erfo_ctx *c, const double *f, int i, int j, int k) {
  double along = (f[IX(c, i, j, k)] - f[IX(c, i, j - 1, k)]) / c->dy;
  if (c->nz == 1) return along;
  return along - c->syv[IX(c, i, j, k)] * 0.5 * (dz_centre(c, f, i, j - 1, k) + dz_centre(c, f, i, j, k));
}

static void pressure_buoyancy(const erfo_ctx *c, double *const S[5], const prim_t *q,
                              double *R[5]) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        R[UU][a] -= grad_x(c, q->pp, i, j, k);
        R[VV][a] -= grad_y(c, q->pp, i, j, k);
        if (k >= 1) {
          size_t b = IX(c, i, j, k - 1);
          double rpa = S[RHO][a] - c->rho0[a], rpb = S[RHO][b] - c->rho0[b];
          R[WW][a] -= (q->pp[a] - q->pp[b]) / c->hw[a] + c->p.g * 0.5 * (rpb + rpa);
        }
      }
}

/* Rayleigh damping layer ("Rayleigh damping and sponge layer(s)"; Appendix C: "The damping strength,
 * an inverse timescale, was ramped using a sine-squared function from 0 at the bottom of the damping layer to the
 * specified value at the top"; Table C1: depth, strength and the damped fields among u, v, w, theta).
 *   tau(z) = ray_coef * sin^2( (pi/2) (z - z_b) / ray_depth ),  z_b = z_top - ray_depth,  0 below z_b
 * The paper prints no equation for the tendency; the reading [R:G28] is relaxation of the primitive variable towards a
 * reference: R_W -= tau W (reference 0), R_U -= tau rho_u (u - u_ref), R_V likewise, R_Theta -= tau rho (theta -
 * theta0) with theta0 the base state, each tau at the height of its own point.  ray_fields: 1 u, 2 v, 4 w, 8 theta. */
static double rayleigh_tau(const erfo_ctx *c, double z, double ztop) {
  double zb = ztop - c->p.ray_depth;
  if (!(c->p.ray_depth > 0.0) || z <= zb) return 0.0;
  double s = sin(0.5 * 3.14159265358979323846 * (z - zb) / c->p.ray_depth);
  return c->p.ray_coef * s * s;
}

static void rayleigh(const erfo_ctx *c, double *const S[5], double *R[5]) {
  int nx = c->nx, ny = c->ny, nz = c->nz, f = c->p.ray_fields;
  if (!f || !(c->p.ray_depth > 0.0)) return;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k), im = IX(c, i - 1, j, k), jm = IX(c, i, j - 1, k);
        size_t t = IX(c, i, j, nz), tim = IX(c, i - 1, j, nz), tjm = IX(c, i, j - 1, nz);
        if (f & 1) {
          double tau = rayleigh_tau(c, 0.5 * (c->zc[im] + c->zc[a]), 0.5 * (c->zw[tim] + c->zw[t]));
          R[UU][a] -= tau * (S[UU][a] - 0.5 * (S[RHO][im] + S[RHO][a]) * c->p.ray_uref);
        }
        if (f & 2) {
          double tau = rayleigh_tau(c, 0.5 * (c->zc[jm] + c->zc[a]), 0.5 * (c->zw[tjm] + c->zw[t]));
          R[VV][a] -= tau * (S[VV][a] - 0.5 * (S[RHO][jm] + S[RHO][a]) * c->p.ray_vref);
        }
        if ((f & 4) && k >= 1) R[WW][a] -= rayleigh_tau(c, c->zw[a], c->zw[t]) * S[WW][a];
        if (f & 8) R[TH][a] -= rayleigh_tau(c, c->zc[a], c->zw[t]) * (S[TH][a] - S[RHO][a] * c->Th0[a] / c->rho0[a]);
      }
}

/* f(S): the slow right-hand side of Eq. 1-3.  Also hands back theta^t, pi^t. */
static void anelastic_pressure_buoyancy(const erfo_ctx *c, const prim_t *q, const double *pan, double *R[5]);

static void slow_rhs_mode(const erfo_ctx *c, double *const S[5], double *R[5], double *theta_t,
                          double *pi_t, const double *pan) {
  prim_t q;
  q.theta = fnew(c); q.pp = fnew(c); q.pi = fnew(c);
  q.u = fnew(c); q.v = fnew(c); q.w = fnew(c);
  primitives(c, S, &q);
  advection(c, S, &q, R);
  if (c->p.diffusion != 0) diffusion(c, S, &q, R);
  if (pan) anelastic_pressure_buoyancy(c, &q, pan, R); /* Sec. 2.2: p' from the projection, B from theta */
  else pressure_buoyancy(c, S, &q, R);
  rayleigh(c, S, R);
  for (int m = 0; m < 5; m++) fill_lateral(c, R[m]);
  if (theta_t) memcpy(theta_t, q.theta, c->n * sizeof(double));
  if (pi_t) memcpy(pi_t, q.pi, c->n * sizeof(double));
  free(q.theta); free(q.pp); free(q.pi); free(q.u); free(q.v); free(q.w);
}

static void slow_rhs(const erfo_ctx *c, double *const S[5], double *R[5], double *theta_t,
                     double *pi_t) {
  slow_rhs_mode(c, S, R, theta_t, pi_t, NULL);
}

/* ------------------------------------------------------------------ */
/* S5: acoustic substeps (Appendix A; Sec. 3.1)   */
/* ------------------------------------------------------------------ */

typedef struct {
  const double *theta_t, *pi_t, *Th_t; /* stage constants */
  double *const *R;                    /* slow tendencies  */
  double *P[5];                        /* S'' = (rho'', U'', V'', W'', Theta'') */
  double *Om;                          /* Omega'' at the end of the previous substep */
  double *Th_prev;                     /* Theta'' one substep back (divergence damping) */
  /* sums over the substeps of the perturbation momenta that advance rho'' (L138: "the time average over the
   * RK stage of the intermediate (rho u . n) values used to advance rho each substep"); NULL = not wanted */
  double *Usum, *Vsum, *Omsum;
} acoustic_t;

/* coefficients of row k (1..nz-1) of the column system for Omega''^{new}.
 * Derivation: eliminate Theta''^{new}, rho''^{new} from the W'' equation of
 * Appendix A (L585) using the time-centred averages of L591; in that line
 * the overbarred rho and pi are BASE-STATE values, the tau-overbars are
 * time averages [R:G4].  s = (dtau*beta2)^2. */
static void tridiag_row(const erfo_ctx *c, const acoustic_t *ac, double dtau, int i, int j,
                        int k, double *A, double *D, double *C) {
  int nz = c->nz;
  double b2 = 0.5 * (1.0 + c->p.beta_s);
  double s = dtau * dtau * b2 * b2;
  double g = c->p.g, gR = c->gam * c->p.Rd;
  size_t a = IX(c, i, j, k), b = IX(c, i, j, k - 1);
  double pif = 0.5 * (ac->pi_t[b] + ac->pi_t[a]);
  double pi0f = 0.5 * (c->pi0[b] + c->pi0[a]);
  double rho0f = 0.5 * (c->rho0[b] + c->rho0[a]);
  double Bf = rho0f * c->rdocv * pif / pi0f;
  double thf_k = 0.5 * (ac->theta_t[b] + ac->theta_t[a]);
  double thf_kp = (k + 1 <= nz - 1) ? 0.5 * (ac->theta_t[a] + ac->theta_t[IX(c, i, j, k + 1)]) : 0.0;
  double thf_km = (k - 1 >= 1) ? 0.5 * (ac->theta_t[IX(c, i, j, k - 2)] + ac->theta_t[b]) : 0.0;
  double hw = c->hw[a], hck = c->hc[a], hcm = c->hc[b];
  double Tk = ac->Th_t[a], Tm = ac->Th_t[b];
  *C = -s * gR * pif * thf_kp / (hw * hck) + s * g * Bf * thf_kp / (2.0 * hck * Tk) -
       s * g / (2.0 * hck);
  *A = -s * gR * pif * thf_km / (hw * hcm) - s * g * Bf * thf_km / (2.0 * hcm * Tm) +
       s * g / (2.0 * hcm);
  *D = 1.0 + s * gR * pif * thf_k * (1.0 / hck + 1.0 / hcm) / hw -
       s * g * Bf * thf_k / 2.0 * (1.0 / (hck * Tk) - 1.0 / (hcm * Tm)) +
       s * g / 2.0 * (1.0 / hck - 1.0 / hcm);
  if (k == nz - 1) *C = 0.0; /* Omega_nz = 0 */
  if (k == 1) *A = 0.0;      /* Omega_0  = 0 */
}

static void acoustic_substep(const erfo_ctx *c, acoustic_t *ac, double dtau) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  double dx = c->dx, dy = c->dy;
  double b1 = 0.5 * (1.0 - c->p.beta_s), b2 = 0.5 * (1.0 + c->p.beta_s); /* L589 */
  double g = c->p.g, gR = c->gam * c->p.Rd;
  double *Upp = ac->P[UU], *Vpp = ac->P[VV], *Wpp = ac->P[WW], *rpp = ac->P[RHO], *Tpp = ac->P[TH];

  /* 1. divergence damping (L144): Theta'' "predicted slightly forward in time" [R:G6] */
  double *Thd = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        Thd[a] = Tpp[a] + c->p.beta_d * (Tpp[a] - ac->Th_prev[a]);
        ac->Th_prev[a] = Tpp[a];
      }
  fill_lateral(c, Thd);

  /* 2. horizontal momenta, explicit (L585 rows 1-2); pi^t averaged to the face */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        double piu = 0.5 * (ac->pi_t[IX(c, i - 1, j, k)] + ac->pi_t[a]);
        double piv = 0.5 * (ac->pi_t[IX(c, i, j - 1, k)] + ac->pi_t[a]);
        Upp[a] += dtau * (-gR * piu * grad_x(c, Thd, i, j, k) + ac->R[UU][a]);
        Vpp[a] += dtau * (-gR * piv * grad_y(c, Thd, i, j, k) + ac->R[VV][a]);
      }
  fill_lateral(c, Upp);
  fill_lateral(c, Vpp);
  if (ac->Usum) /* the horizontal momenta that enter this substep's continuity equation (step 4) */
    for (size_t a = 0; a < c->n; a++) {
      ac->Usum[a] += Upp[a];
      ac->Vsum[a] += Vpp[a];
    }

  /* 3. explicit slope part of W'': omega = sxw avg4(U''new) + syw avg4(V''new) [R:G16] */
  double *om = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 1; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k), b = IX(c, i, j, k - 1);
        double ubar = 0.25 * (Upp[b] + Upp[IX(c, i + 1, j, k - 1)] + Upp[a] + Upp[IX(c, i + 1, j, k)]);
        double vbar = 0.25 * (Vpp[b] + Vpp[IX(c, i, j + 1, k - 1)] + Vpp[a] + Vpp[IX(c, i, j + 1, k)]);
        om[a] = c->sxw[a] * ubar + c->syw[a] * vbar;
      }

  /* 4.-6. per column (columns are independent: each thread of the optional OpenMP build owns its scratch) */
#pragma omp parallel
  {
  double *Ttil = (double *)calloc(nz, sizeof(double)), *rtil = (double *)calloc(nz, sizeof(double));
  double *That = (double *)calloc(nz, sizeof(double)), *rhat = (double *)calloc(nz, sizeof(double));
  double *thf = (double *)calloc(nz + 1, sizeof(double));
  double *A = (double *)calloc(nz + 1, sizeof(double)), *D = (double *)calloc(nz + 1, sizeof(double));
  double *C = (double *)calloc(nz + 1, sizeof(double)), *rhs = (double *)calloc(nz + 1, sizeof(double));
  double *On = (double *)calloc(nz + 1, sizeof(double));
  double *cp_ = (double *)calloc(nz + 1, sizeof(double)), *dp_ = (double *)calloc(nz + 1, sizeof(double));
#pragma omp for schedule(static)
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      /* theta^t at the w-faces; the lid values are never used (Omega = 0 there) */
      thf[0] = thf[nz] = 0.0;
      for (int k = 1; k < nz; k++)
        thf[k] = 0.5 * (ac->theta_t[IX(c, i, j, k - 1)] + ac->theta_t[IX(c, i, j, k)]);
      /* 4. explicit parts (L585 rows 4-5 with the old-time part of the W'' average) */
      for (int k = 0; k < nz; k++) {
        size_t a = IX(c, i, j, k), ip = IX(c, i + 1, j, k), jp = IX(c, i, j + 1, k);
        double thx_m = 0.5 * (ac->theta_t[IX(c, i - 1, j, k)] + ac->theta_t[a]);
        double thx_p = 0.5 * (ac->theta_t[a] + ac->theta_t[ip]);
        double thy_m = 0.5 * (ac->theta_t[IX(c, i, j - 1, k)] + ac->theta_t[a]);
        double thy_p = 0.5 * (ac->theta_t[a] + ac->theta_t[jp]);
        double hc = c->hc[a];
        double DhT = (c->hx[ip] * Upp[ip] * thx_p - c->hx[a] * Upp[a] * thx_m) / dx / hc +
                     (c->hy[jp] * Vpp[jp] * thy_p - c->hy[a] * Vpp[a] * thy_m) / dy / hc;
        double Dh = (c->hx[ip] * Upp[ip] - c->hx[a] * Upp[a]) / dx / hc +
                    (c->hy[jp] * Vpp[jp] - c->hy[a] * Vpp[a]) / dy / hc;
        double om_b = ac->Om[a], om_t = ac->Om[IX(c, i, j, k + 1)]; /* zero on the lids */
        Ttil[k] = Tpp[a] + dtau * (ac->R[TH][a] - DhT - b1 * (thf[k + 1] * om_t - thf[k] * om_b) / hc);
        rtil[k] = rpp[a] + dtau * (ac->R[RHO][a] - Dh - b1 * (om_t - om_b) / hc);
        That[k] = b2 * Ttil[k] + b1 * Tpp[a];
        rhat[k] = b2 * rtil[k] + b1 * rpp[a];
      }
      /* 5. tridiagonal system for Omega''new, k = 1..nz-1 (L144) */
      for (int k = 1; k < nz; k++) {
        size_t a = IX(c, i, j, k), b = IX(c, i, j, k - 1);
        tridiag_row(c, ac, dtau, i, j, k, &A[k], &D[k], &C[k]);
        double pif = 0.5 * (ac->pi_t[b] + ac->pi_t[a]);
        double pi0f = 0.5 * (c->pi0[b] + c->pi0[a]);
        double rho0f = 0.5 * (c->rho0[b] + c->rho0[a]);
        double Bf = rho0f * c->rdocv * pif / pi0f;
        rhs[k] = Wpp[a] +
                 dtau * (ac->R[WW][a] - gR * pif * (That[k] - That[k - 1]) / c->hw[a] +
                         g * Bf * 0.5 * (That[k] / ac->Th_t[a] + That[k - 1] / ac->Th_t[b]) -
                         g * 0.5 * (rhat[k] + rhat[k - 1])) -
                 om[a];
      }
      /* Thomas algorithm */
      On[0] = On[nz] = 0.0;
      if (nz >= 2) {
        cp_[1] = C[1] / D[1];
        dp_[1] = rhs[1] / D[1];
        for (int k = 2; k < nz; k++) {
          double m = D[k] - A[k] * cp_[k - 1];
          cp_[k] = C[k] / m;
          dp_[k] = (rhs[k] - A[k] * dp_[k - 1]) / m;
        }
        On[nz - 1] = dp_[nz - 1];
        for (int k = nz - 2; k >= 1; k--) On[k] = dp_[k] - cp_[k] * On[k + 1];
      }
      /* 6. back-substitution (L585 rows 3-5) */
      for (int k = 1; k < nz; k++) Wpp[IX(c, i, j, k)] = On[k] + om[IX(c, i, j, k)];
      for (int k = 0; k < nz; k++) {
        size_t a = IX(c, i, j, k);
        double hc = c->hc[a];
        Tpp[a] = Ttil[k] - dtau * b2 * (thf[k + 1] * On[k + 1] - thf[k] * On[k]) / hc;
        rpp[a] = rtil[k] - dtau * b2 * (On[k + 1] - On[k]) / hc;
      }
      /* the vertical flux that advanced rho'' in this substep: beta2 Omega''new + beta1 Omega''old (L591) */
      if (ac->Omsum)
        for (int k = 0; k <= nz; k++) ac->Omsum[IX(c, i, j, k)] += b2 * On[k] + b1 * ac->Om[IX(c, i, j, k)];
      for (int k = 0; k <= nz; k++) ac->Om[IX(c, i, j, k)] = On[k];
    }
  free(Ttil); free(rtil); free(That); free(rhat); free(thf);
  free(A); free(D); free(C); free(rhs); free(On); free(cp_); free(dp_);
  }
  free(om);
  free(Thd);
  fill_lateral(c, Wpp);
  fill_lateral(c, Tpp);
  fill_lateral(c, rpp);
  fill_lateral(c, ac->Om);
}

/* run n substeps from S'' (ghosts filled) about stage state St */
static void acoustic_loop(const erfo_ctx *c, double *const St[5], const double *theta_t,
                          const double *pi_t, double *const R[5], double *P[5], double dtau,
                          int n, double *Mavg[3]) {
  acoustic_t ac;
  ac.Usum = Mavg ? Mavg[0] : NULL;
  ac.Vsum = Mavg ? Mavg[1] : NULL;
  ac.Omsum = Mavg ? Mavg[2] : NULL;
  if (Mavg)
    for (int m = 0; m < 3; m++) memset(Mavg[m], 0, c->n * sizeof(double));
  ac.theta_t = theta_t;
  ac.pi_t = pi_t;
  ac.Th_t = St[TH];
  ac.R = R;
  for (int m = 0; m < 5; m++) ac.P[m] = P[m];
  ac.Om = fnew(c);
  ac.Th_prev = fnew(c);
  contravariant_flux(c, P[UU], P[VV], P[WW], ac.Om); /* Omega'' of the initial S'' */
  memcpy(ac.Th_prev, P[TH], c->n * sizeof(double));  /* Theta''_prev = Theta'' */
  for (int s = 0; s < n; s++) acoustic_substep(c, &ac, dtau);
  if (Mavg) /* sums -> time averages over the stage */
    for (int m = 0; m < 3; m++) {
      for (size_t a = 0; a < c->n; a++) Mavg[m][a] /= (double)n;
      fill_lateral(c, Mavg[m]);
    }
  free(ac.Om);
  free(ac.Th_prev);
}

/* ------------------------------------------------------------------ */
/* Eq. 4: one transported scalar (L69), advanced after the substeps    */
/* (L138)                                                              */
/* ------------------------------------------------------------------ */

/* Q_stage = Q^n + dts * [ -div(Mbar phi^t) + div(K grad phi^t) ],  phi^t = Q^t / rho^t.
 * Mbar = (Ub, Vb, Omb): the stage-time-averaged normal momenta (stage momenta + averaged perturbations), so
 * that the scalar sees exactly the mass fluxes that advanced rho in the substeps (L138) -- a constant phi then
 * stays constant.  Interpolation of phi as for theta (Eq. 17-21 with the sign of Mbar; order reduction at the
 * lids [R:G13]).  Diffusion as for theta, conservative form, with the same diffusivity K = rho alpha (+ mu_t/Pr_t)
 * evaluated at the stage state [R:G25]. */
static void scalar_stage(const erfo_ctx *c, double *const St[5], const double *Qt, const double *Qn,
                         const double *Ub, const double *Vb, const double *Omb, double dts, double *Qout) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  int oh = c->p.scalar_adv ? c->p.scalar_adv : c->p.adv_order_h;
  int ov = c->p.scalar_adv ? c->p.scalar_adv : c->p.adv_order_v;
  double dx = c->dx, dy = c->dy;
  double *phi = fnew(c), *Fx = fnew(c), *Fy = fnew(c), *R = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        phi[a] = Qt[a] / St[RHO][a];
        Fx[a] = c->hx[a] * Ub[a];
        Fy[a] = c->hy[a] * Vb[a];
      }
  fill_lateral(c, phi);
  fill_lateral(c, Fx);
  fill_lateral(c, Fy);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        double fxm = Fx[a], fxp = Fx[IX(c, i + 1, j, k)];
        double fym = Fy[a], fyp = Fy[IX(c, i, j + 1, k)];
        double omm = Omb[a], omp = Omb[IX(c, i, j, k + 1)];
        double txm = fxm * interp_x(c, phi, i, j, k, oh, fxm);
        double txp = fxp * interp_x(c, phi, i + 1, j, k, oh, fxp);
        double tym = fym * interp_y(c, phi, i, j, k, oh, fym);
        double typ = fyp * interp_y(c, phi, i, j + 1, k, oh, fyp);
        double tzm = (k >= 1) ? omm * interp_z(c, phi, i, j, k, 0, nz - 1, ov, omm) : 0.0;
        double tzp = (k + 1 <= nz - 1) ? omp * interp_z(c, phi, i, j, k + 1, 0, nz - 1, ov, omp) : 0.0;
        R[a] = -((txp - txm) / dx + (typ - tym) / dy + (tzp - tzm)) / c->hc[a];
      }
  if (c->p.diffusion != 0) {
    prim_t q;
    q.theta = fnew(c); q.pp = fnew(c); q.pi = fnew(c);
    q.u = fnew(c); q.v = fnew(c); q.w = fnew(c);
    primitives(c, St, &q);
    diff_t d;
    d.mu = fnew(c); d.K = fnew(c);
    d.S11 = fnew(c); d.S22 = fnew(c); d.S33 = fnew(c);
    d.S12 = fnew(c); d.S13 = fnew(c); d.S23 = fnew(c);
    d.qu = fnew(c); d.qv = fnew(c);
    strain_and_viscosity(c, St, &q, &d);
    double *qph = fnew(c), *Gx = fnew(c), *Gy = fnew(c), *Gz = fnew(c);
    for (int k = 1; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          size_t a = IX(c, i, j, k);
          qph[a] = (phi[a] - phi[IX(c, i, j, k - 1)]) / c->hw[a];
        }
    fill_lateral(c, qph);
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          size_t a = IX(c, i, j, k);
          size_t z0 = IX(c, i, j, 0), zim = IX(c, i - 1, j, 0), zjm = IX(c, i, j - 1, 0);
          double Kx = 0.5 * (d.K[IX(c, i - 1, j, k)] + d.K[a]);
          double Ky = 0.5 * (d.K[IX(c, i, j - 1, k)] + d.K[a]);
          double dpx = (phi[a] - phi[IX(c, i - 1, j, k)]) / dx - c->sxu[a] * avg_q_valid(c, qph, zim, z0, k);
          double dpy = (phi[a] - phi[IX(c, i, j - 1, k)]) / dy - c->syv[a] * avg_q_valid(c, qph, zjm, z0, k);
          Gx[a] = -Kx * dpx;
          Gy[a] = -Ky * dpy;
        }
    fill_lateral(c, Gx);
    fill_lateral(c, Gy);
    for (int k = 1; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          size_t a = IX(c, i, j, k);
          double Kw = 0.5 * (d.K[IX(c, i, j, k - 1)] + d.K[a]);
          double gxb = 0.25 * (Gx[IX(c, i, j, k - 1)] + Gx[IX(c, i + 1, j, k - 1)] + Gx[a] + Gx[IX(c, i + 1, j, k)]);
          double gyb = 0.25 * (Gy[IX(c, i, j, k - 1)] + Gy[IX(c, i, j + 1, k - 1)] + Gy[a] + Gy[IX(c, i, j + 1, k)]);
          Gz[a] = -Kw * qph[a] - c->sxw[a] * gxb - c->syw[a] * gyb;
        } /* Gz = 0 on the lids */
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          size_t a = IX(c, i, j, k);
          size_t ip = IX(c, i + 1, j, k), jp = IX(c, i, j + 1, k), kp = IX(c, i, j, k + 1);
          R[a] -= ((c->hx[ip] * Gx[ip] - c->hx[a] * Gx[a]) / dx + (c->hy[jp] * Gy[jp] - c->hy[a] * Gy[a]) / dy +
                   (Gz[kp] - Gz[a])) / c->hc[a];
        }
    free(qph); free(Gx); free(Gy); free(Gz);
    free(d.mu); free(d.K); free(d.S11); free(d.S22); free(d.S33);
    free(d.S12); free(d.S13); free(d.S23); free(d.qu); free(d.qv);
    free(q.theta); free(q.pp); free(q.pi); free(q.u); free(q.v); free(q.w);
  }
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        Qout[a] = Qn[a] + dts * R[a];
      }
  fill_lateral(c, Qout);
  free(phi); free(Fx); free(Fy); free(R);
}

/* ------------------------------------------------------------------ */
/* S6: RK3 driver (Eq. 11-13) with the schedule of L170     */
/* ------------------------------------------------------------------ */

void erfo_schedule(int stage, double dt, int n_acoustic, int *nsub, double *dtau, double *dts) {
  if (stage == 1) { *nsub = 1; *dtau = dt / 3.0; *dts = dt / 3.0; }              /* one substep [P:L170] */
  else if (stage == 2) { *nsub = n_acoustic / 2; *dtau = dt / n_acoustic; *dts = dt / 2.0; }
  else { *nsub = n_acoustic; *dtau = dt / n_acoustic; *dts = dt; }
}

int erfo_rk3_step(erfo_ctx *c, double dt, int n_acoustic) {
  if (!c || !(dt > 0.0)) return -1;
  if (c->p.substep_mode == 1 && (n_acoustic < 2 || (n_acoustic & 1))) return -1;
  double *St[5], *R[5], *P[5];
  for (int m = 0; m < 5; m++) { St[m] = fnew(c); R[m] = fnew(c); P[m] = fnew(c); }
  double *theta_t = fnew(c), *pi_t = fnew(c);
  for (int m = 0; m < 5; m++) memcpy(St[m], c->S[m], c->n * sizeof(double)); /* S^t = S^n */
  /* transported scalar: stage value Q^t, time-averaged momenta of the stage */
  double *Qt = NULL, *Qnew = NULL, *Mavg[3] = {NULL, NULL, NULL}, *Omt = NULL;
  if (c->Q) {
    Qt = fnew(c); Qnew = fnew(c); Omt = fnew(c);
    for (int m = 0; m < 3; m++) Mavg[m] = fnew(c);
    memcpy(Qt, c->Q, c->n * sizeof(double));
  }
  for (int stage = 1; stage <= 3; stage++) {
    int nsub; double dtau, dts;
    erfo_schedule(stage, dt, n_acoustic, &nsub, &dtau, &dts);
    slow_rhs(c, St, R, theta_t, pi_t); /* f(S^t), recomputed every stage (L140) */
    if (c->p.substep_mode == 0) {
      /* no substepping (L140): S_stage = S^n + dts * f(S^t) */
      if (c->Q) { /* no substepping: the stage momenta themselves advect the scalar */
        contravariant_flux(c, St[UU], St[VV], St[WW], Omt);
        scalar_stage(c, St, Qt, c->Q, St[UU], St[VV], Omt, dts, Qnew);
        memcpy(Qt, Qnew, c->n * sizeof(double));
      }
      for (int m = 0; m < 5; m++)
        for (size_t a = 0; a < c->n; a++) St[m][a] = c->S[m][a] + dts * R[m][a];
    } else {
      /* perturbation about the most recent stage (L581); every stage starts from S^n [R:G7] */
      for (int m = 0; m < 5; m++)
        for (size_t a = 0; a < c->n; a++) P[m][a] = c->S[m][a] - St[m][a];
      acoustic_loop(c, St, theta_t, pi_t, R, P, dtau, nsub, c->Q ? Mavg : NULL);
      if (c->Q) { /* Eq. 4 after the substeps (L138): averaged momenta = stage momenta + averaged perturbations */
        contravariant_flux(c, St[UU], St[VV], St[WW], Omt);
        for (size_t a = 0; a < c->n; a++) {
          Mavg[0][a] += St[UU][a];
          Mavg[1][a] += St[VV][a];
          Mavg[2][a] += Omt[a];
        }
        scalar_stage(c, St, Qt, c->Q, Mavg[0], Mavg[1], Mavg[2], dts, Qnew);
        memcpy(Qt, Qnew, c->n * sizeof(double));
      }
      for (int m = 0; m < 5; m++) /* L593 */
        for (size_t a = 0; a < c->n; a++) St[m][a] = St[m][a] + P[m][a];
    }
    impose_inflow(c, St);
    for (int m = 0; m < 5; m++) fill_lateral(c, St[m]);
    impose_lids(c, St[UU], St[VV], St[WW]);
  }
  for (int m = 0; m < 5; m++) memcpy(c->S[m], St[m], c->n * sizeof(double));
  for (int m = 0; m < 5; m++) { free(St[m]); free(R[m]); free(P[m]); }
  free(theta_t); free(pi_t);
  if (c->Q) {
    memcpy(c->Q, Qt, c->n * sizeof(double));
    free(Qt); free(Qnew); free(Omt);
    for (int m = 0; m < 3; m++) free(Mavg[m]);
  }
  return 0;
}

/* ------------------------------------------------------------------ */
/* Anelastic mode (Sec. 2.2 L88-L96 Eq. 8; Sec. 3.2 */
/* Eq. 14-16).  Flat, laterally periodic grids (stretched levels ok).  */
/* ------------------------------------------------------------------ */

/* L96: "the buoyancy force B for dry air [is] rho0 (theta - theta0)/theta0 g"; "the pressure perturbation p' that enters
 * the momentum equation is computed solely from the Poisson equation".  R_U -= Gx(p'), R_V -= Gy(p') with the operators of
 * S4; at w-faces R_W -= (p'(k) - p'(k-1))/hw(k) and R_W += g * mean of B/g over the two adjacent cells [R:G11]. */
static void anelastic_pressure_buoyancy(const erfo_ctx *c, const prim_t *q, const double *pan, double *R[5]) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        R[UU][a] -= grad_x(c, pan, i, j, k);
        R[VV][a] -= grad_y(c, pan, i, j, k);
        if (k >= 1) {
          size_t b = IX(c, i, j, k - 1);
          double th0a = c->Th0[a] / c->rho0[a], th0b = c->Th0[b] / c->rho0[b];
          double Ba = c->rho0[a] * (q->theta[a] - th0a) / th0a, Bb = c->rho0[b] * (q->theta[b] - th0b) / th0b;
          R[WW][a] += -(pan[a] - pan[b]) / c->hw[a] + c->p.g * 0.5 * (Bb + Ba);
        }
      }
}

/* discrete divergence of the momenta at cell centres: D(M) = dU/dx + dV/dy + dW/dz (flat grid: Omega = W, hx = hy = hc) */
static void divergence(const erfo_ctx *c, const double *U, const double *V, const double *W, double *D) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        D[a] = (U[IX(c, i + 1, j, k)] - U[a]) / c->dx + (V[IX(c, i, j + 1, k)] - V[a]) / c->dy +
               (W[IX(c, i, j, k + 1)] - W[a]) / c->hc[a];
      }
}

/* Eq. 16: dt div(grad psi) = div(rho0 u**), then rho0 u* = rho0 u** - dt grad psi and p' += psi (L158-L162).
 * grad psi lives on the faces: (psi(i) - psi(i-1))/dx, (psi(j) - psi(j-1))/dy, (psi(k) - psi(k-1))/hw(k) on interior
 * w-faces, nothing on the rigid lids (W = 0 there): the discrete Laplacian is div of this grad, symmetric, with the
 * constants as its null space.  "ERF provides several options for solving the Poisson equation: geometric multigrid,
 * Fast Fourier Transforms (FFTs) and ..." (L164): here the discrete Fourier transform in the two periodic directions,
 * written out as its definition, and one tridiagonal system in z per horizontal mode (m, n):
 *   [lx(m) + ly(n)] P_k + [ (P_{k+1} - P_k)/hw_{k+1} - (P_k - P_{k-1})/hw_k ] / dz_k = Dhat_k / dt,
 *   lx(m) = -(4/dx^2) sin^2(pi m / nx),  ly(n) = -(4/dy^2) sin^2(pi n / ny);
 * the singular mode (0, 0) is fixed by psi_hat(k = 0) = 0 [R:G29]. */
static void project(erfo_ctx *c, double *U, double *V, double *W, double dt) {
  int nx = c->nx, ny = c->ny, nz = c->nz;
  const double PI = 3.14159265358979323846;
  size_t nh = (size_t)nx * ny;
  double *D = fnew(c);
  divergence(c, U, V, W, D);
  /* forward transform: Dhat(m, n, k) = sum_{i,j} D(i, j, k) exp(-2 pi I (m i / nx + n j / ny)) */
  double *Ar = (double *)malloc(nh * nz * sizeof(double)), *Ai = (double *)malloc(nh * nz * sizeof(double));
  double *Br = (double *)malloc(nh * nz * sizeof(double)), *Bi = (double *)malloc(nh * nz * sizeof(double));
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++) {
    for (int j = 0; j < ny; j++)
      for (int m = 0; m < nx; m++) { /* x */
        double sr = 0.0, si = 0.0;
        for (int i = 0; i < nx; i++) {
          double ph = -2.0 * PI * (double)((long long)m * i % nx) / nx;
          double d = D[IX(c, i, j, k)];
          sr += d * cos(ph);
          si += d * sin(ph);
        }
        Ar[(size_t)k * nh + (size_t)j * nx + m] = sr;
        Ai[(size_t)k * nh + (size_t)j * nx + m] = si;
      }
    for (int n = 0; n < ny; n++)
      for (int m = 0; m < nx; m++) { /* y */
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < ny; j++) {
          double ph = -2.0 * PI * (double)((long long)n * j % ny) / ny;
          double cr = cos(ph), ci = sin(ph);
          double ar = Ar[(size_t)k * nh + (size_t)j * nx + m], ai = Ai[(size_t)k * nh + (size_t)j * nx + m];
          sr += ar * cr - ai * ci;
          si += ar * ci + ai * cr;
        }
        Br[(size_t)k * nh + (size_t)n * nx + m] = sr;
        Bi[(size_t)k * nh + (size_t)n * nx + m] = si;
      }
  }
  /* one real tridiagonal matrix per mode, solved (Thomas) for the real and the imaginary part */
#pragma omp parallel for schedule(static)
  for (int n = 0; n < ny; n++)
    for (int m = 0; m < nx; m++) {
      double sx = sin(PI * m / nx), sy = sin(PI * n / ny);
      double lam = -4.0 * sx * sx / (c->dx * c->dx) - 4.0 * sy * sy / (c->dy * c->dy);
      double *cp = (double *)malloc(nz * sizeof(double));
      double *dr = (double *)malloc(nz * sizeof(double)), *di = (double *)malloc(nz * sizeof(double));
      for (int k = 0; k < nz; k++) {
        size_t a = IX(c, 0, 0, k); /* flat grid: level metrics from column (0, 0) */
        double dz = c->hc[a];
        double lo = k >= 1 ? 1.0 / (c->hw[a] * dz) : 0.0;
        double up = k <= nz - 2 ? 1.0 / (c->hw[IX(c, 0, 0, k + 1)] * dz) : 0.0;
        double diag = lam - lo - up;
        size_t q = (size_t)k * nh + (size_t)n * nx + m;
        double rr = Br[q] / dt, ri = Bi[q] / dt;
        if (m == 0 && n == 0 && k == 0) { lo = 0.0; up = 0.0; diag = 1.0; rr = 0.0; ri = 0.0; }
        double den = diag - (k >= 1 ? lo * cp[k - 1] : 0.0);
        cp[k] = up / den;
        dr[k] = (rr - (k >= 1 ? lo * dr[k - 1] : 0.0)) / den;
        di[k] = (ri - (k >= 1 ? lo * di[k - 1] : 0.0)) / den;
      }
      for (int k = nz - 1; k >= 0; k--) {
        size_t q = (size_t)k * nh + (size_t)n * nx + m;
        double pr = dr[k] - (k <= nz - 2 ? cp[k] * Br[q + nh] : 0.0);
        double pi = di[k] - (k <= nz - 2 ? cp[k] * Bi[q + nh] : 0.0);
        Br[q] = pr;
        Bi[q] = pi;
      }
      free(cp); free(dr); free(di);
    }
  /* inverse transform (real part; the imaginary part vanishes for a real right-hand side) */
  double *psi = fnew(c);
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++) {
    for (int j = 0; j < ny; j++)
      for (int m = 0; m < nx; m++) { /* y */
        double sr = 0.0, si = 0.0;
        for (int n = 0; n < ny; n++) {
          double ph = 2.0 * PI * (double)((long long)n * j % ny) / ny;
          double cr = cos(ph), ci = sin(ph);
          double br = Br[(size_t)k * nh + (size_t)n * nx + m], bi = Bi[(size_t)k * nh + (size_t)n * nx + m];
          sr += br * cr - bi * ci;
          si += br * ci + bi * cr;
        }
        Ar[(size_t)k * nh + (size_t)j * nx + m] = sr;
        Ai[(size_t)k * nh + (size_t)j * nx + m] = si;
      }
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) { /* x */
        double sr = 0.0;
        for (int m = 0; m < nx; m++) {
          double ph = 2.0 * PI * (double)((long long)m * i % nx) / nx;
          sr += Ar[(size_t)k * nh + (size_t)j * nx + m] * cos(ph) - Ai[(size_t)k * nh + (size_t)j * nx + m] * sin(ph);
        }
        psi[IX(c, i, j, k)] = sr / ((double)nx * ny);
      }
  }
  free(Ar); free(Ai); free(Br); free(Bi);
  fill_lateral(c, psi);
  /* correct the momenta, accumulate the pressure */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        U[a] -= dt * (psi[a] - psi[IX(c, i - 1, j, k)]) / c->dx;
        V[a] -= dt * (psi[a] - psi[IX(c, i, j - 1, k)]) / c->dy;
        if (k >= 1) W[a] -= dt * (psi[a] - psi[IX(c, i, j, k - 1)]) / c->hw[a];
        c->pan[a] += psi[a];
      }
  fill_lateral(c, U); fill_lateral(c, V); fill_lateral(c, W); fill_lateral(c, c->pan);
  free(D); free(psi);
}

static int anelastic_ok(erfo_ctx *c, int flat) {
  if (!c || !flat || !c->perx || !c->pery) return 0;
  if (!c->pan) c->pan = fnew(c);
  return 1;
}

/* test entry points: project the current momenta with time step dt; the divergence of the current momenta; p' */
int erfo_project(erfo_ctx *c, double dt) {
  if (!anelastic_ok(c, c ? c->flat : 0) || !(dt > 0.0)) return -1;
  project(c, c->S[UU], c->S[VV], c->S[WW], dt);
  return 0;
}

int erfo_divergence(erfo_ctx *c, double *D) {
  if (!c || !D) return -1;
  double *d = fnew(c);
  divergence(c, c->S[UU], c->S[VV], c->S[WW], d);
  get_dense(c, d, D, c->nz);
  free(d);
  return 0;
}

int erfo_get_pprime(erfo_ctx *c, double *pp) {
  if (!c || !pp || !c->pan) return -1;
  get_dense(c, c->pan, pp, c->nz);
  return 0;
}

/* One RK2 step of the anelastic equations (Eq. 14-15), a projection after each stage (L154-L162):
 *   S*      = S^n + dt f(S^n),                  projected with dt;
 *   S^{n+1} = S^n + dt/2 (f(S^n) + f(S*)),      projected with dt ("an analogous procedure", L162).
 * rho is held at rho0 ("we can replace rho_d by rho_0 ... which makes the continuity equation redundant", L94): the
 * density of the context's state is overwritten by the base state.  f is f(S) of the compressible core with the
 * pressure-gradient / buoyancy pair of Sec. 2.2; no acoustic substeps ("with no substepping in each RK stage", L148).
 * p' accumulates psi after EACH projection, as printed (L160) [R:G29]. */
int erfo_anelastic_step(erfo_ctx *c, double dt) {
  if (!anelastic_ok(c, c ? c->flat : 0) || !(dt > 0.0)) return -1;
  memcpy(c->S[RHO], c->rho0, c->n * sizeof(double));
  double *St[5], *R1[5], *R2[5];
  for (int m = 0; m < 5; m++) { St[m] = fnew(c); R1[m] = fnew(c); R2[m] = fnew(c); }
  slow_rhs_mode(c, c->S, R1, NULL, NULL, c->pan);
  for (int m = 0; m < 5; m++)
    for (size_t a = 0; a < c->n; a++) St[m][a] = m == RHO ? c->S[m][a] : c->S[m][a] + dt * R1[m][a];
  for (int m = 0; m < 5; m++) fill_lateral(c, St[m]);
  impose_lids(c, St[UU], St[VV], St[WW]);
  project(c, St[UU], St[VV], St[WW], dt);
  slow_rhs_mode(c, St, R2, NULL, NULL, c->pan);
  for (int m = 0; m < 5; m++)
    for (size_t a = 0; a < c->n; a++)
      St[m][a] = m == RHO ? c->S[m][a] : c->S[m][a] + 0.5 * dt * (R1[m][a] + R2[m][a]);
  for (int m = 0; m < 5; m++) fill_lateral(c, St[m]);
  impose_lids(c, St[UU], St[VV], St[WW]);
  project(c, St[UU], St[VV], St[WW], dt);
  for (int m = 0; m < 5; m++) memcpy(c->S[m], St[m], c->n * sizeof(double));
  for (int m = 0; m < 5; m++) { free(St[m]); free(R1[m]); free(R2[m]); }
  return 0;
}

/* ------------------------------------------------------------------ */
/* context                                                             */
/* ------------------------------------------------------------------ */

int erfo_create(const erfo_grid *g, const erfo_metrics *m, const erfo_params *p, erfo_ctx **out) {
  if (!g || !m || !p || !out) return -1;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1 || !(g->dx > 0) || !(g->dy > 0)) return -1;
  if (!m->rho0 || !m->rhotheta0 || (!m->z_nodes && !m->z_levels)) return -1;
  if (p->adv_order_h < 2 || p->adv_order_h > 6 || p->adv_order_v < 2 || p->adv_order_v > 6) return -1;
  if (p->scalar_adv != 0 && p->scalar_adv != 13 && p->scalar_adv != 15 && p->scalar_adv != 23 && p->scalar_adv != 25)
    return -1;
  erfo_ctx *c = (erfo_ctx *)calloc(1, sizeof(erfo_ctx));
  c->nx = g->nx; c->ny = g->ny; c->nz = g->nz; c->dx = g->dx; c->dy = g->dy;
  c->perx = g->periodic_x == 1; c->pery = g->periodic_y == 1;
  c->inx = g->periodic_x == 2; c->iny = g->periodic_y == 2;
  c->flat = m->z_nodes == NULL;
  c->p = *p;
  c->cv = p->cp - p->Rd;
  c->gam = p->cp / c->cv;
  c->rdocv = p->Rd / c->cv;
  c->sj = (size_t)(g->nx + 2 * NG);
  c->sk = c->sj * (size_t)(g->ny + 2 * NG);
  c->n = c->sk * (size_t)(g->nz + 1);
  double **geo[] = {&c->zxf, &c->zyf, &c->zw, &c->hx, &c->hy, &c->hc, &c->zc, &c->hw, &c->hu,
                    &c->hv, &c->sxw, &c->syw, &c->sxu, &c->syv, &c->rho0, &c->Th0, &c->p0, &c->pi0};
  for (size_t a = 0; a < sizeof(geo) / sizeof(geo[0]); a++) *geo[a] = fnew(c);
  for (int s = 0; s < 5; s++) c->S[s] = fnew(c);
  /* node heights */
  int nx = c->nx, ny = c->ny, nz = c->nz;
  size_t nn = (size_t)(nx + 1) * (ny + 1) * (nz + 1);
  double *zn = (double *)malloc(nn * sizeof(double));
  if (m->z_nodes) memcpy(zn, m->z_nodes, nn * sizeof(double));
  else
    for (int k = 0; k <= nz; k++)
      for (size_t a = 0; a < (size_t)(nx + 1) * (ny + 1); a++)
        zn[(size_t)k * (nx + 1) * (ny + 1) + a] = m->z_levels[k];
  build_geometry(c, zn);
  free(zn);
  /* base state: rho0, Theta0 given; p0, pi0 from Eq. 7 [R:S1] */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t a = IX(c, i, j, k);
        size_t s = m->base_is_1d ? (size_t)k : ((size_t)k * ny + j) * nx + i;
        c->rho0[a] = m->rho0[s];
        c->Th0[a] = m->rhotheta0[s];
        c->p0[a] = p->p00 * pow(p->Rd * c->Th0[a] / p->p00, c->gam);
        c->pi0[a] = pow(p->Rd * c->Th0[a] / p->p00, c->rdocv);
      }
  fill_lateral(c, c->rho0); fill_lateral(c, c->Th0);
  fill_lateral(c, c->p0); fill_lateral(c, c->pi0);
  *out = c;
  return 0;
}

void erfo_destroy(erfo_ctx *c) {
  if (!c) return;
  double *all[] = {c->zxf, c->zyf, c->zw, c->hx, c->hy, c->hc, c->zc, c->hw, c->hu, c->hv,
                   c->sxw, c->syw, c->sxu, c->syv, c->rho0, c->Th0, c->p0, c->pi0,
                   c->S[0], c->S[1], c->S[2], c->S[3], c->S[4]};
  for (size_t a = 0; a < sizeof(all) / sizeof(all[0]); a++) free(all[a]);
  free(c->Q);
  free(c->pan);
  for (int m = 0; m < 5; m++) free(c->inflow[m]);
  free(c);
}

int erfo_set_state(erfo_ctx *c, const double *rho, const double *rhou, const double *rhov,
                   const double *rhow, const double *rhotheta) {
  if (!c || !rho || !rhou || !rhov || !rhow || !rhotheta) return -1;
  put_dense(c, c->S[RHO], rho, c->nz);
  put_dense(c, c->S[UU], rhou, c->nz);
  put_dense(c, c->S[VV], rhov, c->nz);
  put_dense(c, c->S[WW], rhow, c->nz + 1);
  put_dense(c, c->S[TH], rhotheta, c->nz);
  impose_lids(c, c->S[UU], c->S[VV], c->S[WW]);
  if (c->inx || c->iny)
    for (int m = 0; m < 5; m++) {
      if (!c->inflow[m]) c->inflow[m] = fnew(c);
      memcpy(c->inflow[m], c->S[m], c->n * sizeof(double));
    }
  return 0;
}

/* Eq. 4 (L69): give the context one transported scalar, as rho*phi [nz][ny][nx]; erfo_rk3_step then advances it */
int erfo_set_scalar(erfo_ctx *c, const double *rhophi) {
  if (!c || !rhophi) return -1;
  if (!c->Q) c->Q = fnew(c);
  put_dense(c, c->Q, rhophi, c->nz);
  return 0;
}

int erfo_get_scalar(erfo_ctx *c, double *rhophi) {
  if (!c || !rhophi || !c->Q) return -1;
  get_dense(c, c->Q, rhophi, c->nz);
  return 0;
}

int erfo_get_state(erfo_ctx *c, double *rho, double *rhou, double *rhov, double *rhow,
                   double *rhotheta) {
  if (!c) return -1;
  if (rho) get_dense(c, c->S[RHO], rho, c->nz);
  if (rhou) get_dense(c, c->S[UU], rhou, c->nz);
  if (rhov) get_dense(c, c->S[VV], rhov, c->nz);
  if (rhow) get_dense(c, c->S[WW], rhow, c->nz + 1);
  if (rhotheta) get_dense(c, c->S[TH], rhotheta, c->nz);
  return 0;
}

/* ------------------------------------------------------------------ */
/* test entry points                                                   */
/* ------------------------------------------------------------------ */

int erfo_slow_rhs(erfo_ctx *c, double *R_rho, double *R_U, double *R_V, double *R_W,
                  double *R_Theta) {
  if (!c) return -1;
  double *R[5];
  for (int m = 0; m < 5; m++) R[m] = fnew(c);
  slow_rhs(c, c->S, R, NULL, NULL);
  if (R_rho) get_dense(c, R[RHO], R_rho, c->nz);
  if (R_U) get_dense(c, R[UU], R_U, c->nz);
  if (R_V) get_dense(c, R[VV], R_V, c->nz);
  if (R_W) get_dense(c, R[WW], R_W, c->nz + 1);
  if (R_Theta) get_dense(c, R[TH], R_Theta, c->nz);
  for (int m = 0; m < 5; m++) free(R[m]);
  return 0;
}

int erfo_viscosity(erfo_ctx *c, double *mu) {
  if (!c || !mu) return -1;
  prim_t q;
  q.theta = fnew(c); q.pp = fnew(c); q.pi = fnew(c);
  q.u = fnew(c); q.v = fnew(c); q.w = fnew(c);
  primitives(c, c->S, &q);
  diff_t d;
  d.mu = fnew(c); d.K = fnew(c);
  d.S11 = fnew(c); d.S22 = fnew(c); d.S33 = fnew(c);
  d.S12 = fnew(c); d.S13 = fnew(c); d.S23 = fnew(c);
  d.qu = fnew(c); d.qv = fnew(c);
  strain_and_viscosity(c, c->S, &q, &d);
  get_dense(c, d.mu, mu, c->nz);
  free(d.mu); free(d.K); free(d.S11); free(d.S22); free(d.S33);
  free(d.S12); free(d.S13); free(d.S23); free(d.qu); free(d.qv);
  free(q.theta); free(q.pp); free(q.pi); free(q.u); free(q.v); free(q.w);
  return 0;
}

int erfo_get_geometry(erfo_ctx *c, const char *name, double *out) {
  if (!c || !name || !out) return -1;
  const char *names[] = {"hc", "zc", "hw", "hx", "hy", "hu", "hv", "sxw", "syw", "sxu", "syv", "zw"};
  double *arr[] = {c->hc, c->zc, c->hw, c->hx, c->hy, c->hu, c->hv, c->sxw, c->syw, c->sxu, c->syv, c->zw};
  for (size_t a = 0; a < sizeof(arr) / sizeof(arr[0]); a++)
    if (strcmp(name, names[a]) == 0) {
      get_dense(c, arr[a], out, c->nz + 1);
      return 0;
    }
  return -1;
}

int erfo_acoustic(erfo_ctx *c, double dtau, int n, const double *R_rho, const double *R_U,
                  const double *R_V, const double *R_W, const double *R_Theta, double *rho_pp,
                  double *U_pp, double *V_pp, double *W_pp, double *Theta_pp) {
  if (!c) return -1;
  double *R[5], *P[5];
  for (int m = 0; m < 5; m++) { R[m] = fnew(c); P[m] = fnew(c); }
  put_dense(c, R[RHO], R_rho, c->nz); put_dense(c, R[UU], R_U, c->nz);
  put_dense(c, R[VV], R_V, c->nz); put_dense(c, R[WW], R_W, c->nz + 1);
  put_dense(c, R[TH], R_Theta, c->nz);
  put_dense(c, P[RHO], rho_pp, c->nz); put_dense(c, P[UU], U_pp, c->nz);
  put_dense(c, P[VV], V_pp, c->nz); put_dense(c, P[WW], W_pp, c->nz + 1);
  put_dense(c, P[TH], Theta_pp, c->nz);
  prim_t q;
  q.theta = fnew(c); q.pp = fnew(c); q.pi = fnew(c);
  q.u = fnew(c); q.v = fnew(c); q.w = fnew(c);
  primitives(c, c->S, &q);
  acoustic_loop(c, c->S, q.theta, q.pi, R, P, dtau, n, NULL);
  get_dense(c, P[RHO], rho_pp, c->nz); get_dense(c, P[UU], U_pp, c->nz);
  get_dense(c, P[VV], V_pp, c->nz); get_dense(c, P[WW], W_pp, c->nz + 1);
  get_dense(c, P[TH], Theta_pp, c->nz);
  free(q.theta); free(q.pp); free(q.pi); free(q.u); free(q.v); free(q.w);
  for (int m = 0; m < 5; m++) { free(R[m]); free(P[m]); }
  return 0;
}

int erfo_tridiag_rows(erfo_ctx *c, double dtau, int i, int j, double *A, double *D, double *C) {
  if (!c || !A || !D || !C) return -1;
  prim_t q;
  q.theta = fnew(c); q.pp = fnew(c); q.pi = fnew(c);
  q.u = fnew(c); q.v = fnew(c); q.w = fnew(c);
  primitives(c, c->S, &q);
  acoustic_t ac;
  memset(&ac, 0, sizeof(ac));
  ac.theta_t = q.theta; ac.pi_t = q.pi; ac.Th_t = c->S[TH];
  A[0] = D[0] = C[0] = 0.0;
  for (int k = 1; k < c->nz; k++) tridiag_row(c, &ac, dtau, i, j, k, &A[k], &D[k], &C[k]);
  free(q.theta); free(q.pp); free(q.pi); free(q.u); free(q.v); free(q.w);
  return 0;
}
