// general_cells.cuh -- per-cell bodies of the GENERAL (unfused, terrain-capable) path.
//
// One function per operator pass of the discretisation D0: each computes the
// value(s) of one output field at one index from fields in HBM.  The __global__ wrappers in
// k_general.cu launch them one thread per (i,j,k).  This path keeps every intermediate
// field in HBM; it exists (a) to serve terrain-following grids, where the metric terms make
// the operators too irregular for the fused flat-grid kernels, and (b) as an on-device
// cross-check of those fused kernels at full problem size.
//
// Citations are to /root/reference/PAPER.md; [R:Gn] are the readings listed in DESIGN.md.
#pragma once
#include <math.h>

#include "erf_view.cuh"

namespace erfb {
namespace gen {

// ---------------------------------------------------------------- geometry (S0) [R:G14]
// L178: terrain at nodes, vertical deformation only.  All metrics = differences of node heights.
struct NodeH {
  const double *zn;  // [(nz+1)][(ny+1)][(nx+1)] or null
  const double *zl;  // [(nz+1)] (flat)
  int nx, ny;
  ERF_HD double operator()(int i, int j, int k) const {
    return zn ? zn[((size_t)k * (ny + 1) + j) * (nx + 1) + i] : zl[k];
  }
};

template <class VT>
ERF_HD void geo_faces(const VT &c, const NodeH &Z, double *zxf, double *zyf, double *zw, int i,
                      int j, int k) {  // k = 0..nz
  size_t a = IX(c, i, j, k);
  zxf[a] = 0.5 * (Z(i, j, k) + Z(i, j + 1, k));
  zyf[a] = 0.5 * (Z(i, j, k) + Z(i + 1, j, k));
  zw[a] = 0.25 * (Z(i, j, k) + Z(i + 1, j, k) + Z(i, j + 1, k) + Z(i + 1, j + 1, k));
}

template <class VT>
ERF_HD void geo_cells(const VT &c, const double *zxf, const double *zyf, const double *zw,
                      double *hx, double *hy, double *hc, double *zc, int i, int j, int k) {  // k<nz
  size_t a = IX(c, i, j, k), t = IX(c, i, j, k + 1);
  hx[a] = zxf[t] - zxf[a];
  hy[a] = zyf[t] - zyf[a];
  hc[a] = zw[t] - zw[a];
  zc[a] = 0.5 * (zw[a] + zw[t]);
}

template <class VT>
ERF_HD void geo_derived(const VT &c, const double *zxf, const double *zyf, const double *hc,
                        const double *zc, double *hw, double *hu, double *hv, double *sxu,
                        double *syv, double *sxw, double *syw, int i, int j, int k) {  // k = 0..nz
  size_t a = IX(c, i, j, k);
  if (k < c.nz) {
    size_t im = IX(c, i - 1, j, k), jm = IX(c, i, j - 1, k);
    hu[a] = 0.5 * (hc[im] + hc[a]);
    hv[a] = 0.5 * (hc[jm] + hc[a]);
    sxu[a] = (zc[a] - zc[im]) / c.dx;
    syv[a] = (zc[a] - zc[jm]) / c.dy;
    hw[a] = (k >= 1) ? zc[a] - zc[IX(c, i, j, k - 1)] : 0.0;
  }
  sxw[a] = (zxf[IX(c, i + 1, j, k)] - zxf[a]) / c.dx;
  syw[a] = (zyf[IX(c, i, j + 1, k)] - zyf[a]) / c.dy;
}

// base state p0, pi0 from Theta0 through Eq. 7 (L80) [R:S1]
template <class VT>
ERF_HD void base_state(const VT &c, const double *rho0_in, const double *Th0_in, int base1d,
                       double *rho0, double *Th0, double *p0, double *pi0, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  size_t s = base1d ? (size_t)k : a;
  double T0 = Th0_in[s];
  rho0[a] = rho0_in[s];
  Th0[a] = T0;
  p0[a] = c.p00 * pow(c.Rd * T0 / c.p00, c.gam);
  pi0[a] = pow(c.Rd * T0 / c.p00, c.rdocv);
}

// ---------------------------------------------------------------- lids and Omega [R:G14,G15]
// kinematic W on the lids: Omega = 0 there
template <class VT>
ERF_HD void lids(const VT &c, const double *U, const double *V, double *W, int i, int j) {
  int nz = c.nz;
  W[IX(c, i, j, 0)] = c.sxw[IX(c, i, j, 0)] * 0.5 * (U[IX(c, i, j, 0)] + U[IX(c, i + 1, j, 0)]) +
                      c.syw[IX(c, i, j, 0)] * 0.5 * (V[IX(c, i, j, 0)] + V[IX(c, i, j + 1, 0)]);
  W[IX(c, i, j, nz)] =
      c.sxw[IX(c, i, j, nz)] * 0.5 * (U[IX(c, i, j, nz - 1)] + U[IX(c, i + 1, j, nz - 1)]) +
      c.syw[IX(c, i, j, nz)] * 0.5 * (V[IX(c, i, j, nz - 1)] + V[IX(c, i, j + 1, nz - 1)]);
}

// contravariant vertical mass flux (L196): Omega = W - sxw avg4(U) - syw avg4(V); 0 on lids
template <class VT>
ERF_HD double omega_at(const VT &c, const double *U, const double *V, const double *W, int i,
                       int j, int k) {
  if (k < 1 || k > c.nz - 1) return 0.0;
  double ubar = 0.25 * (U[IX(c, i, j, k - 1)] + U[IX(c, i + 1, j, k - 1)] + U[IX(c, i, j, k)] +
                        U[IX(c, i + 1, j, k)]);
  double vbar = 0.25 * (V[IX(c, i, j, k - 1)] + V[IX(c, i, j + 1, k - 1)] + V[IX(c, i, j, k)] +
                        V[IX(c, i, j + 1, k)]);
  size_t a = IX(c, i, j, k);
  return W[a] - c.sxw[a] * ubar - c.syw[a] * vbar;
}

// ---------------------------------------------------------------- primitives (S1)
struct Prim {
  double *theta, *pp, *pi, *u, *v, *w;
};

template <class VT>
ERF_HD void primitives(const VT &c, const double *const *S, const Prim &q, int i, int j,
                       int k) {  // k = 0..nz
  size_t a = IX(c, i, j, k);
  int nz = c.nz;
  if (k < nz) {
    double rho = S[RHO][a], Th = S[TH][a];
    q.theta[a] = Th / rho;
    double T0 = c.Th0[a];
    q.pp[a] = c.p0[a] * expm1(c.gam * log1p((Th - T0) / T0));  // Eq. 7 as p - p0 [R:S1]
    q.pi[a] = pow(c.Rd * Th / c.p00, c.rdocv);                // Exner (L84, L587)
    q.u[a] = S[UU][a] / (0.5 * (S[RHO][IX(c, i - 1, j, k)] + rho));
    q.v[a] = S[VV][a] / (0.5 * (S[RHO][IX(c, i, j - 1, k)] + rho));
  }
  double rw;
  if (k == 0) rw = S[RHO][a];
  else if (k == nz) rw = S[RHO][IX(c, i, j, nz - 1)];
  else rw = 0.5 * (S[RHO][IX(c, i, j, k - 1)] + S[RHO][a]);
  q.w[a] = S[WW][a] / rw;
}

// ---------------------------------------------------------------- Eq. 17-21 (L200-L211)
// q[0..5] = q_{m-3} .. q_{m+2}; flux point m-1/2.  Eq. 21 with sign/index repaired [R:G1].
// WENO-JS (kind 1) / WENO-Z (kind 2) of order 3 or 5 for cell-centred scalars (L213) [R:G26].  Written around the
// undivided differences of the window (e1 = q[k+1] - q[k]) rather than the textbook coefficient form: candidate
// values are the upwind cell plus a combination of its neighbouring differences.
ERF_HD double weno_up(int kind, int ord, double vm2, double vm1, double v0, double vp1, double vp2) {
  const double dm = v0 - vm1, dp = vp1 - v0;  // differences next to the upwind cell
  if (ord == 3) {
    const double b0 = dm * dm, b1 = dp * dp;
    double a0, a1;
    if (kind == 1) {
      const double e0 = 1e-6 + b0, e1 = 1e-6 + b1;
      a0 = 1.0 / (3.0 * e0 * e0);
      a1 = 2.0 / (3.0 * e1 * e1);
    } else {
      const double tau = fabs(b0 - b1);
      a0 = (1.0 + tau / (b0 + 1e-40)) / 3.0;
      a1 = (1.0 + tau / (b1 + 1e-40)) * (2.0 / 3.0);
    }
    return v0 + 0.5 * (a0 * dm + a1 * dp) / (a0 + a1);
  }
  const double dmm = vm1 - vm2, dpp = vp2 - vp1;
  // candidates: v0 + (1/6)(-2 dmm + 5 dm), v0 + (1/6)(dm + 2 dp), v0 + (1/6)(4 dp - dpp)... written out from the
  // sub-stencil parabolas in terms of differences
  const double c0 = (5.0 * dm - 2.0 * dmm) / 6.0, c1 = (dm + 2.0 * dp) / 6.0, c2 = (4.0 * dp - dpp) / 6.0;
  const double s0 = dm - dmm, s1 = dp - dm, s2 = dpp - dp;                    // second differences
  const double t0 = 3.0 * dm - dmm, t1 = dm + dp, t2 = 3.0 * dp - dpp;       // one-sided first differences (x2)
  const double b0 = (13.0 / 12.0) * s0 * s0 + 0.25 * t0 * t0;
  const double b1 = (13.0 / 12.0) * s1 * s1 + 0.25 * t1 * t1;
  const double b2 = (13.0 / 12.0) * s2 * s2 + 0.25 * t2 * t2;
  double a0, a1, a2;
  if (kind == 1) {
    const double e0 = 1e-6 + b0, e1 = 1e-6 + b1, e2 = 1e-6 + b2;
    a0 = 0.1 / (e0 * e0); a1 = 0.6 / (e1 * e1); a2 = 0.3 / (e2 * e2);
  } else {
    const double tau = fabs(b0 - b2);
    a0 = 0.1 * (1.0 + tau / (b0 + 1e-40)); a1 = 0.6 * (1.0 + tau / (b1 + 1e-40)); a2 = 0.3 * (1.0 + tau / (b2 + 1e-40));
  }
  return v0 + (a0 * c0 + a1 * c1 + a2 * c2) / (a0 + a1 + a2);
}

// order: 2..6 = Eq. 17-21; 13, 15 / 23, 25 = WENO-JS / WENO-Z of order 3, 5
ERF_HD double interp6(int order, double sgn, const double *q) {
  if (order >= 10)
    return sgn > 0.0 ? weno_up(order / 10, order % 10, q[0], q[1], q[2], q[3], q[4])
                     : weno_up(order / 10, order % 10, q[5], q[4], q[3], q[2], q[1]);
  double s2 = q[3] + q[2];
  if (order == 2) return 0.5 * s2;
  double s4 = q[4] + q[1];
  double q4 = (7.0 / 12.0) * s2 - (1.0 / 12.0) * s4;
  if (order == 4) return q4;
  if (order == 3) return q4 + sgn * (1.0 / 12.0) * ((q[4] - q[1]) - 3.0 * (q[3] - q[2]));
  double q6 = (37.0 / 60.0) * s2 - (2.0 / 15.0) * s4 + (1.0 / 60.0) * (q[5] + q[0]);
  if (order == 6) return q6;
  return q6 - sgn * (1.0 / 60.0) * ((q[5] - q[0]) - 5.0 * (q[4] - q[1]) + 10.0 * (q[3] - q[2]));
}

ERF_HD int vertical_order(int requested, int r) {  // [R:G13]
  if (requested >= 10) {  // WENO: 5-cell stencil needs 3 valid cells on either side, the 3-cell one 2
    if (r >= (requested % 10 + 1) / 2) return requested;
    return r >= 2 ? 10 * (requested / 10) + 3 : 2;
  }
  int need = (requested + 1) / 2;
  if (r >= need) return requested;
  if (r >= 2 && requested >= 3) return (requested & 1) ? 3 : 4;
  return 2;
}

ERF_HD double sgn_of(double m) { return m < 0.0 ? -1.0 : 1.0; }  // [R:G19]

template <class VT>
ERF_HD double interp_x(const VT &c, const double *f, int m, int j, int k, int order, double M) {
  double q[6] = {0, 0, 0, 0, 0, 0};
  int half = (order % 10 + 1) / 2;
  for (int n = 3 - half; n < 3 + half; n++) q[n] = f[IX(c, m - 3 + n, j, k)];
  return interp6(order, sgn_of(M), q);
}
template <class VT>
ERF_HD double interp_y(const VT &c, const double *f, int i, int m, int k, int order, double M) {
  double q[6] = {0, 0, 0, 0, 0, 0};
  int half = (order % 10 + 1) / 2;
  for (int n = 3 - half; n < 3 + half; n++) q[n] = f[IX(c, i, m - 3 + n, k)];
  return interp6(order, sgn_of(M), q);
}
// between levels m-1 and m; valid levels lo..hi
template <class VT>
ERF_HD double interp_z(const VT &c, const double *f, int i, int j, int m, int lo, int hi,
                       int order_req, double M) {
  int below = m - lo, above = hi - m + 1;
  int r = below < above ? below : above;
  int order = vertical_order(order_req, r);
  int half = (order % 10 + 1) / 2;
  double q[6] = {0, 0, 0, 0, 0, 0};
  for (int n = 3 - half; n < 3 + half; n++) q[n] = f[IX(c, i, j, m - 3 + n)];
  return interp6(order, sgn_of(M), q);
}

// ---------------------------------------------------------------- advection (S2)
// mass fluxes: Fx = hx U, Fy = hy V, Omega (precomputed field Om)
template <class VT>
ERF_HD double FX(const VT &c, const double *U, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  return c.hx[a] * U[a];
}
template <class VT>
ERF_HD double FY(const VT &c, const double *V, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  return c.hy[a] * V[a];
}

// R_rho, R_Theta, R_U, R_V at cell (i,j,k), k < nz   (Eq. 1-3 first terms; L196)
template <class VT>
ERF_HD void advect_cell(const VT &c, const double *const *S, const double *Om, const Prim &q,
                        double *const *R, int i, int j, int k) {
  const int nz = c.nz, oh = c.oh, ov = c.ov;
  const double *U = S[UU], *V = S[VV];
  size_t a = IX(c, i, j, k);
  double fxm = FX(c, U, i, j, k), fxp = FX(c, U, i + 1, j, k);
  double fym = FY(c, V, i, j, k), fyp = FY(c, V, i, j + 1, k);
  double omm = Om[a], omp = Om[IX(c, i, j, k + 1)];
  double rhc = 1.0 / c.hc[a];
  R[RHO][a] = -((fxp - fxm) / c.dx + (fyp - fym) / c.dy + (omp - omm)) * rhc;
  {
    const int sh = c.osh, sv = c.osv;  // cell-centred scalars: Eq. 17-21 or a WENO scheme (L213)
    double txm = fxm * interp_x(c, q.theta, i, j, k, sh, fxm);
    double txp = fxp * interp_x(c, q.theta, i + 1, j, k, sh, fxp);
    double tym = fym * interp_y(c, q.theta, i, j, k, sh, fym);
    double typ = fyp * interp_y(c, q.theta, i, j + 1, k, sh, fyp);
    double tzm = (k >= 1) ? omm * interp_z(c, q.theta, i, j, k, 0, nz - 1, sv, omm) : 0.0;
    double tzp = (k + 1 <= nz - 1) ? omp * interp_z(c, q.theta, i, j, k + 1, 0, nz - 1, sv, omp) : 0.0;
    R[TH][a] = -((txp - txm) / c.dx + (typ - tym) / c.dy + (tzp - tzm)) * rhc;
  }
  {  // U(i-1/2,j,k): momentum averaged to the flux location (L196) [R:G11]
    double fxmm = FX(c, U, i - 1, j, k);
    double Mxm = 0.5 * (fxmm + fxm), Mxp = 0.5 * (fxm + fxp);
    double Mym = 0.5 * (FY(c, V, i - 1, j, k) + fym);
    double Myp = 0.5 * (FY(c, V, i - 1, j + 1, k) + fyp);
    double Mzm = 0.5 * (Om[IX(c, i - 1, j, k)] + omm);
    double Mzp = 0.5 * (Om[IX(c, i - 1, j, k + 1)] + omp);
    double gxm = Mxm * interp_x(c, q.u, i, j, k, oh, Mxm);
    double gxp = Mxp * interp_x(c, q.u, i + 1, j, k, oh, Mxp);
    double gym = Mym * interp_y(c, q.u, i, j, k, oh, Mym);
    double gyp = Myp * interp_y(c, q.u, i, j + 1, k, oh, Myp);
    double gzm = (k >= 1) ? Mzm * interp_z(c, q.u, i, j, k, 0, nz - 1, ov, Mzm) : 0.0;
    double gzp = (k + 1 <= nz - 1) ? Mzp * interp_z(c, q.u, i, j, k + 1, 0, nz - 1, ov, Mzp) : 0.0;
    R[UU][a] = -((gxp - gxm) / c.dx + (gyp - gym) / c.dy + (gzp - gzm)) / c.hu[a];
  }
  {  // V(i,j-1/2,k)
    double fymm = FY(c, V, i, j - 1, k);
    double Mxm = 0.5 * (FX(c, U, i, j - 1, k) + fxm);
    double Mxp = 0.5 * (FX(c, U, i + 1, j - 1, k) + fxp);
    double Mym = 0.5 * (fymm + fym), Myp = 0.5 * (fym + fyp);
    double Mzm = 0.5 * (Om[IX(c, i, j - 1, k)] + omm);
    double Mzp = 0.5 * (Om[IX(c, i, j - 1, k + 1)] + omp);
    double gxm = Mxm * interp_x(c, q.v, i, j, k, oh, Mxm);
    double gxp = Mxp * interp_x(c, q.v, i + 1, j, k, oh, Mxp);
    double gym = Mym * interp_y(c, q.v, i, j, k, oh, Mym);
    double gyp = Myp * interp_y(c, q.v, i, j + 1, k, oh, Myp);
    double gzm = (k >= 1) ? Mzm * interp_z(c, q.v, i, j, k, 0, nz - 1, ov, Mzm) : 0.0;
    double gzp = (k + 1 <= nz - 1) ? Mzp * interp_z(c, q.v, i, j, k + 1, 0, nz - 1, ov, Mzp) : 0.0;
    R[VV][a] = -((gxp - gxm) / c.dx + (gyp - gym) / c.dy + (gzp - gzm)) / c.hv[a];
  }
}

// R_W at face (i,j,k), k = 0..nz (zero on the lids)
template <class VT>
ERF_HD void advect_wface(const VT &c, const double *const *S, const double *Om, const Prim &q,
                         double *const *R, int i, int j, int k) {
  const int nz = c.nz, oh = c.oh, ov = c.ov;
  const double *U = S[UU], *V = S[VV];
  size_t a = IX(c, i, j, k);
  if (k == 0 || k == nz) {
    R[WW][a] = 0.0;
    return;
  }
  double Mxm = 0.5 * (FX(c, U, i, j, k - 1) + FX(c, U, i, j, k));
  double Mxp = 0.5 * (FX(c, U, i + 1, j, k - 1) + FX(c, U, i + 1, j, k));
  double Mym = 0.5 * (FY(c, V, i, j, k - 1) + FY(c, V, i, j, k));
  double Myp = 0.5 * (FY(c, V, i, j + 1, k - 1) + FY(c, V, i, j + 1, k));
  double Mzm = 0.5 * (Om[IX(c, i, j, k - 1)] + Om[a]);
  double Mzp = 0.5 * (Om[a] + Om[IX(c, i, j, k + 1)]);
  double gxm = Mxm * interp_x(c, q.w, i, j, k, oh, Mxm);
  double gxp = Mxp * interp_x(c, q.w, i + 1, j, k, oh, Mxp);
  double gym = Mym * interp_y(c, q.w, i, j, k, oh, Mym);
  double gyp = Myp * interp_y(c, q.w, i, j + 1, k, oh, Myp);
  double gzm = Mzm * interp_z(c, q.w, i, j, k, 0, nz, ov, Mzm);
  double gzp = Mzp * interp_z(c, q.w, i, j, k + 1, 0, nz, ov, Mzp);
  R[WW][a] = -((gxp - gxm) / c.dx + (gyp - gym) / c.dy + (gzp - gzm)) / c.hw[a];
}

// ---------------------------------------------------------------- diffusion (S3)
struct Diff {
  double *mu, *K;
  double *S11, *S22, *S33, *S12, *S13, *S23;
  double *qu, *qv;                      // du/dz, dv/dz at xz-/yz-edges
  double *t11, *t22, *t33, *t12, *t13, *t23;
  double *q11, *q22, *q12, *q13, *q23, *qth;
  double *ze12;
  double *Fx, *Fy, *Fz;
};

// mean of the valid (k' in 1..nz-1) quotients at levels k, k+1 and two columns [R:G14]
template <class VT>
ERF_HD double avg_q_valid(const VT &c, const double *qv, int i0, int j0, int i1, int j1, int k) {
  double s = 0.0;
  int n = 0;
  for (int kk = k; kk <= k + 1; kk++)
    if (kk >= 1 && kk <= c.nz - 1) {
      s += qv[IX(c, i0, j0, kk)] + qv[IX(c, i1, j1, kk)];
      n += 2;
    }
  return n ? s / n : 0.0;
}

// pass D1: qu, qv (k = 1..nz-1; 0 elsewhere), S33 (k < nz)
template <class VT>
ERF_HD void diff_pass1(const VT &c, const Prim &q, const Diff &d, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  if (k >= 1 && k <= c.nz - 1) {
    size_t b = IX(c, i, j, k - 1);
    double hwx = 0.5 * (c.hw[IX(c, i - 1, j, k)] + c.hw[a]);
    double hwy = 0.5 * (c.hw[IX(c, i, j - 1, k)] + c.hw[a]);
    d.qu[a] = (q.u[a] - q.u[b]) / hwx;
    d.qv[a] = (q.v[a] - q.v[b]) / hwy;
  } else {
    d.qu[a] = 0.0;
    d.qv[a] = 0.0;
  }
  if (k < c.nz) d.S33[a] = (q.w[IX(c, i, j, k + 1)] - q.w[a]) / c.hc[a];
}

// pass D2: S11, S22, S12 (k < nz); S13, S23 (k = 1..nz-1, 0 on the lids)
template <class VT>
ERF_HD void diff_pass2(const VT &c, const Prim &q, const Diff &d, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  const double dx = c.dx, dy = c.dy;
  if (k < c.nz) {
    auto ZCU = [&](int ii, int jj) { return 0.5 * (c.zc[IX(c, ii - 1, jj, k)] + c.zc[IX(c, ii, jj, k)]); };
    auto ZCV = [&](int ii, int jj) { return 0.5 * (c.zc[IX(c, ii, jj - 1, k)] + c.zc[IX(c, ii, jj, k)]); };
    {
      double s = (ZCU(i + 1, j) - ZCU(i, j)) / dx;
      size_t e0 = a, e1 = IX(c, i + 1, j, k), e0u = IX(c, i, j, k + 1), e1u = IX(c, i + 1, j, k + 1);
      double m = 0.25 * (d.qu[e0] + d.qu[e1] + d.qu[e0u] + d.qu[e1u]);
      d.S11[a] = (q.u[e1] - q.u[e0]) / dx - s * m;
    }
    {
      double s = (ZCV(i, j + 1) - ZCV(i, j)) / dy;
      size_t e0 = a, e1 = IX(c, i, j + 1, k), e0u = IX(c, i, j, k + 1), e1u = IX(c, i, j + 1, k + 1);
      double m = 0.25 * (d.qv[e0] + d.qv[e1] + d.qv[e0u] + d.qv[e1u]);
      d.S22[a] = (q.v[e1] - q.v[e0]) / dy - s * m;
    }
    {  // S12 at (i-1/2, j-1/2, k)
      double sa = (ZCU(i, j) - ZCU(i, j - 1)) / dy;
      size_t e0 = IX(c, i, j - 1, k), e1 = a, e0u = IX(c, i, j - 1, k + 1), e1u = IX(c, i, j, k + 1);
      double ma = 0.25 * (d.qu[e0] + d.qu[e1] + d.qu[e0u] + d.qu[e1u]);
      double dudy = (q.u[e1] - q.u[e0]) / dy - sa * ma;
      double sb = (ZCV(i, j) - ZCV(i - 1, j)) / dx;
      size_t f0 = IX(c, i - 1, j, k), f1 = a, f0u = IX(c, i - 1, j, k + 1), f1u = e1u;
      double mb = 0.25 * (d.qv[f0] + d.qv[f1] + d.qv[f0u] + d.qv[f1u]);
      double dvdx = (q.v[f1] - q.v[f0]) / dx - sb * mb;
      d.S12[a] = 0.5 * (dudy + dvdx);
    }
  }
  if (k >= 1 && k <= c.nz - 1) {
    size_t im = IX(c, i - 1, j, k), jm = IX(c, i, j - 1, k);
    {
      double s = (c.zw[a] - c.zw[im]) / dx;
      double m = 0.25 * (d.S33[IX(c, i - 1, j, k - 1)] + d.S33[IX(c, i, j, k - 1)] + d.S33[im] + d.S33[a]);
      double dwdx = (q.w[a] - q.w[im]) / dx - s * m;
      d.S13[a] = 0.5 * (d.qu[a] + dwdx);
    }
    {
      double s = (c.zw[a] - c.zw[jm]) / dy;
      double m = 0.25 * (d.S33[IX(c, i, j - 1, k - 1)] + d.S33[IX(c, i, j, k - 1)] + d.S33[jm] + d.S33[a]);
      double dwdy = (q.w[a] - q.w[jm]) / dy - s * m;
      d.S23[a] = 0.5 * (d.qv[a] + dwdy);
    }
  } else {
    d.S13[a] = 0.0;
    d.S23[a] = 0.0;
  }
}

// pass D3: mu, K at centres (k < nz).  Smagorinsky-Lilly [R:G9]; mu_m = rho nu [R:G10]
template <class VT>
ERF_HD void diff_pass3(const VT &c, const double *rhof, const Diff &d, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  double rho = rhof[a];
  double mu = rho * c.nu, K = rho * c.alpha;
  if (c.diffusion == 2) {
    size_t a10 = IX(c, i + 1, j, k), a01 = IX(c, i, j + 1, k), a11 = IX(c, i + 1, j + 1, k);
    size_t au = IX(c, i, j, k + 1), a10u = IX(c, i + 1, j, k + 1), a01u = IX(c, i, j + 1, k + 1);
    double s12 = 0.25 * (d.S12[a] + d.S12[a10] + d.S12[a01] + d.S12[a11]);
    double s13 = 0.25 * (d.S13[a] + d.S13[a10] + d.S13[au] + d.S13[a10u]);
    double s23 = 0.25 * (d.S23[a] + d.S23[a01] + d.S23[au] + d.S23[a01u]);
    double ss = 2.0 * (d.S11[a] * d.S11[a] + d.S22[a] * d.S22[a] + d.S33[a] * d.S33[a]) +
                4.0 * (s12 * s12 + s13 * s13 + s23 * s23);
    double delta = cbrt(c.dx * c.dy * c.hc[a]);
    double mut = rho * (c.Cs * delta) * (c.Cs * delta) * sqrt(ss);
    mu += mut;
    K += mut / c.Prt;
  }
  d.mu[a] = mu;
  d.K[a] = K;
}

// pass D4: stresses tau = -2 mu sigma (Eq. 9) and the xy-edge height (k < nz; t13,t23 = 0 at k = 0, nz)
template <class VT>
ERF_HD void diff_pass4(const VT &c, const Diff &d, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  if (k >= c.nz) {
    d.t13[a] = 0.0;
    d.t23[a] = 0.0;
    return;
  }
  double div3 = (d.S11[a] + d.S22[a] + d.S33[a]) / 3.0;
  double mu = d.mu[a];
  d.t11[a] = -2.0 * mu * (d.S11[a] - div3);
  d.t22[a] = -2.0 * mu * (d.S22[a] - div3);
  d.t33[a] = -2.0 * mu * (d.S33[a] - div3);
  double mu12 = 0.25 * (d.mu[IX(c, i - 1, j - 1, k)] + d.mu[IX(c, i, j - 1, k)] + d.mu[IX(c, i - 1, j, k)] + mu);
  d.t12[a] = -2.0 * mu12 * d.S12[a];
  if (k >= 1) {
    double mu13 = 0.25 * (d.mu[IX(c, i - 1, j, k - 1)] + d.mu[IX(c, i, j, k - 1)] + d.mu[IX(c, i - 1, j, k)] + mu);
    double mu23 = 0.25 * (d.mu[IX(c, i, j - 1, k - 1)] + d.mu[IX(c, i, j, k - 1)] + d.mu[IX(c, i, j - 1, k)] + mu);
    d.t13[a] = -2.0 * mu13 * d.S13[a];
    d.t23[a] = -2.0 * mu23 * d.S23[a];
  } else {
    d.t13[a] = 0.0;
    d.t23[a] = 0.0;
  }
  d.ze12[a] = 0.25 * (c.zc[IX(c, i - 1, j - 1, k)] + c.zc[IX(c, i, j - 1, k)] + c.zc[IX(c, i - 1, j, k)] + c.zc[a]);
}

// pass D5: vertical two-point quotients of the stresses and of theta (chain rule) [R:G14]
template <class VT>
ERF_HD void diff_pass5(const VT &c, const Prim &q, const Diff &d, int i, int j, int k) {  // k<nz
  size_t a = IX(c, i, j, k);
  if (k >= 1) {
    size_t b = IX(c, i, j, k - 1);
    double hw = c.hw[a];
    d.q11[a] = (d.t11[a] - d.t11[b]) / hw;
    d.q22[a] = (d.t22[a] - d.t22[b]) / hw;
    d.qth[a] = (q.theta[a] - q.theta[b]) / hw;
    d.q12[a] = (d.t12[a] - d.t12[b]) / (d.ze12[a] - d.ze12[b]);
  } else {
    d.q11[a] = d.q22[a] = d.qth[a] = d.q12[a] = 0.0;
  }
  size_t t = IX(c, i, j, k + 1);
  double ze13a = 0.5 * (c.zw[IX(c, i - 1, j, k)] + c.zw[a]);
  double ze13t = 0.5 * (c.zw[IX(c, i - 1, j, k + 1)] + c.zw[t]);
  double ze23a = 0.5 * (c.zw[IX(c, i, j - 1, k)] + c.zw[a]);
  double ze23t = 0.5 * (c.zw[IX(c, i, j - 1, k + 1)] + c.zw[t]);
  d.q13[a] = (d.t13[t] - d.t13[a]) / (ze13t - ze13a);
  d.q23[a] = (d.t23[t] - d.t23[a]) / (ze23t - ze23a);
}

// pass D6: momentum R -= div tau; horizontal scalar fluxes Fx, Fy (k < nz)
template <class VT>
ERF_HD void diff_pass6(const VT &c, const Prim &q, const Diff &d, double *const *R, int i, int j,
                       int k) {
  size_t a = IX(c, i, j, k);
  const double dx = c.dx, dy = c.dy;
  {  // U at (i-1/2, j, k)
    double d11 = (d.t11[a] - d.t11[IX(c, i - 1, j, k)]) / dx - c.sxu[a] * avg_q_valid(c, d.q11, i - 1, j, i, j, k);
    double s12 = (d.ze12[IX(c, i, j + 1, k)] - d.ze12[a]) / dy;
    double d12 = (d.t12[IX(c, i, j + 1, k)] - d.t12[a]) / dy - s12 * avg_q_valid(c, d.q12, i, j, i, j + 1, k);
    double d13 = (d.t13[IX(c, i, j, k + 1)] - d.t13[a]) / c.hu[a];
    R[UU][a] -= d11 + d12 + d13;
  }
  {  // V at (i, j-1/2, k)
    double s12 = (d.ze12[IX(c, i + 1, j, k)] - d.ze12[a]) / dx;
    double d12 = (d.t12[IX(c, i + 1, j, k)] - d.t12[a]) / dx - s12 * avg_q_valid(c, d.q12, i, j, i + 1, j, k);
    double d22 = (d.t22[a] - d.t22[IX(c, i, j - 1, k)]) / dy - c.syv[a] * avg_q_valid(c, d.q22, i, j - 1, i, j, k);
    double d23 = (d.t23[IX(c, i, j, k + 1)] - d.t23[a]) / c.hv[a];
    R[VV][a] -= d12 + d22 + d23;
  }
  if (k >= 1) {  // W at (i, j, k-1/2)
    double zwa = c.zw[a];
    double ze_i = 0.5 * (c.zw[IX(c, i - 1, j, k)] + zwa), ze_ip = 0.5 * (zwa + c.zw[IX(c, i + 1, j, k)]);
    double ze_j = 0.5 * (c.zw[IX(c, i, j - 1, k)] + zwa), ze_jp = 0.5 * (zwa + c.zw[IX(c, i, j + 1, k)]);
    double m13 = 0.25 * (d.q13[IX(c, i, j, k - 1)] + d.q13[IX(c, i + 1, j, k - 1)] + d.q13[a] + d.q13[IX(c, i + 1, j, k)]);
    double m23 = 0.25 * (d.q23[IX(c, i, j, k - 1)] + d.q23[IX(c, i, j + 1, k - 1)] + d.q23[a] + d.q23[IX(c, i, j + 1, k)]);
    double d13 = (d.t13[IX(c, i + 1, j, k)] - d.t13[a]) / dx - (ze_ip - ze_i) / dx * m13;
    double d23 = (d.t23[IX(c, i, j + 1, k)] - d.t23[a]) / dy - (ze_jp - ze_j) / dy * m23;
    double d33 = (d.t33[a] - d.t33[IX(c, i, j, k - 1)]) / c.hw[a];
    R[WW][a] -= d13 + d23 + d33;
  }
  // scalar fluxes (conservative form) [R:G17]
  double Kx = 0.5 * (d.K[IX(c, i - 1, j, k)] + d.K[a]);
  double Ky = 0.5 * (d.K[IX(c, i, j - 1, k)] + d.K[a]);
  double dthx = (q.theta[a] - q.theta[IX(c, i - 1, j, k)]) / dx - c.sxu[a] * avg_q_valid(c, d.qth, i - 1, j, i, j, k);
  double dthy = (q.theta[a] - q.theta[IX(c, i, j - 1, k)]) / dy - c.syv[a] * avg_q_valid(c, d.qth, i, j - 1, i, j, k);
  d.Fx[a] = -Kx * dthx;
  d.Fy[a] = -Ky * dthy;
}

// pass D7: contravariant vertical scalar flux at w-faces, k = 0..nz (0 on lids)
template <class VT>
ERF_HD void diff_pass7(const VT &c, const Diff &d, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  if (k < 1 || k > c.nz - 1) {
    d.Fz[a] = 0.0;
    return;
  }
  double Kw = 0.5 * (d.K[IX(c, i, j, k - 1)] + d.K[a]);
  double fz = -Kw * d.qth[a];
  double fxb = 0.25 * (d.Fx[IX(c, i, j, k - 1)] + d.Fx[IX(c, i + 1, j, k - 1)] + d.Fx[a] + d.Fx[IX(c, i + 1, j, k)]);
  double fyb = 0.25 * (d.Fy[IX(c, i, j, k - 1)] + d.Fy[IX(c, i, j + 1, k - 1)] + d.Fy[a] + d.Fy[IX(c, i, j + 1, k)]);
  d.Fz[a] = fz - c.sxw[a] * fxb - c.syw[a] * fyb;
}

// pass D8: R_Theta -= div F (k < nz)
template <class VT>
ERF_HD void diff_pass8(const VT &c, const Diff &d, double *const *R, int i, int j, int k) {
  size_t a = IX(c, i, j, k), ip = IX(c, i + 1, j, k), jp = IX(c, i, j + 1, k), kp = IX(c, i, j, k + 1);
  R[TH][a] -= ((c.hx[ip] * d.Fx[ip] - c.hx[a] * d.Fx[a]) / c.dx + (c.hy[jp] * d.Fy[jp] - c.hy[a] * d.Fy[a]) / c.dy +
               (d.Fz[kp] - d.Fz[a])) / c.hc[a];
}

// ---------------------------------------------------------------- pressure gradient, buoyancy (S4)
template <class VT>
ERF_HD double dz_centre(const VT &c, const double *f, int i, int j, int k) {
  int kb = k > 0 ? k - 1 : 0;
  int kt = k < c.nz - 1 ? k + 1 : c.nz - 1;
  return (f[IX(c, i, j, kt)] - f[IX(c, i, j, kb)]) / (c.zc[IX(c, i, j, kt)] - c.zc[IX(c, i, j, kb)]);
}
template <class VT>
ERF_HD double grad_x(const VT &c, const double *f, int i, int j, int k) {
  double along = (f[IX(c, i, j, k)] - f[IX(c, i - 1, j, k)]) / c.dx;
  if (c.nz == 1 || c.flat) return along;
  return along - c.sxu[IX(c, i, j, k)] * 0.5 * (dz_centre(c, f, i - 1, j, k) + dz_centre(c, f, i, j, k));
}
template <class VT>
ERF_HD double grad_y(const VT &c, const double *f, int i, int j, int k) {
  double along = (f[IX(c, i, j, k)] - f[IX(c, i, j - 1, k)]) / c.dy;
  if (c.nz == 1 || c.flat) return along;
  return along - c.syv[IX(c, i, j, k)] * 0.5 * (dz_centre(c, f, i, j - 1, k) + dz_centre(c, f, i, j, k));
}

template <class VT>
ERF_HD void pgbuoy_cell(const VT &c, const double *const *S, const Prim &q, double *const *R, int i,
                        int j, int k) {  // k < nz
  size_t a = IX(c, i, j, k);
  R[UU][a] -= grad_x(c, q.pp, i, j, k);
  R[VV][a] -= grad_y(c, q.pp, i, j, k);
  if (k >= 1) {
    size_t b = IX(c, i, j, k - 1);
    double rpa = S[RHO][a] - c.rho0[a], rpb = S[RHO][b] - c.rho0[b];
    R[WW][a] -= (q.pp[a] - q.pp[b]) / c.hw[a] + c.g * 0.5 * (rpb + rpa);
  }
}

// anelastic pair (Sec. 2.2): -grad of the projection's lagged p' and B = rho0 (theta - theta0)/theta0 g at w-faces
template <class VT>
ERF_HD void anel_pgbuoy_cell(const VT &c, const Prim &q, const double *pan, double *const *R, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  R[UU][a] -= grad_x(c, pan, i, j, k);
  R[VV][a] -= grad_y(c, pan, i, j, k);
  if (k >= 1) {
    size_t b = IX(c, i, j, k - 1);
    double th0a = c.Th0[a] / c.rho0[a], th0b = c.Th0[b] / c.rho0[b];
    double Ba = c.rho0[a] * (q.theta[a] - th0a) / th0a, Bb = c.rho0[b] * (q.theta[b] - th0b) / th0b;
    R[WW][a] += -(pan[a] - pan[b]) / c.hw[a] + c.g * 0.5 * (Bb + Ba);
  }
}

// ---------------------------------------------------------------- Rayleigh damping layer (L219, L622) [R:G28]
// tau(z) = ray_coef sin^2((pi/2)(z - z_b)/ray_depth) above z_b = z_top - ray_depth (L622: sine-squared ramp from 0 at
// the bottom of the layer to the stated inverse time scale at the top)
ERF_HD double rayleigh_tau(double depth, double coef, double z, double ztop) {
  const double zb = ztop - depth;
  if (z <= zb) return 0.0;
  const double s = sin(0.5 * 3.14159265358979323846 * (z - zb) / depth);
  return coef * s * s;
}

// relaxation of the masked primitives towards their references (u_ref, v_ref, 0, theta0), k < nz
template <class VT>
ERF_HD void rayleigh_cell(const VT &c, const double *const *S, double *const *R, int i, int j, int k) {
  const int nz = c.nz, f = c.ray_fields;
  const size_t a = IX(c, i, j, k), t = IX(c, i, j, nz);
  if (f & 1) {
    const size_t im = IX(c, i - 1, j, k), tim = IX(c, i - 1, j, nz);
    const double tau = rayleigh_tau(c.ray_depth, c.ray_coef, 0.5 * (c.zc[im] + c.zc[a]), 0.5 * (c.zw[tim] + c.zw[t]));
    R[UU][a] -= tau * (S[UU][a] - 0.5 * (S[RHO][im] + S[RHO][a]) * c.ray_uref);
  }
  if (f & 2) {
    const size_t jm = IX(c, i, j - 1, k), tjm = IX(c, i, j - 1, nz);
    const double tau = rayleigh_tau(c.ray_depth, c.ray_coef, 0.5 * (c.zc[jm] + c.zc[a]), 0.5 * (c.zw[tjm] + c.zw[t]));
    R[VV][a] -= tau * (S[VV][a] - 0.5 * (S[RHO][jm] + S[RHO][a]) * c.ray_vref);
  }
  if ((f & 4) && k >= 1) R[WW][a] -= rayleigh_tau(c.ray_depth, c.ray_coef, c.zw[a], c.zw[t]) * S[WW][a];
  if (f & 8)
    R[TH][a] -= rayleigh_tau(c.ray_depth, c.ray_coef, c.zc[a], c.zw[t]) * (S[TH][a] - S[RHO][a] * c.Th0[a] / c.rho0[a]);
}

// ---------------------------------------------------------------- acoustic substeps (S5)
struct Acou {
  const double *theta_t, *pi_t, *Th_t;  // stage constants
  const double *R[5];                   // slow tendencies
  double *P[5];                         // S''
  double *Om;                           // Omega'' at the end of the previous substep
  double *Th_prev, *Thd;                // divergence damping (L144) [R:G6]
  double *om;                           // explicit slope part of W''
  double *Ttil, *rtil, *cpr, *dpr;      // column scratch
  double *Usum, *Vsum, *Omsum;          // sums of the momenta that advance rho'' (L138), for the scalars; may be null
};

// step 1: Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev); prev <- Theta''
template <class VT>
ERF_HD void ac_damp(const VT &c, const Acou &A, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  double T = A.P[TH][a];
  A.Thd[a] = T + c.beta_d * (T - A.Th_prev[a]);
  A.Th_prev[a] = T;
}

// step 2: explicit horizontal momenta (L585 rows 1-2)
template <class VT>
ERF_HD void ac_horiz(const VT &c, const Acou &A, double dtau, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  double gR = c.gam * c.Rd;
  double piu = 0.5 * (A.pi_t[IX(c, i - 1, j, k)] + A.pi_t[a]);
  double piv = 0.5 * (A.pi_t[IX(c, i, j - 1, k)] + A.pi_t[a]);
  const double Un = A.P[UU][a] + dtau * (-gR * piu * grad_x(c, A.Thd, i, j, k) + A.R[UU][a]);
  const double Vn = A.P[VV][a] + dtau * (-gR * piv * grad_y(c, A.Thd, i, j, k) + A.R[VV][a]);
  A.P[UU][a] = Un;
  A.P[VV][a] = Vn;
  if (A.Usum) {  // the horizontal momenta of this substep's continuity equation
    A.Usum[a] += Un;
    A.Vsum[a] += Vn;
  }
}

// step 3: omega = sxw avg4(U''new) + syw avg4(V''new), k = 1..nz-1 [R:G16]
template <class VT>
ERF_HD void ac_slope(const VT &c, const Acou &A, int i, int j, int k) {
  size_t a = IX(c, i, j, k);
  if (k < 1 || k > c.nz - 1) {
    A.om[a] = 0.0;
    return;
  }
  const double *U = A.P[UU], *V = A.P[VV];
  double ubar = 0.25 * (U[IX(c, i, j, k - 1)] + U[IX(c, i + 1, j, k - 1)] + U[a] + U[IX(c, i + 1, j, k)]);
  double vbar = 0.25 * (V[IX(c, i, j, k - 1)] + V[IX(c, i, j + 1, k - 1)] + V[a] + V[IX(c, i, j + 1, k)]);
  A.om[a] = c.sxw[a] * ubar + c.syw[a] * vbar;
}

// steps 4-6: one column.  Forward sweep builds the explicit parts, the rows of the
// tridiagonal system for Omega''new (L144; S5) and eliminates; backward sweep
// substitutes and updates W'', Theta'', rho'' (L585 rows 3-5, L591).
template <class VT>
ERF_HD void ac_column(const VT &c, const Acou &A, double dtau, int i, int j) {
  const int nz = c.nz;
  const double b1 = 0.5 * (1.0 - c.beta_s), b2 = 0.5 * (1.0 + c.beta_s);  // L589
  const double g = c.g, gR = c.gam * c.Rd;
  const double s = dtau * dtau * b2 * b2;
  const double *U = A.P[UU], *V = A.P[VV];
  double That_m = 0.0, rhat_m = 0.0, cp_m = 0.0, dp_m = 0.0;
  for (int k = 0; k < nz; k++) {
    size_t a = IX(c, i, j, k), ip = IX(c, i + 1, j, k), jp = IX(c, i, j + 1, k);
    size_t im = IX(c, i - 1, j, k), jm = IX(c, i, j - 1, k), kp = IX(c, i, j, k + 1);
    double th = A.theta_t[a];
    double thx_m = 0.5 * (A.theta_t[im] + th), thx_p = 0.5 * (th + A.theta_t[ip]);
    double thy_m = 0.5 * (A.theta_t[jm] + th), thy_p = 0.5 * (th + A.theta_t[jp]);
    double hc = c.hc[a];
    double fxp = c.hx[ip] * U[ip], fxm = c.hx[a] * U[a];
    double fyp = c.hy[jp] * V[jp], fym = c.hy[a] * V[a];
    double DhT = (fxp * thx_p - fxm * thx_m) / c.dx / hc + (fyp * thy_p - fym * thy_m) / c.dy / hc;
    double Dh = (fxp - fxm) / c.dx / hc + (fyp - fym) / c.dy / hc;
    double thf_b = (k >= 1) ? 0.5 * (A.theta_t[IX(c, i, j, k - 1)] + th) : 0.0;
    double thf_t = (k + 1 <= nz - 1) ? 0.5 * (th + A.theta_t[kp]) : 0.0;
    double om_b = A.Om[a], om_t = A.Om[kp];
    double Tpp = A.P[TH][a], rpp = A.P[RHO][a];
    double Ttil = Tpp + dtau * (A.R[TH][a] - DhT - b1 * (thf_t * om_t - thf_b * om_b) / hc);
    double rtil = rpp + dtau * (A.R[RHO][a] - Dh - b1 * (om_t - om_b) / hc);
    double That = b2 * Ttil + b1 * Tpp, rhat = b2 * rtil + b1 * rpp;
    A.Ttil[a] = Ttil;
    A.rtil[a] = rtil;
    if (k >= 1) {
      size_t b = IX(c, i, j, k - 1);
      double pif = 0.5 * (A.pi_t[b] + A.pi_t[a]);
      double pi0f = 0.5 * (c.pi0[b] + c.pi0[a]);
      double rho0f = 0.5 * (c.rho0[b] + c.rho0[a]);
      double Bf = rho0f * c.rdocv * pif / pi0f;
      double thf_kp = thf_t;
      double thf_km = (k - 1 >= 1) ? 0.5 * (A.theta_t[IX(c, i, j, k - 2)] + A.theta_t[b]) : 0.0;
      double hw = c.hw[a], hcm = c.hc[b];
      double Tk = A.Th_t[a], Tm = A.Th_t[b];
      double Cc = -s * gR * pif * thf_kp / (hw * hc) + s * g * Bf * thf_kp / (2.0 * hc * Tk) - s * g / (2.0 * hc);
      double Ac = -s * gR * pif * thf_km / (hw * hcm) - s * g * Bf * thf_km / (2.0 * hcm * Tm) + s * g / (2.0 * hcm);
      double Dc = 1.0 + s * gR * pif * thf_b * (1.0 / hc + 1.0 / hcm) / hw -
                  s * g * Bf * thf_b / 2.0 * (1.0 / (hc * Tk) - 1.0 / (hcm * Tm)) + s * g / 2.0 * (1.0 / hc - 1.0 / hcm);
      if (k == nz - 1) Cc = 0.0;
      if (k == 1) Ac = 0.0;
      double rhs = A.P[WW][a] +
                   dtau * (A.R[WW][a] - gR * pif * (That - That_m) / hw + g * Bf * 0.5 * (That / Tk + That_m / Tm) -
                           g * 0.5 * (rhat + rhat_m)) -
                   A.om[a];
      double m = Dc - Ac * cp_m;  // Thomas forward elimination (cp_m = dp_m = 0 at k = 1)
      cp_m = Cc / m;
      dp_m = (rhs - Ac * dp_m) / m;
      A.cpr[a] = cp_m;
      A.dpr[a] = dp_m;
    }
    That_m = That;
    rhat_m = rhat;
  }
  // backward sweep
  double On_t = 0.0;  // Omega_{k+1}, starting from the lid Omega_nz = 0
  for (int k = nz - 1; k >= 0; k--) {
    size_t a = IX(c, i, j, k);
    double On_b = 0.0;
    if (k >= 1) {
      On_b = A.dpr[a] - A.cpr[a] * On_t;
      A.P[WW][a] = On_b + A.om[a];
      if (A.Omsum) A.Omsum[a] += b2 * On_b + b1 * A.Om[a];  // the vertical flux that advanced rho'' (L591)
    }
    double th = A.theta_t[a];
    double thf_b = (k >= 1) ? 0.5 * (A.theta_t[IX(c, i, j, k - 1)] + th) : 0.0;
    double thf_t = (k + 1 <= nz - 1) ? 0.5 * (th + A.theta_t[IX(c, i, j, k + 1)]) : 0.0;
    double hc = c.hc[a];
    A.P[TH][a] = A.Ttil[a] - dtau * b2 * (thf_t * On_t - thf_b * On_b) / hc;
    A.P[RHO][a] = A.rtil[a] - dtau * b2 * (On_t - On_b) / hc;
    A.Om[IX(c, i, j, k + 1)] = On_t;
    On_t = On_b;
  }
  A.Om[IX(c, i, j, 0)] = 0.0;
}

}  // namespace gen
}  // namespace erfb
