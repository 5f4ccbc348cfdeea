// k_fused_slow.cu -- the slow right-hand side f(S) of PAPER.md Eq. 1-3 on flat grids.
//
// Four kernels per evaluation:
//   k_prim_flat   S -> theta, u, v, w, p', pi^t, 1/Theta^t        (Eq. 7; L196)
//   k_visc_flat   u, v, w, rho -> mu, K                            (Eq. 9; Smagorinsky [R:G9])
//   k_adv_flat    advection (Eq. 17-21) + pressure gradient + buoyancy (L84) -> R
//   k_diff_flat   R -= div(tau), R_Theta -= div(F)                 (Eq. 2-3, Eq. 9)
// k_adv_flat and k_diff_flat give one thread a whole (i,j) column and march upward in k: the
// vertical stencil lives in a register window (one new level loaded per step), vertical face
// fluxes are computed once and carried from a cell to the one above, and the horizontal
// neighbours are read through L1 (a warp's shifted 256-B rows share lines).
// On a flat grid all metric terms are per-level constants (tables), Omega = W, and every
// horizontal slope term of D0 vanishes identically.
#include "slow_flat.cuh"

namespace erfb {

// ------------------------------------------------------------------ primitives
__global__ void __launch_bounds__(256) k_prim_flat(const SlowFlat p) {
  const size_t plane = (size_t)p.nx * p.ny;
  const size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= plane * (p.nz + 1)) return;
  const int k = (int)(a / plane);
  const size_t r = a - (size_t)k * plane;
  const int j = (int)(r / p.nx), i = (int)(r - (size_t)j * p.nx);
  const double *__restrict__ rho = p.rho;
  if (k < p.nz) {
    const double rc = rho[a], Th = p.Th[a];
    const int im = i == 0 ? p.nx - 1 : i - 1, jm = j == 0 ? p.ny - 1 : j - 1;
    const size_t kk = (size_t)k * plane;
    p.theta[a] = Th / rc;
    // x = Theta/Theta0 - 1.  gamma = 1 + Rd/cv, so with e = (1+x)^(Rd/cv) - 1 = expm1((Rd/cv) log1p(x)):
    //   pi = pi0 (1 + e)                     pi = pi0 (Theta/Theta0)^(Rd/cv)
    //   p' = p0 [(1+x)(1+e) - 1] = p0 (x + e + x e)   p' = p0 [(Theta/Theta0)^gamma - 1]   [R:S1]
    // one log1p and one expm1 per cell, no cancellation (x, e are small and enter linearly)
    const double x = (Th - p.Th0[k]) * p.rTh0[k];
    const double e = expm1(p.rdocv * log1p(x));
    p.pp[a] = p.p0[k] * (x + e + x * e);
    p.pi[a] = p.pi0[k] * (1.0 + e);
    p.iT[a] = 1.0 / Th;
    p.u[a] = p.U[a] / (0.5 * (rho[kk + (size_t)j * p.nx + im] + rc));
    p.v[a] = p.V[a] / (0.5 * (rho[kk + (size_t)jm * p.nx + i] + rc));
    const double rw = k == 0 ? rc : 0.5 * (rho[a - plane] + rc);
    p.w[a] = p.W[a] / rw;
  } else {
    p.w[a] = p.W[a] / rho[a - plane];
  }
}

// ------------------------------------------------------------------ viscosity
// mu = rho nu + mu_t, K = rho alpha + mu_t / Pr_t; mu_t = rho (Cs Delta)^2 |S| [R:G9,G10]
__global__ void __launch_bounds__(256) k_visc_flat(const SlowFlat p) {
  const size_t plane = (size_t)p.nx * p.ny;
  const size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= plane * p.nz) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int k = (int)(a / plane);
  const size_t r = a - (size_t)k * plane;
  const int j = (int)(r / nx), i = (int)(r - (size_t)j * nx);
  const double rc = p.rho[a];
  double mu = rc * p.nu, K = rc * p.alpha;
  if (p.diffusion == 2) {
    const double *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w;
    const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
    const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
    const size_t kk = (size_t)k * plane;
    auto at = [&](int ii, int jj) { return kk + (size_t)jj * nx + ii; };
    const double rdx = p.rdx, rdy = p.rdy;
    const double u_c = u[a], u_p = u[at(ip, j)], v_c = v[a], v_p = v[at(i, jp)];
    const double S11 = (u_p - u_c) * rdx, S22 = (v_p - v_c) * rdy;
    const double w_c = w[a], w_t = w[a + plane];
    const double S33 = (w_t - w_c) * p.rdz[k];
    // S12 at the four xy-edges around the centre
    const double u_jm = u[at(i, jm)], u_jp = u[at(i, jp)], u_pjm = u[at(ip, jm)], u_pjp = u[at(ip, jp)];
    const double v_im = v[at(im, j)], v_ip = v[at(ip, j)], v_imp = v[at(im, jp)], v_ipp = v[at(ip, jp)];
    const double e00 = 0.5 * ((u_c - u_jm) * rdy + (v_c - v_im) * rdx);
    const double e10 = 0.5 * ((u_p - u_pjm) * rdy + (v_ip - v_c) * rdx);
    const double e01 = 0.5 * ((u_jp - u_c) * rdy + (v_p - v_imp) * rdx);
    const double e11 = 0.5 * ((u_pjp - u_p) * rdy + (v_ipp - v_p) * rdx);
    const double s12 = 0.25 * (e00 + e10 + e01 + e11);
    // S13 at (i,k), (i+1,k), (i,k+1), (i+1,k+1); S23 likewise; zero on the lids
    double s13 = 0.0, s23 = 0.0;
    const double w_im = w[at(im, j)], w_ip = w[at(ip, j)], w_jm = w[at(i, jm)], w_jp = w[at(i, jp)];
    if (k >= 1) {
      const double rhw = p.rhw[k];
      s13 += 0.5 * ((u_c - u[a - plane]) * rhw + (w_c - w_im) * rdx) +
             0.5 * ((u_p - u[at(ip, j) - plane]) * rhw + (w_ip - w_c) * rdx);
      s23 += 0.5 * ((v_c - v[a - plane]) * rhw + (w_c - w_jm) * rdy) +
             0.5 * ((v_p - v[at(i, jp) - plane]) * rhw + (w_jp - w_c) * rdy);
    }
    if (k + 1 <= nz - 1) {
      const double rhw = p.rhw[k + 1];
      const double wt_im = w[at(im, j) + plane], wt_ip = w[at(ip, j) + plane];
      const double wt_jm = w[at(i, jm) + plane], wt_jp = w[at(i, jp) + plane];
      s13 += 0.5 * ((u[a + plane] - u_c) * rhw + (w_t - wt_im) * rdx) +
             0.5 * ((u[at(ip, j) + plane] - u_p) * rhw + (wt_ip - w_t) * rdx);
      s23 += 0.5 * ((v[a + plane] - v_c) * rhw + (w_t - wt_jm) * rdy) +
             0.5 * ((v[at(i, jp) + plane] - v_p) * rhw + (wt_jp - w_t) * rdy);
    }
    s13 *= 0.25;
    s23 *= 0.25;
    const double ss = 2.0 * (S11 * S11 + S22 * S22 + S33 * S33) + 4.0 * (s12 * s12 + s13 * s13 + s23 * s23);
    const double mut = rc * p.csd2[k] * sqrt(ss);
    mu += mut;
    K += mut * p.rPrt;
  }
  p.mu[a] = mu;
  p.K[a] = K;
}

// ------------------------------------------------------------------ advection + PG + buoyancy
template <int OH>
__global__ void __launch_bounds__(128) k_adv_flat(const SlowFlat p) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i >= p.nx || j >= p.ny) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz, ov = p.ov;
  const size_t plane = (size_t)nx * ny;
  constexpr int HW = (OH + 1) / 2;  // half width of the horizontal stencil
  // wrapped neighbour columns i-3..i+3 (row j) and rows j-3..j+3 (column i)
  int ox[7], oy[7];
#pragma unroll
  for (int n = 0; n < 7; n++) {
    int ii = i + n - 3, jj = j + n - 3;
    while (ii < 0) ii += nx;
    while (ii >= nx) ii -= nx;
    while (jj < 0) jj += ny;
    while (jj >= ny) jj -= ny;
    ox[n] = j * nx + ii;
    oy[n] = jj * nx + i;
  }
  const int o_xm_yp = (oy[4] - i) + (ox[2] - j * nx);  // (i-1, j+1)
  const int o_xp_ym = (oy[2] - i) + (ox[4] - j * nx);  // (i+1, j-1)
  const int oc = ox[3];
  const double *__restrict__ U = p.U, *__restrict__ V = p.V, *__restrict__ W = p.W, *__restrict__ rho = p.rho;
  const double *__restrict__ th = p.theta, *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w;
  const double *__restrict__ pp = p.pp;
  double *__restrict__ Rrho = p.Rrho, *__restrict__ RU = p.RU, *__restrict__ RV = p.RV;
  double *__restrict__ RW = p.RW, *__restrict__ RTh = p.RTh;
  const double rdx = p.rdx, rdy = p.rdy;

  // vertical register windows: cells k-3..k+2 (theta,u,v), faces k-2..k+3 (w)
  double wt[6], wu[6], wv[6], ww[6];
#pragma unroll
  for (int n = 0; n < 6; n++) {
    const int kc = n - 3, kf = n - 2;
    const bool okc = kc >= 0 && kc < nz, okf = kf >= 0 && kf <= nz;
    const size_t ac = (size_t)(okc ? kc : 0) * plane + oc, af = (size_t)(okf ? kf : 0) * plane + oc;
    wt[n] = okc ? th[ac] : 0.0;
    wu[n] = okc ? u[ac] : 0.0;
    wv[n] = okc ? v[ac] : 0.0;
    ww[n] = okf ? w[af] : 0.0;
  }
  double fT_b = 0.0, fU_b = 0.0, fV_b = 0.0, om_b = 0.0;  // face fluxes at the bottom of the previous cell
  double HT = 0.0, HU = 0.0, HV = 0.0, Hr = 0.0;          // horizontal parts of the previous cell
  double Gz_m = 0.0;                                      // w flux at centre k-1
  double U_cm = 0.0, U_pm = 0.0, V_cm = 0.0, V_pm = 0.0;  // dz*U(i), dz*U(i+1), dz*V(j), dz*V(j+1) at level k-1
  double pp_m = 0.0, rp_m = 0.0;                          // p', rho' at level k-1
  double om_c = 0.0;                                      // Omega at face k (lid: 0)

#pragma unroll 1
  for (int k = 0; k <= nz; k++) {
    const size_t kk = (size_t)k * plane;
    // ---- face k: vertical fluxes of theta, u, v (zero on the lids)
    double fT = 0.0, fU = 0.0, fV = 0.0;
    const bool inner = k >= 1 && k <= nz - 1;
    if (inner) {
      const int ord = vorder(ov, min(k, nz - k));
      const double om_xm = W[kk + ox[2]], om_ym = W[kk + oy[2]];
      fT = flux_rt(ord, om_c, wt);
      fU = flux_rt(ord, 0.5 * (om_xm + om_c), wu);
      fV = flux_rt(ord, 0.5 * (om_ym + om_c), wv);
    }
    // ---- finish cell k-1
    if (k >= 1) {
      const size_t am = kk - plane + oc;
      const double rdzm = p.rdz[k - 1];
      Rrho[am] = -(Hr + (om_c - om_b) * rdzm);
      RTh[am] = -(HT + (fT - fT_b) * rdzm);
      RU[am] = -(HU + (fU - fU_b) * rdzm);
      RV[am] = -(HV + (fV - fV_b) * rdzm);
    }
    if (k == nz) {
      RW[kk + oc] = 0.0;
      break;
    }
    fT_b = fT; fU_b = fU; fV_b = fV; om_b = om_c;
    // ---- cell k: horizontal flux divergences
    const double U_m1 = U[kk + ox[2]], U_c = U[kk + oc], U_p1 = U[kk + ox[4]];
    const double U_ym = U[kk + oy[2]], U_pym = U[kk + o_xp_ym];
    const double V_m1 = V[kk + oy[2]], V_c = V[kk + oc], V_p1 = V[kk + oy[4]];
    const double V_xm = V[kk + ox[2]], V_xmp = V[kk + o_xm_yp];
    double tx[7], ty[7], ux[7], uy[7], vx[7], vy[7], wx[7], wy[7];
#pragma unroll
    for (int n = 0; n < 7; n++) {
      const bool need = (n >= 3 - HW && n <= 3 + HW) && n != 3;
      tx[n] = need ? th[kk + ox[n]] : 0.0;
      ty[n] = need ? th[kk + oy[n]] : 0.0;
      ux[n] = need ? u[kk + ox[n]] : 0.0;
      uy[n] = need ? u[kk + oy[n]] : 0.0;
      vx[n] = need ? v[kk + ox[n]] : 0.0;
      vy[n] = need ? v[kk + oy[n]] : 0.0;
      wx[n] = need ? w[kk + ox[n]] : 0.0;
      wy[n] = need ? w[kk + oy[n]] : 0.0;
    }
    tx[3] = ty[3] = wt[3];
    ux[3] = uy[3] = wu[3];
    vx[3] = vy[3] = wv[3];
    wx[3] = wy[3] = ww[2];  // w at face k
    Hr = (U_p1 - U_c) * rdx + (V_p1 - V_c) * rdy;
    HT = (flux_c<OH>(U_p1, tx[1], tx[2], tx[3], tx[4], tx[5], tx[6]) - flux_c<OH>(U_c, tx[0], tx[1], tx[2], tx[3], tx[4], tx[5])) * rdx +
         (flux_c<OH>(V_p1, ty[1], ty[2], ty[3], ty[4], ty[5], ty[6]) - flux_c<OH>(V_c, ty[0], ty[1], ty[2], ty[3], ty[4], ty[5])) * rdy;
    const double pp_c = pp[kk + oc];
    HU = (flux_c<OH>(0.5 * (U_c + U_p1), ux[1], ux[2], ux[3], ux[4], ux[5], ux[6]) -
          flux_c<OH>(0.5 * (U_m1 + U_c), ux[0], ux[1], ux[2], ux[3], ux[4], ux[5])) * rdx +
         (flux_c<OH>(0.5 * (V_xmp + V_p1), uy[1], uy[2], uy[3], uy[4], uy[5], uy[6]) -
          flux_c<OH>(0.5 * (V_xm + V_c), uy[0], uy[1], uy[2], uy[3], uy[4], uy[5])) * rdy +
         (pp_c - pp[kk + ox[2]]) * rdx;
    HV = (flux_c<OH>(0.5 * (U_pym + U_p1), vx[1], vx[2], vx[3], vx[4], vx[5], vx[6]) -
          flux_c<OH>(0.5 * (U_ym + U_c), vx[0], vx[1], vx[2], vx[3], vx[4], vx[5])) * rdx +
         (flux_c<OH>(0.5 * (V_c + V_p1), vy[1], vy[2], vy[3], vy[4], vy[5], vy[6]) -
          flux_c<OH>(0.5 * (V_m1 + V_c), vy[0], vy[1], vy[2], vy[3], vy[4], vy[5])) * rdy +
         (pp_c - pp[kk + oy[2]]) * rdy;
    // ---- w equation at face k; vertical flux at centre k
    const double om_t = (k + 1 <= nz - 1) ? W[kk + plane + oc] : 0.0;
    const double Gz = flux_rt(vorder(ov, min(k + 1, nz - k)), 0.5 * (om_c + om_t), ww);
    const double dzk = p.dz[k];
    const double U_cd = dzk * U_c, U_pd = dzk * U_p1, V_cd = dzk * V_c, V_pd = dzk * V_p1;
    const double rp_c = rho[kk + oc] - p.rho0[k];
    if (k >= 1) {
      const double rhw = p.rhw[k];
      const double adv =
          (flux_c<OH>(0.5 * (U_pm + U_pd), wx[1], wx[2], wx[3], wx[4], wx[5], wx[6]) -
           flux_c<OH>(0.5 * (U_cm + U_cd), wx[0], wx[1], wx[2], wx[3], wx[4], wx[5])) * rdx +
          (flux_c<OH>(0.5 * (V_pm + V_pd), wy[1], wy[2], wy[3], wy[4], wy[5], wy[6]) -
           flux_c<OH>(0.5 * (V_cm + V_cd), wy[0], wy[1], wy[2], wy[3], wy[4], wy[5])) * rdy +
          (Gz - Gz_m);
      RW[kk + oc] = -adv * rhw - ((pp_c - pp_m) * rhw + p.g * 0.5 * (rp_m + rp_c));
    } else {
      RW[kk + oc] = 0.0;
    }
    Gz_m = Gz;
    U_cm = U_cd; U_pm = U_pd; V_cm = V_cd; V_pm = V_pd;
    pp_m = pp_c; rp_m = rp_c;
    om_c = om_t;
    // ---- shift the vertical windows: bring in cell k+3 and face k+4
#pragma unroll
    for (int n = 0; n < 5; n++) {
      wt[n] = wt[n + 1]; wu[n] = wu[n + 1]; wv[n] = wv[n + 1]; ww[n] = ww[n + 1];
    }
    {
      const int kc = k + 3, kf = k + 4;
      const bool okc = kc < nz, okf = kf <= nz;
      const size_t ac = (size_t)(okc ? kc : 0) * plane + oc, af = (size_t)(okf ? kf : 0) * plane + oc;
      wt[5] = okc ? th[ac] : 0.0;
      wu[5] = okc ? u[ac] : 0.0;
      wv[5] = okc ? v[ac] : 0.0;
      ww[5] = okf ? w[af] : 0.0;
    }
  }
}

// ------------------------------------------------------------------ diffusion
// R_U,V,W -= div(tau), tau = -2 mu (S - 1/3 div u I) (Eq. 9); R_Theta -= div(-K grad theta) (Eq. 3);
// free-slip lids: tau13 = tau23 = 0 and no scalar flux at k = 0, nz (Table C1 "Slip Wall").
__global__ void __launch_bounds__(128) k_diff_flat(const SlowFlat p) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i >= p.nx || j >= p.ny) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const size_t plane = (size_t)nx * ny;
  const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const int c = j * nx + i, xm = j * nx + im, xp = j * nx + ip, ym = jm * nx + i, yp = jp * nx + i;
  const int xmym = jm * nx + im, xpym = jm * nx + ip, xmyp = jp * nx + im;
  const double *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w, *__restrict__ th = p.theta;
  const double *__restrict__ mu = p.mu, *__restrict__ Kf = p.K;
  double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW, *__restrict__ RTh = p.RTh;
  const double rdx = p.rdx, rdy = p.rdy;

  // carried from level k-1 / face k
  double u_cm = 0, u_pm = 0, v_cm = 0, v_pm = 0;                  // u(i), u(i+1), v(j), v(j+1) at k-1
  double mu_cm = 0, mu_xmm = 0, mu_xpm = 0, mu_ymm = 0, mu_ypm = 0;  // mu at k-1: c, xm, xp, ym, yp
  double K_m = 0, th_m = 0, t33_m = 0;
  double t13_b = 0, t23_b = 0, Fz_b = 0;  // face k-1 ... (bottom face of the previous cell)
  double HU = 0, HV = 0, HT = 0;
  // w at face k: c, xm, xp, ym, yp
  double w_c = w[c], w_xm = w[xm], w_xp = w[xp], w_ym = w[ym], w_yp = w[yp];

#pragma unroll 1
  for (int k = 0; k <= nz; k++) {
    const size_t kk = (size_t)k * plane;
    const bool cell = k < nz, inner = k >= 1 && k <= nz - 1;
    double u_c = 0, u_p = 0, v_c = 0, v_p = 0, mu_c = 0, mu_xm = 0, mu_xp = 0, mu_ym = 0, mu_yp = 0, K_c = 0, th_c = 0;
    if (cell) {
      u_c = u[kk + c]; u_p = u[kk + xp]; v_c = v[kk + c]; v_p = v[kk + yp];
      mu_c = mu[kk + c]; mu_xm = mu[kk + xm]; mu_xp = mu[kk + xp]; mu_ym = mu[kk + ym]; mu_yp = mu[kk + yp];
      K_c = Kf[kk + c]; th_c = th[kk + c];
    }
    // ---- face k: tau13 at (i,k) and (i+1,k), tau23 at (j,k) and (j+1,k), vertical scalar flux
    double t13 = 0, t13p = 0, t23 = 0, t23p = 0, Fz = 0;
    if (inner) {
      const double rhw = p.rhw[k];
      const double S13 = 0.5 * ((u_c - u_cm) * rhw + (w_c - w_xm) * rdx);
      const double S13p = 0.5 * ((u_p - u_pm) * rhw + (w_xp - w_c) * rdx);
      const double S23 = 0.5 * ((v_c - v_cm) * rhw + (w_c - w_ym) * rdy);
      const double S23p = 0.5 * ((v_p - v_pm) * rhw + (w_yp - w_c) * rdy);
      t13 = -2.0 * (0.25 * (mu_xmm + mu_cm + mu_xm + mu_c)) * S13;
      t13p = -2.0 * (0.25 * (mu_cm + mu_xpm + mu_c + mu_xp)) * S13p;
      t23 = -2.0 * (0.25 * (mu_ymm + mu_cm + mu_ym + mu_c)) * S23;
      t23p = -2.0 * (0.25 * (mu_cm + mu_ypm + mu_c + mu_yp)) * S23p;
      Fz = -0.5 * (K_m + K_c) * ((th_c - th_m) * rhw);
    }
    // ---- finish cell k-1
    if (k >= 1) {
      const size_t am = kk - plane + c;
      const double rdzm = p.rdz[k - 1];
      RU[am] -= HU + (t13 - t13_b) * rdzm;
      RV[am] -= HV + (t23 - t23_b) * rdzm;
      RTh[am] -= HT + (Fz - Fz_b) * rdzm;
    }
    if (!cell) break;
    t13_b = t13; t23_b = t23; Fz_b = Fz;
    // ---- cell k
    const double u_m = u[kk + xm], u_ym = u[kk + ym], u_pym = u[kk + xpym], u_yp = u[kk + yp];
    const double v_m = v[kk + ym], v_xm = v[kk + xm], v_xmp = v[kk + xmyp], v_xp = v[kk + xp];
    const double wt_c = w[kk + plane + c], wt_xm = w[kk + plane + xm], wt_xp = w[kk + plane + xp];
    const double wt_ym = w[kk + plane + ym], wt_yp = w[kk + plane + yp];
    const double rdz = p.rdz[k];
    // normal stresses at centres c, xm, ym
    const double S11c = (u_p - u_c) * rdx, S22c = (v_p - v_c) * rdy, S33c = (wt_c - w_c) * rdz;
    const double S11x = (u_c - u_m) * rdx, S22x = (v_xmp - v_xm) * rdy, S33x = (wt_xm - w_xm) * rdz;
    const double S11y = (u_pym - u_ym) * rdx, S22y = (v_c - v_m) * rdy, S33y = (wt_ym - w_ym) * rdz;
    const double d3c = (S11c + S22c + S33c) / 3.0, d3x = (S11x + S22x + S33x) / 3.0, d3y = (S11y + S22y + S33y) / 3.0;
    const double t11c = -2.0 * mu_c * (S11c - d3c), t22c = -2.0 * mu_c * (S22c - d3c), t33c = -2.0 * mu_c * (S33c - d3c);
    const double t11x = -2.0 * mu_xm * (S11x - d3x);
    const double t22y = -2.0 * mu_ym * (S22y - d3y);
    // tau12 at edges (i,j), (i,j+1), (i+1,j)
    const double mu_xmym = mu[kk + xmym], mu_xpym = mu[kk + xpym], mu_xmyp = mu[kk + xmyp];
    const double S12 = 0.5 * ((u_c - u_ym) * rdy + (v_c - v_xm) * rdx);
    const double S12yp = 0.5 * ((u_yp - u_c) * rdy + (v_p - v_xmp) * rdx);
    const double S12xp = 0.5 * ((u_p - u_pym) * rdy + (v_xp - v_c) * rdx);
    const double t12 = -2.0 * (0.25 * (mu_xmym + mu_ym + mu_xm + mu_c)) * S12;
    const double t12yp = -2.0 * (0.25 * (mu_xm + mu_c + mu_xmyp + mu_yp)) * S12yp;
    const double t12xp = -2.0 * (0.25 * (mu_ym + mu_xpym + mu_c + mu_xp)) * S12xp;
    HU = (t11c - t11x) * rdx + (t12yp - t12) * rdy;
    HV = (t12xp - t12) * rdx + (t22c - t22y) * rdy;
    // scalar fluxes through the x- and y-faces
    const double th_xm = th[kk + xm], th_xp = th[kk + xp], th_ym = th[kk + ym], th_yp = th[kk + yp];
    const double K_xm = Kf[kk + xm], K_xp = Kf[kk + xp], K_ym = Kf[kk + ym], K_yp = Kf[kk + yp];
    const double Fx = -0.5 * (K_xm + K_c) * ((th_c - th_xm) * rdx), Fxp = -0.5 * (K_c + K_xp) * ((th_xp - th_c) * rdx);
    const double Fy = -0.5 * (K_ym + K_c) * ((th_c - th_ym) * rdy), Fyp = -0.5 * (K_c + K_yp) * ((th_yp - th_c) * rdy);
    HT = (Fxp - Fx) * rdx + (Fyp - Fy) * rdy;
    if (k >= 1) RW[kk + c] -= (t13p - t13) * rdx + (t23p - t23) * rdy + (t33c - t33_m) * p.rhw[k];
    // carry
    u_cm = u_c; u_pm = u_p; v_cm = v_c; v_pm = v_p;
    mu_cm = mu_c; mu_xmm = mu_xm; mu_xpm = mu_xp; mu_ymm = mu_ym; mu_ypm = mu_yp;
    K_m = K_c; th_m = th_c; t33_m = t33c;
    w_c = wt_c; w_xm = wt_xm; w_xp = wt_xp; w_ym = wt_ym; w_yp = wt_yp;
  }
}

template <int OH>
static void launch_adv(const SlowFlat &p, dim3 grid, dim3 block, cudaStream_t st) {
  k_adv_flat<OH><<<grid, block, 0, st>>>(p);
}

void launch_slow_flat(erf_ctx *c, const F5 &S, cudaStream_t st) {
  Timed t(c, T_SLOW_FUSED, st);
  FusedState *z = c->fz;
  SlowFlat p;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.ov = c->p.adv_order_v;
  p.rdx = 1.0 / c->v.dx; p.rdy = 1.0 / c->v.dy; p.g = c->v.g;
  p.rho = S.f[RHO]; p.U = S.f[UU]; p.V = S.f[VV]; p.W = S.f[WW]; p.Th = S.f[TH];
  p.theta = c->theta_t; p.pi = c->pi_t; p.iT = z->iT;
  p.u = c->prim.u; p.v = c->prim.v; p.w = c->prim.w; p.pp = c->prim.pp;
  p.Rrho = c->R.f[RHO]; p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.RTh = c->R.f[TH];
  p.mu = z->mu; p.K = z->Kd;
  p.dz = z->tab.dz; p.rdz = z->tab.rdz; p.rhw = z->tab.rhw; p.rho0 = z->tab.rho0; p.Th0 = z->tab.Th0;
  p.rTh0 = z->tab.rTh0; p.p0 = z->tab.p0; p.pi0 = z->tab.pi0; p.csd2 = z->tab.csd2;
  p.gam = c->v.gam; p.rdocv = c->v.rdocv; p.nu = c->v.nu; p.alpha = c->v.alpha;
  p.rPrt = c->p.diffusion == 2 ? 1.0 / c->v.Prt : 0.0;
  p.diffusion = c->p.diffusion;
  const size_t plane = (size_t)c->nx * c->ny;
  k_prim_flat<<<(unsigned)((plane * (c->nz + 1) + 255) / 256), 256, 0, st>>>(p);
  c->launches++;
  const bool tiled = !(z->variant & 8);  // variant bit 8 (developer knob): the first, untiled column kernels
  dim3 block(32, 4), grid((c->nx + 31) / 32, (c->ny + 3) / 4);
  if (tiled) {
    launch_adv_diff_tiled(c, p, st);
  } else {
    switch (c->p.adv_order_h) {
      case 2: launch_adv<2>(p, grid, block, st); break;
      case 3: launch_adv<3>(p, grid, block, st); break;
      case 4: launch_adv<4>(p, grid, block, st); break;
      case 5: launch_adv<5>(p, grid, block, st); break;
      default: launch_adv<6>(p, grid, block, st); break;
    }
    c->launches++;
  }
  if (c->p.diffusion != 0) {
    if (tiled) {
      launch_visc_tiled(c, p, st);
      launch_diff_tiled(c, p, st);
    } else {
      k_visc_flat<<<(unsigned)((plane * c->nz + 255) / 256), 256, 0, st>>>(p);
      c->launches++;
      k_diff_flat<<<grid, block, 0, st>>>(p);
      c->launches++;
    }
  }
}

}  // namespace erfb
