// k_acoustic_terrain.cu -- one acoustic substep (Appendix A; L138-L144) on TERRAIN-FOLLOWING
// grids as one kernel: the explicit horizontal momenta with the metric part of the pressure gradient (L178)
// [R:G14], the slope part omega of W'' [R:G16], the explicit parts of rho'' and Theta'', the column tridiagonal
// system for Omega'' (Thomas) and the back-substitution -- the passes ac_horiz, ac_slope and ac_column of the
// general path (general_cells.cuh, whose arithmetic this file follows term by term) fused into one thread-per-column
// sweep.  Theta''_d (divergence damping, L144) still comes from the small ac_damp pass.
//
// Mapping as in k_fused_acoustic.cu: one thread per (i,j) column, a warp = 32 consecutive i, forward elimination
// upward, back-substitution downward; the new U'', V'' of the +x / +y neighbour faces are recomputed (no exchange),
// so U'', V'' are double-buffered across substeps.  Column scratch (c', d', Theta~, rho~, omega) in HBM arrays.
#include "erf_ctx.cuh"

namespace erfb {

struct AcTerr {
  int nx, ny, nz;
  double dtau, rdx, rdy, b1, b2, g, gR, rdocv;
  const double *Thd;                 // Theta''_d
  const double *U_in, *V_in;
  double *U_out, *V_out;
  double *W, *Om, *rho, *Th;         // W'', Omega'' (end of the previous substep), rho'', Theta''
  const double *RU, *RV, *RW, *Rrho, *RTh;
  const double *theta, *pi, *Th_t;   // stage constants theta^t, pi^t, Theta^t
  const double *hc, *hx, *hy, *hw, *sxw, *syw, *sxu, *syv, *rdzc, *rho0, *pi0;  // geometry and base state (3-D)
  double *cpr, *dpr, *Ttil, *rtil, *om;  // column scratch
};

// 1 / (zc(kt) - zc(kb)), kt = min(k+1, nz-1), kb = max(k-1, 0): the denominator of the centred vertical difference
// in the metric part of the horizontal gradient (dz_centre of the general path); 0 when nz == 1
__global__ void k_rdzc(int nx, int ny, int nz, const double *zc, double *rdzc) {
  const size_t plane = (size_t)nx * ny;
  const size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= plane * nz) return;
  const int k = (int)(a / plane);
  const size_t o = a - (size_t)k * plane;
  const int kb = k > 0 ? k - 1 : 0, kt = k < nz - 1 ? k + 1 : nz - 1;
  rdzc[a] = kt > kb ? 1.0 / (zc[(size_t)kt * plane + o] - zc[(size_t)kb * plane + o]) : 0.0;
}

__global__ void __launch_bounds__(128, 2) k_acoustic_terrain(const AcTerr p) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
  if (i >= p.nx || j >= p.ny) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const size_t plane = (size_t)nx * ny;
  const size_t oc = (size_t)j * nx + i, oxm = (size_t)j * nx + im, oxp = (size_t)j * nx + ip;
  const size_t oym = (size_t)jm * nx + i, oyp = (size_t)jp * nx + i;
  const double *__restrict__ Thd = p.Thd, *__restrict__ U_in = p.U_in, *__restrict__ V_in = p.V_in;
  const double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW;
  const double *__restrict__ Rrho = p.Rrho, *__restrict__ RTh = p.RTh;
  const double *__restrict__ theta = p.theta, *__restrict__ pi = p.pi, *__restrict__ Th_t = p.Th_t;
  const double *__restrict__ hc_ = p.hc, *__restrict__ hx = p.hx, *__restrict__ hy = p.hy, *__restrict__ hw_ = p.hw;
  const double *__restrict__ sxw = p.sxw, *__restrict__ syw = p.syw, *__restrict__ sxu = p.sxu, *__restrict__ syv = p.syv;
  const double *__restrict__ rdzc = p.rdzc, *__restrict__ rho0 = p.rho0, *__restrict__ pi0 = p.pi0;
  const double dtau = p.dtau, b1 = p.b1, b2 = p.b2, g = p.g, gR = p.gR, rdx = p.rdx, rdy = p.rdy;
  const double s = dtau * dtau * b2 * b2;

  // Theta''_d of the five columns at levels k-1, k, k+1 (one-sided at the lids: the clamped level repeats)
  double dm_c, dm_xm, dm_xp, dm_ym, dm_yp;  // level max(k-1, 0)
  double d_c, d_xm, d_xp, d_ym, d_yp;       // level k
  d_c = Thd[oc]; d_xm = Thd[oxm]; d_xp = Thd[oxp]; d_ym = Thd[oym]; d_yp = Thd[oyp];
  dm_c = d_c; dm_xm = d_xm; dm_xp = d_xp; dm_ym = d_ym; dm_yp = d_yp;
  double Um_m = 0.0, Up_m = 0.0, Vm_m = 0.0, Vp_m = 0.0;  // new face momenta of level k-1
  double th_m = 0.0, th_mm = 0.0;                          // theta^t at k-1, k-2
  double pi_m = 0.0, pi0_m = 0.0, rho0_m = 0.0, hc_m = 0.0, Tt_m = 0.0;
  double That_m = 0.0, rhat_m = 0.0, cp_m = 0.0, dp_m = 0.0;
  double th_c = theta[oc];

#pragma unroll 1
  for (int k = 0; k < nz; k++) {
    const size_t kk = (size_t)k * plane;
    const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
    const bool top = k + 1 >= nz;
    const size_t up = top ? 0 : plane;  // clamped level k+1
    const double dp_c = Thd[a + up], dp_xm = Thd[axm + up], dp_xp = Thd[axp + up], dp_ym = Thd[aym + up],
                 dp_yp = Thd[ayp + up];
    // centred vertical differences of Theta''_d (dz_centre) in the five columns
    const double z_c = (dp_c - dm_c) * rdzc[a], z_xm = (dp_xm - dm_xm) * rdzc[axm], z_xp = (dp_xp - dm_xp) * rdzc[axp];
    const double z_ym = (dp_ym - dm_ym) * rdzc[aym], z_yp = (dp_yp - dm_yp) * rdzc[ayp];
    const double pi_c = pi[a];
    // explicit horizontal momenta (L585 rows 1-2) with G_x(phi) = d_x phi / dx - sxu avg(d_z phi) [R:G14]
    const double Gxm = (d_c - d_xm) * rdx - sxu[a] * 0.5 * (z_xm + z_c);
    const double Gxp = (d_xp - d_c) * rdx - sxu[axp] * 0.5 * (z_c + z_xp);
    const double Gym = (d_c - d_ym) * rdy - syv[a] * 0.5 * (z_ym + z_c);
    const double Gyp = (d_yp - d_c) * rdy - syv[ayp] * 0.5 * (z_c + z_yp);
    const double Um = U_in[a] + dtau * (-gR * (0.5 * (pi[axm] + pi_c)) * Gxm + RU[a]);
    const double Up = U_in[axp] + dtau * (-gR * (0.5 * (pi_c + pi[axp])) * Gxp + RU[axp]);
    const double Vm = V_in[a] + dtau * (-gR * (0.5 * (pi[aym] + pi_c)) * Gym + RV[a]);
    const double Vp = V_in[ayp] + dtau * (-gR * (0.5 * (pi_c + pi[ayp])) * Gyp + RV[ayp]);
    p.U_out[a] = Um;
    p.V_out[a] = Vm;
    // explicit parts of Theta'' and rho'' (L585 rows 4-5 with the old-time part of the Omega'' average)
    const double th_t = top ? 0.0 : theta[a + plane];
    const double thx_m = 0.5 * (theta[axm] + th_c), thx_p = 0.5 * (th_c + theta[axp]);
    const double thy_m = 0.5 * (theta[aym] + th_c), thy_p = 0.5 * (th_c + theta[ayp]);
    const double hc = hc_[a], rhc = 1.0 / hc;
    const double fxp = hx[axp] * Up, fxm = hx[a] * Um, fyp = hy[ayp] * Vp, fym = hy[a] * Vm;
    const double DhT = ((fxp * thx_p - fxm * thx_m) * rdx + (fyp * thy_p - fym * thy_m) * rdy) * rhc;
    const double Dh = ((fxp - fxm) * rdx + (fyp - fym) * rdy) * rhc;
    const double thf_b = k >= 1 ? 0.5 * (th_m + th_c) : 0.0;
    const double thf_t = top ? 0.0 : 0.5 * (th_c + th_t);
    const double om_b = p.Om[a], om_t = p.Om[a + plane];
    const double Tpp = p.Th[a], rpp = p.rho[a];
    const double Ttil = Tpp + dtau * (RTh[a] - DhT - b1 * (thf_t * om_t - thf_b * om_b) * rhc);
    const double rtil = rpp + dtau * (Rrho[a] - Dh - b1 * (om_t - om_b) * rhc);
    const double That = b2 * Ttil + b1 * Tpp, rhat = b2 * rtil + b1 * rpp;
    p.Ttil[a] = Ttil;
    p.rtil[a] = rtil;
    const double pi0_c = pi0[a], rho0_c = rho0[a], Tk = Th_t[a];
    if (k >= 1) {
      // slope part of W'' from the new momenta [R:G16], then row k of the tridiagonal system (S5)
      const double om = sxw[a] * (0.25 * (Um_m + Up_m + Um + Up)) + syw[a] * (0.25 * (Vm_m + Vp_m + Vm + Vp));
      const double pif = 0.5 * (pi_m + pi_c);
      const double Bf = (0.5 * (rho0_m + rho0_c)) * p.rdocv * pif / (0.5 * (pi0_m + pi0_c));
      const double thf_km = k >= 2 ? 0.5 * (th_mm + th_m) : 0.0;
      const double rhw = 1.0 / hw_[a], rhcm = 1.0 / hc_m, rTk = 1.0 / Tk, rTm = 1.0 / Tt_m;
      double Cc = -s * gR * pif * thf_t * rhw * rhc + s * g * Bf * thf_t * 0.5 * rhc * rTk - s * g * 0.5 * rhc;
      double Ac = -s * gR * pif * thf_km * rhw * rhcm - s * g * Bf * thf_km * 0.5 * rhcm * rTm + s * g * 0.5 * rhcm;
      const double Dc = 1.0 + s * gR * pif * thf_b * (rhc + rhcm) * rhw - s * g * Bf * thf_b * 0.5 * (rhc * rTk - rhcm * rTm) +
                        s * g * 0.5 * (rhc - rhcm);
      if (k == nz - 1) Cc = 0.0;
      if (k == 1) Ac = 0.0;
      const double rhs = p.W[a] + dtau * (RW[a] - gR * pif * (That - That_m) * rhw +
                                          g * Bf * 0.5 * (That * rTk + That_m * rTm) - g * 0.5 * (rhat + rhat_m)) - om;
      const double minv = 1.0 / (Dc - Ac * cp_m);
      cp_m = Cc * minv;
      dp_m = (rhs - Ac * dp_m) * minv;
      p.cpr[a] = cp_m;
      p.dpr[a] = dp_m;
      p.om[a] = om;
    }
    // carry
    dm_c = d_c; dm_xm = d_xm; dm_xp = d_xp; dm_ym = d_ym; dm_yp = d_yp;
    d_c = dp_c; d_xm = dp_xm; d_xp = dp_xp; d_ym = dp_ym; d_yp = dp_yp;
    Um_m = Um; Up_m = Up; Vm_m = Vm; Vp_m = Vp;
    th_mm = th_m; th_m = th_c; th_c = th_t;
    pi_m = pi_c; pi0_m = pi0_c; rho0_m = rho0_c; hc_m = hc; Tt_m = Tk;
    That_m = That; rhat_m = rhat;
  }
  // ---------------- backward sweep: k = nz-1 .. 0 ----------------
  double On_t = 0.0;  // Omega''new(k+1); lid: 0
  double thc = theta[(size_t)(nz - 1) * plane + oc], tht = 0.0;
  const double cb = dtau * b2;
#pragma unroll 1
  for (int k = nz - 1; k >= 0; k--) {
    const size_t a = (size_t)k * plane + oc;
    double On_b = 0.0, thm = 0.0;
    if (k >= 1) {
      On_b = p.dpr[a] - p.cpr[a] * On_t;
      p.W[a] = On_b + p.om[a];
      thm = theta[a - plane];
    }
    const double thf_b = k >= 1 ? 0.5 * (thm + thc) : 0.0;
    const double thf_t = k + 1 <= nz - 1 ? 0.5 * (thc + tht) : 0.0;
    const double rhc = 1.0 / hc_[a];
    p.Th[a] = p.Ttil[a] - cb * (thf_t * On_t - thf_b * On_b) * rhc;
    p.rho[a] = p.rtil[a] - cb * (On_t - On_b) * rhc;
    p.Om[a + plane] = On_t;
    On_t = On_b;
    tht = thc;
    thc = thm;
  }
  p.Om[oc] = 0.0;
}

// ------------------------------------------------------------------ driver
bool terrain_acoustic_available(const erf_ctx *c) {
  return !c->v.flat && c->p.substep_mode == 1 && c->v.perx && c->v.pery;  // the kernel wraps its neighbour indices
}

// n substeps of size dtau about the stage state St (theta_t, pi_t, R, P set by the caller): general_acoustic with
// its three heavy passes per substep fused into k_acoustic_terrain
void terrain_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st) {
  View v = c->v;
  const int nz = c->nz;
  if (!c->terr_U2) {  // first use: second U'', V'' buffers and the metric denominators
    c->terr_U2 = c->alloc(c->NW);
    c->terr_V2 = c->alloc(c->NW);
    c->terr_rdzc = c->alloc(c->NW);
    if (!c->terr_U2 || !c->terr_V2 || !c->terr_rdzc) return;
    const size_t nc = (size_t)c->nx * c->ny * nz;
    k_rdzc<<<(unsigned)((nc + 255) / 256), 256, 0, st>>>(c->nx, c->ny, nz, v.zc, c->terr_rdzc);
    c->launches++;
  }
  gen::Acou A = c->ac;
  A.theta_t = c->theta_t;
  A.pi_t = c->pi_t;
  A.Th_t = St.f[TH];
  for (int m = 0; m < 5; m++) {
    A.R[m] = c->R.f[m];
    A.P[m] = c->P.f[m];
  }
  // Omega'' of the initial S''; Theta''_prev = Theta''
  launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) {
    size_t a = IX(v, i, j, k);
    A.Om[a] = gen::omega_at(v, A.P[UU], A.P[VV], A.P[WW], i, j, k);
    if (k < v.nz) A.Th_prev[a] = A.P[TH][a];
  });
  AcTerr p;
  p.nx = c->nx; p.ny = c->ny; p.nz = nz;
  p.dtau = dtau; p.rdx = 1.0 / v.dx; p.rdy = 1.0 / v.dy;
  p.b1 = 0.5 * (1.0 - v.beta_s); p.b2 = 0.5 * (1.0 + v.beta_s);  // L589
  p.g = v.g; p.gR = v.gam * v.Rd; p.rdocv = v.rdocv;
  p.Thd = A.Thd;
  p.W = c->P.f[WW]; p.Om = A.Om; p.rho = c->P.f[RHO]; p.Th = c->P.f[TH];
  p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.Rrho = c->R.f[RHO]; p.RTh = c->R.f[TH];
  p.theta = c->theta_t; p.pi = c->pi_t; p.Th_t = St.f[TH];
  p.hc = v.hc; p.hx = v.hx; p.hy = v.hy; p.hw = v.hw; p.sxw = v.sxw; p.syw = v.syw; p.sxu = v.sxu; p.syv = v.syv;
  p.rdzc = c->terr_rdzc; p.rho0 = v.rho0; p.pi0 = v.pi0;
  p.cpr = A.cpr; p.dpr = A.dpr; p.Ttil = A.Ttil; p.rtil = A.rtil; p.om = A.om;
  dim3 block(32, 4), grid((c->nx + 31) / 32, (c->ny + 3) / 4);
  for (int s = 0; s < n; s++) {
    launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::ac_damp(v, A, i, j, k); });
    p.U_in = c->P.f[UU]; p.V_in = c->P.f[VV]; p.U_out = c->terr_U2; p.V_out = c->terr_V2;
    k_acoustic_terrain<<<grid, block, 0, st>>>(p);
    c->launches++;
    double *t1 = c->P.f[UU]; c->P.f[UU] = c->terr_U2; c->terr_U2 = t1;
    double *t2 = c->P.f[VV]; c->P.f[VV] = c->terr_V2; c->terr_V2 = t2;
  }
}

}  // namespace erfb
