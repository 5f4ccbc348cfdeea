// k_fused_acoustic.cu -- one acoustic substep (Appendix A; L138-L144) as ONE
// kernel on flat grids: explicit horizontal momenta, explicit parts of rho'' and Theta'', the
// column tridiagonal system for W'' (Thomas), back-substitution, and the divergence-damped
// Theta''_d for the next substep.
//
// Mapping.  One thread per (i,j) column, a warp = 32 consecutive i (coalesced 256-B rows), a
// block = ROWS consecutive j.  Each thread marches k upward (forward elimination) and then
// downward (back-substitution).  The horizontal momenta a column needs from its +x / +y
// neighbours are recomputed from the neighbours' inputs (no inter-thread exchange, so no
// barrier in the k loop); therefore U'', V'' and Theta''_d are double-buffered across
// substeps (a neighbour may still need the old value after the owner has produced the new).
//
// Column scratch between the two sweeps (4 values per level): c' of the Thomas sweep lives in
// shared memory when it fits (else in an HBM array), d' is parked in the W'' array, the explicit
// parts of Theta'' and rho'' in the Theta''_d output buffer and the rho'' array -- all addresses
// this column alone owns and rewrites in the backward sweep, so the round trip stays in L2.
//
// Algorithmic HBM traffic per cell per substep: reads U'',V'',W'',rho'',Theta'',Theta''_d, the 5
// slow tendencies, theta^t, pi^t, 1/Theta^t (14); writes U'',V'',W'',rho'',Theta'',Theta''_d (6).
#include "fused.cuh"

namespace erfb {

struct AcFlat {
  int nx, ny, nz;
  double dtau, rdx, rdy, b1, b2, beta_d, g, gR;
  const double *thd_in;
  double *thd_out;
  const double *U_in, *V_in;
  double *U_out, *V_out;
  double *W, *rho, *Th;
  const double *RU, *RV, *RW, *Rrho, *RTh;
  const double *theta, *pi, *iT;
  const double *rdz, *rhw, *tabB;
  double *cp_scr;
};

template <int ROWS, bool CP_SMEM>
__global__ void __launch_bounds__(32 * ROWS) k_acoustic_flat(const AcFlat p) {
  extern __shared__ double s_cp[];  // [nz][32*ROWS] when CP_SMEM
  const int lane = threadIdx.x, row = threadIdx.y;
  const int i = blockIdx.x * 32 + lane, j = blockIdx.y * ROWS + row;
  if (i >= p.nx || j >= p.ny) return;
  const int tid = row * 32 + lane, nthr = 32 * ROWS;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const size_t plane = (size_t)nx * ny;
  const size_t oc = (size_t)j * nx + i, oxm = (size_t)j * nx + im, oxp = (size_t)j * nx + ip;
  const size_t oym = (size_t)jm * nx + i, oyp = (size_t)jp * nx + i;

  const double dtau = p.dtau, b1 = p.b1, b2 = p.b2, g = p.g, gR = p.gR;
  const double cU = dtau * gR * 0.5 * p.rdx, cV = dtau * gR * 0.5 * p.rdy;
  const double hx = 0.5 * p.rdx, hy = 0.5 * p.rdy;  // face theta = 0.5 (a + b), folded with 1/dx
  const double s = dtau * dtau * b2 * b2;
  const double sg2 = s * g * 0.5;

  // ---------------- forward sweep: k = 0 .. nz-1 ----------------
  double pi_m = 0.0, th_m = 0.0;        // pi^t, theta^t at level k-1
  double thf_b = 0.0, thf_bm = 0.0;     // theta^t at w-faces k and k-1
  double iT_m = 0.0, rT_m = 0.0, rhc_m = 0.0;
  double That_m = 0.0, rhat_m = 0.0, cp_m = 0.0, dp_m = 0.0;
  double om_b = 0.0;                    // Omega''(k) = W''(k) at the end of the previous substep (0 on the lid)
  double th_c = p.theta[oc];            // theta^t(k), loaded one level ahead
  for (int k = 0; k < nz; k++) {
    const size_t kk = (size_t)k * plane;
    const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
    // explicit horizontal momenta (L585 rows 1-2) at the four faces of the column
    const double d_c = p.thd_in[a], d_xm = p.thd_in[axm], d_xp = p.thd_in[axp], d_ym = p.thd_in[aym],
                 d_yp = p.thd_in[ayp];
    const double pi_c = p.pi[a], pi_xm = p.pi[axm], pi_xp = p.pi[axp], pi_ym = p.pi[aym], pi_yp = p.pi[ayp];
    const double Um = p.U_in[a] + dtau * p.RU[a] - cU * (pi_xm + pi_c) * (d_c - d_xm);
    const double Up = p.U_in[axp] + dtau * p.RU[axp] - cU * (pi_c + pi_xp) * (d_xp - d_c);
    const double Vm = p.V_in[a] + dtau * p.RV[a] - cV * (pi_ym + pi_c) * (d_c - d_ym);
    const double Vp = p.V_in[ayp] + dtau * p.RV[ayp] - cV * (pi_c + pi_yp) * (d_yp - d_c);
    p.U_out[a] = Um;
    p.V_out[a] = Vm;
    // explicit parts of Theta'' and rho'' (L585 rows 4-5 with the old-time part of the W'' average)
    const double th_xm = p.theta[axm], th_xp = p.theta[axp], th_ym = p.theta[aym], th_yp = p.theta[ayp];
    const double th_t = (k + 1 < nz) ? p.theta[a + plane] : 0.0;  // theta^t(k+1)
    const double thf_t = (k + 1 < nz) ? 0.5 * (th_c + th_t) : 0.0;
    const double om_t = (k + 1 < nz) ? p.W[a + plane] : 0.0;
    const double rhc = p.rdz[k];
    const double DhT = (Up * (th_c + th_xp) - Um * (th_xm + th_c)) * hx + (Vp * (th_c + th_yp) - Vm * (th_ym + th_c)) * hy;
    const double Dh = (Up - Um) * p.rdx + (Vp - Vm) * p.rdy;
    const double Tpp = p.Th[a], rpp = p.rho[a];
    const double Ttil = Tpp + dtau * (p.RTh[a] - DhT - b1 * (thf_t * om_t - thf_b * om_b) * rhc);
    const double rtil = rpp + dtau * (p.Rrho[a] - Dh - b1 * (om_t - om_b) * rhc);
    const double That = b2 * Ttil + b1 * Tpp, rhat = b2 * rtil + b1 * rpp;
    p.thd_out[a] = Ttil;  // parked until the backward sweep
    p.rho[a] = rtil;
    const double iT = p.iT[a];
    const double rT = rhc * iT;
    if (k >= 1) {
      // row k of the tridiagonal system for Omega''new (S5), Thomas forward elimination
      const double pif = 0.5 * (pi_m + pi_c);
      const double rhw = p.rhw[k];
      const double Bf = p.tabB[k] * pif;
      const double a1 = s * gR * pif * rhw, bB = sg2 * Bf;
      double Cc = thf_t * (bB * rT - a1 * rhc) - sg2 * rhc;
      double Ac = sg2 * rhc_m - thf_bm * (a1 * rhc_m + bB * rT_m);
      const double Dc = 1.0 + thf_b * (a1 * (rhc + rhc_m) - bB * (rT - rT_m)) + sg2 * (rhc - rhc_m);
      if (k == nz - 1) Cc = 0.0;
      if (k == 1) Ac = 0.0;
      const double rhs = om_b + dtau * (p.RW[a] - gR * pif * rhw * (That - That_m) +
                                        g * Bf * 0.5 * (That * iT + That_m * iT_m) - g * 0.5 * (rhat + rhat_m));
      const double minv = 1.0 / (Dc - Ac * cp_m);
      cp_m = Cc * minv;
      dp_m = (rhs - Ac * dp_m) * minv;
      if (CP_SMEM) s_cp[k * nthr + tid] = cp_m;
      else p.cp_scr[a] = cp_m;
      p.W[a] = dp_m;  // parked
    }
    pi_m = pi_c;
    th_m = th_c;
    th_c = th_t;
    thf_bm = thf_b;
    thf_b = thf_t;
    iT_m = iT;
    rT_m = rT;
    rhc_m = rhc;
    That_m = That;
    rhat_m = rhat;
    om_b = om_t;
  }
  (void)th_m;
  // ---------------- backward sweep: k = nz-1 .. 0 ----------------
  double On_t = 0.0;  // Omega''new(k+1); lid: 0
  double thc = p.theta[(size_t)(nz - 1) * plane + oc];
  double thft = 0.0;  // theta^t at face k+1
  const double cb = dtau * b2;
  for (int k = nz - 1; k >= 0; k--) {
    const size_t a = (size_t)k * plane + oc;
    double On_b = 0.0, thfb = 0.0, thm = 0.0;
    if (k >= 1) {
      const double cp = CP_SMEM ? s_cp[k * nthr + tid] : p.cp_scr[a];
      On_b = p.W[a] - cp * On_t;
      p.W[a] = On_b;  // W'' = Omega'' on a flat grid
      thm = p.theta[a - plane];
      thfb = 0.5 * (thm + thc);
    }
    const double rhc = p.rdz[k];
    const double Tnew = p.thd_out[a] - cb * (thft * On_t - thfb * On_b) * rhc;
    const double rnew = p.rho[a] - cb * (On_t - On_b) * rhc;
    const double Told = p.Th[a];
    p.Th[a] = Tnew;
    p.rho[a] = rnew;
    p.thd_out[a] = Tnew + p.beta_d * (Tnew - Told);  // divergence damping for the next substep (L144) [R:G6]
    On_t = On_b;
    thft = thfb;
    thc = thm;
  }
}

void launch_acoustic_flat(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st) {
  (void)St;
  FusedState *z = c->fz;
  AcFlat p;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
  p.dtau = dtau; p.rdx = 1.0 / c->v.dx; p.rdy = 1.0 / c->v.dy;
  p.b1 = 0.5 * (1.0 - c->v.beta_s); p.b2 = 0.5 * (1.0 + c->v.beta_s);  // L589
  p.beta_d = c->v.beta_d; p.g = c->v.g; p.gR = c->v.gam * c->v.Rd;
  p.W = c->P.f[WW]; p.rho = c->P.f[RHO]; p.Th = c->P.f[TH];
  p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.Rrho = c->R.f[RHO]; p.RTh = c->R.f[TH];
  p.theta = c->theta_t; p.pi = c->pi_t; p.iT = z->iT;
  p.rdz = z->tab.rdz; p.rhw = z->tab.rhw; p.tabB = z->tab.tabB;
  p.cp_scr = z->cp_scr;
  constexpr int ROWS = 4;
  dim3 block(32, ROWS), grid((c->nx + 31) / 32, (c->ny + ROWS - 1) / ROWS);
  size_t smem = (size_t)c->nz * 32 * ROWS * sizeof(double);
  bool cp_smem = smem <= 200 * 1024 && z->variant != 1;
  if (cp_smem) cudaFuncSetAttribute(k_acoustic_flat<ROWS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int cur = 0;
  for (int sidx = 0; sidx < n; sidx++) {
    Timed t(c, T_ACOUSTIC_FUSED, st);
    p.thd_in = z->Thd[cur]; p.thd_out = z->Thd[cur ^ 1];
    p.U_in = c->P.f[UU]; p.V_in = c->P.f[VV]; p.U_out = z->U2; p.V_out = z->V2;
    if (cp_smem) k_acoustic_flat<ROWS, true><<<grid, block, smem, st>>>(p);
    else k_acoustic_flat<ROWS, false><<<grid, block, 0, st>>>(p);
    c->launches++;
    // the new U'', V'' are the current ones: swap buffers
    double *t1 = c->P.f[UU]; c->P.f[UU] = z->U2; z->U2 = t1;
    double *t2 = c->P.f[VV]; c->P.f[VV] = z->V2; z->V2 = t2;
    cur ^= 1;
  }
  if (cur) {  // keep Thd[0] the live buffer
    double *t = z->Thd[0]; z->Thd[0] = z->Thd[1]; z->Thd[1] = t;
  }
}

}  // namespace erfb
