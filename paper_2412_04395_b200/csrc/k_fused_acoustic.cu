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

// everything the forward sweep reads at one level
struct FwdIn {
  double d_c, d_xm, d_xp, d_ym, d_yp;       // Theta''_d
  double pi_c, pi_xm, pi_xp, pi_ym, pi_yp;  // pi^t
  double th_xm, th_xp, th_ym, th_yp, th_t;  // theta^t neighbours and theta^t(k+1)
  double U_c, U_xp, RU_c, RU_xp, V_c, V_yp, RV_c, RV_yp;
  double om_t, RW, Tpp, rpp, RTh, Rrho, iT;
};

// PF: forward-sweep software prefetch depth in levels (0 or 1); BD: backward-sweep prefetch depth;
// MINB: blocks per SM the register allocation must allow.
template <int ROWS, bool CP_SMEM, int PF, int MINB>
__global__ void __launch_bounds__(32 * ROWS, MINB) k_acoustic_flat(const AcFlat p) {
  constexpr int BD = 4;
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

  const double *__restrict__ thd_in = p.thd_in;
  double *__restrict__ thd_out = p.thd_out;
  const double *__restrict__ U_in = p.U_in, *__restrict__ V_in = p.V_in;
  double *__restrict__ U_out = p.U_out, *__restrict__ V_out = p.V_out;
  double *__restrict__ Wf = p.W, *__restrict__ rhof = p.rho, *__restrict__ Thf = p.Th;
  const double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW;
  const double *__restrict__ Rrho = p.Rrho, *__restrict__ RTh = p.RTh;
  const double *__restrict__ theta = p.theta, *__restrict__ pi = p.pi, *__restrict__ iTf = p.iT;
  const double *__restrict__ rdz = p.rdz, *__restrict__ rhwt = p.rhw, *__restrict__ tabB = p.tabB;
  double *__restrict__ cp_scr = p.cp_scr;

  const double dtau = p.dtau, b1 = p.b1, b2 = p.b2, g = p.g, gR = p.gR;
  const double cU = dtau * gR * 0.5 * p.rdx, cV = dtau * gR * 0.5 * p.rdy;
  const double hx = 0.5 * p.rdx, hy = 0.5 * p.rdy;  // face theta = 0.5 (a + b), folded with 1/dx
  const double s = dtau * dtau * b2 * b2;
  const double sg2 = s * g * 0.5;

  auto load_fwd = [&](int k, FwdIn &q) {
    const size_t kk = (size_t)k * plane;
    const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
    q.d_c = thd_in[a]; q.d_xm = thd_in[axm]; q.d_xp = thd_in[axp]; q.d_ym = thd_in[aym]; q.d_yp = thd_in[ayp];
    q.pi_c = pi[a]; q.pi_xm = pi[axm]; q.pi_xp = pi[axp]; q.pi_ym = pi[aym]; q.pi_yp = pi[ayp];
    q.th_xm = theta[axm]; q.th_xp = theta[axp]; q.th_ym = theta[aym]; q.th_yp = theta[ayp];
    q.U_c = U_in[a]; q.U_xp = U_in[axp]; q.RU_c = RU[a]; q.RU_xp = RU[axp];
    q.V_c = V_in[a]; q.V_yp = V_in[ayp]; q.RV_c = RV[a]; q.RV_yp = RV[ayp];
    const bool top = k + 1 >= nz;
    q.th_t = top ? 0.0 : theta[a + plane];
    q.om_t = top ? 0.0 : Wf[a + plane];
    q.RW = RW[a]; q.Tpp = Thf[a]; q.rpp = rhof[a]; q.RTh = RTh[a]; q.Rrho = Rrho[a]; q.iT = iTf[a];
  };

  // ---------------- forward sweep: k = 0 .. nz-1 ----------------
  double pi_m = 0.0;                 // pi^t at level k-1
  double thf_b = 0.0, thf_bm = 0.0;  // theta^t at w-faces k and k-1
  double iT_m = 0.0, rT_m = 0.0, rhc_m = 0.0;
  double That_m = 0.0, rhat_m = 0.0, cp_m = 0.0, dp_m = 0.0;
  double om_b = 0.0;                 // Omega''(k) = W''(k) at the end of the previous substep (0 on the lid)
  double th_c = theta[oc];           // theta^t(k)
  FwdIn cur, nxt;
  if (PF) load_fwd(0, cur);
#pragma unroll 1
  for (int k = 0; k < nz; k++) {
    if (PF) {
      if (k + 1 < nz) load_fwd(k + 1, nxt);  // software pipeline: next level's loads fly during this level's math
    } else {
      load_fwd(k, cur);
    }
    const size_t a = (size_t)k * plane + oc;
    const bool top = k + 1 >= nz;
    // explicit horizontal momenta (L585 rows 1-2) at the four faces of the column
    const double Um = cur.U_c + dtau * cur.RU_c - cU * (cur.pi_xm + cur.pi_c) * (cur.d_c - cur.d_xm);
    const double Up = cur.U_xp + dtau * cur.RU_xp - cU * (cur.pi_c + cur.pi_xp) * (cur.d_xp - cur.d_c);
    const double Vm = cur.V_c + dtau * cur.RV_c - cV * (cur.pi_ym + cur.pi_c) * (cur.d_c - cur.d_ym);
    const double Vp = cur.V_yp + dtau * cur.RV_yp - cV * (cur.pi_c + cur.pi_yp) * (cur.d_yp - cur.d_c);
    // explicit parts of Theta'' and rho'' (L585 rows 4-5 with the old-time part of the W'' average)
    const double thf_t = top ? 0.0 : 0.5 * (th_c + cur.th_t);
    const double om_t = cur.om_t;
    const double rhc = rdz[k];
    const double DhT = (Up * (th_c + cur.th_xp) - Um * (cur.th_xm + th_c)) * hx +
                       (Vp * (th_c + cur.th_yp) - Vm * (cur.th_ym + th_c)) * hy;
    const double Dh = (Up - Um) * p.rdx + (Vp - Vm) * p.rdy;
    const double Tpp = cur.Tpp, rpp = cur.rpp;
    const double Ttil = Tpp + dtau * (cur.RTh - DhT - b1 * (thf_t * om_t - thf_b * om_b) * rhc);
    const double rtil = rpp + dtau * (cur.Rrho - Dh - b1 * (om_t - om_b) * rhc);
    const double That = b2 * Ttil + b1 * Tpp, rhat = b2 * rtil + b1 * rpp;
    const double iT = cur.iT;
    const double rT = rhc * iT;
    const double pi_c = cur.pi_c;
    if (k >= 1) {
      // row k of the tridiagonal system for Omega''new (S5), Thomas forward elimination
      const double pif = 0.5 * (pi_m + pi_c);
      const double rhw = rhwt[k];
      const double Bf = tabB[k] * pif;
      const double a1 = s * gR * pif * rhw, bB = sg2 * Bf;
      double Cc = thf_t * (bB * rT - a1 * rhc) - sg2 * rhc;
      double Ac = sg2 * rhc_m - thf_bm * (a1 * rhc_m + bB * rT_m);
      const double Dc = 1.0 + thf_b * (a1 * (rhc + rhc_m) - bB * (rT - rT_m)) + sg2 * (rhc - rhc_m);
      if (k == nz - 1) Cc = 0.0;
      if (k == 1) Ac = 0.0;
      const double rhs = om_b + dtau * (cur.RW - gR * pif * rhw * (That - That_m) +
                                        g * Bf * 0.5 * (That * iT + That_m * iT_m) - g * 0.5 * (rhat + rhat_m));
      const double minv = 1.0 / (Dc - Ac * cp_m);
      cp_m = Cc * minv;
      dp_m = (rhs - Ac * dp_m) * minv;
      if (CP_SMEM) s_cp[k * nthr + tid] = cp_m;
      else cp_scr[a] = cp_m;
      Wf[a] = dp_m;  // parked until the backward sweep
    }
    U_out[a] = Um;
    V_out[a] = Vm;
    thd_out[a] = Ttil;  // parked
    rhof[a] = rtil;     // parked
    pi_m = pi_c;
    th_c = cur.th_t;
    thf_bm = thf_b;
    thf_b = thf_t;
    iT_m = iT;
    rT_m = rT;
    rhc_m = rhc;
    That_m = That;
    rhat_m = rhat;
    om_b = om_t;
    if (PF) cur = nxt;
  }
  // ---------------- backward sweep: k = nz-1 .. 0 ----------------
  struct BwdIn {
    double dp, cp, Ttil, rtil, Told, thm;
  };
  auto load_bwd = [&](int k, BwdIn &q) {
    const size_t a = (size_t)k * plane + oc;
    if (k >= 1) {
      q.dp = Wf[a];
      q.cp = CP_SMEM ? s_cp[k * nthr + tid] : cp_scr[a];
      q.thm = theta[a - plane];
    } else {
      q.dp = 0.0; q.cp = 0.0; q.thm = 0.0;
    }
    q.Ttil = thd_out[a]; q.rtil = rhof[a]; q.Told = Thf[a];
  };
  double On_t = 0.0;  // Omega''new(k+1); lid: 0
  double thc = theta[(size_t)(nz - 1) * plane + oc];
  double thft = 0.0;  // theta^t at face k+1
  const double cb = dtau * b2;
  BwdIn ring[BD];  // modulo-scheduled ring: ring[n] holds level kb - n
#pragma unroll
  for (int n = 0; n < BD; n++)
    if (nz - 1 - n >= 0) load_bwd(nz - 1 - n, ring[n]);
#pragma unroll 1
  for (int kb = nz - 1; kb >= 0; kb -= BD) {
#pragma unroll
    for (int n = 0; n < BD; n++) {
      const int k = kb - n;
      if (k >= 0) {
        const BwdIn bc = ring[n];
        if (k - BD >= 0) load_bwd(k - BD, ring[n]);
        const size_t a = (size_t)k * plane + oc;
        double On_b = 0.0, thfb = 0.0;
        if (k >= 1) {
          On_b = bc.dp - bc.cp * On_t;
          thfb = 0.5 * (bc.thm + thc);
        }
        const double rhc = rdz[k];
        const double Tnew = bc.Ttil - cb * (thft * On_t - thfb * On_b) * rhc;
        const double rnew = bc.rtil - cb * (On_t - On_b) * rhc;
        if (k >= 1) Wf[a] = On_b;  // W'' = Omega'' on a flat grid
        Thf[a] = Tnew;
        rhof[a] = rnew;
        thd_out[a] = Tnew + p.beta_d * (Tnew - bc.Told);  // divergence damping for the next substep (L144) [R:G6]
        On_t = On_b;
        thft = thfb;
        thc = bc.thm;
      }
    }
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
  // variant bits (developer knob): 1 = forward prefetch, 2 = c' scratch in shared memory, 4 = allow 255 registers
  const int var = z->variant;
  bool cp_smem = smem <= 200 * 1024 && (var & 2);
  auto kern = k_acoustic_flat<ROWS, false, 0, 4>;
  switch (var & 7) {
    case 1: kern = k_acoustic_flat<ROWS, false, 1, 4>; break;
    case 2: kern = k_acoustic_flat<ROWS, true, 0, 4>; break;
    case 3: kern = k_acoustic_flat<ROWS, true, 1, 4>; break;
    case 4: kern = k_acoustic_flat<ROWS, false, 0, 1>; break;
    case 5: kern = k_acoustic_flat<ROWS, false, 1, 1>; break;
    case 6: kern = k_acoustic_flat<ROWS, true, 0, 1>; break;
    case 7: kern = k_acoustic_flat<ROWS, true, 1, 1>; break;
    default: break;
  }
  if (!cp_smem) smem = 0;
  else cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int cur = 0;
  for (int sidx = 0; sidx < n; sidx++) {
    Timed t(c, T_ACOUSTIC_FUSED, st);
    p.thd_in = z->Thd[cur]; p.thd_out = z->Thd[cur ^ 1];
    p.U_in = c->P.f[UU]; p.V_in = c->P.f[VV]; p.U_out = z->U2; p.V_out = z->V2;
    kern<<<grid, block, smem, st>>>(p);
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
