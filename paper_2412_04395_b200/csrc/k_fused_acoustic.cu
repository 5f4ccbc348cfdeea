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
// Column scratch between the two sweeps (4 values per level): c' of the Thomas sweep in an HBM
// array, d' parked in the W'' output, the explicit parts of Theta'' and rho'' in the Theta'' and
// rho'' outputs -- all addresses this column alone owns and rewrites in the backward sweep.
//
// Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev) (L144) [R:G6] is formed at load time from the
// current and the previous Theta'' (three rotating buffers) instead of being stored.
//
// Stage combine folded in (MODE bits).  FIRST: S'' = S^n - S^t is formed at load time (L581) [R:G7]
// (ZERO: RK stage 1, S'' = 0, nothing is loaded).  LAST: the kernel writes S^t + S'' (L593) and the
// flat lids W = 0, so no separate stage-init / stage-finish pass touches HBM.
//
// Algorithmic HBM traffic per cell per substep: reads U'',V'',W'',rho'',Theta'',Theta''_prev, the 5
// slow tendencies, theta^t, pi^t, 1/Theta^t (14); writes U'',V'',W'',rho'',Theta'' (5).
#include "acoustic_args.cuh"

namespace erfb {

// everything the forward sweep reads at one level
struct FwdIn {
  double T_c, d_c, d_xm, d_xp, d_ym, d_yp;  // Theta'' of the own cell; Theta''_d
  double pi_c, pi_xm, pi_xp, pi_ym, pi_yp;  // pi^t
  double th_xm, th_xp, th_ym, th_yp, th_t;  // theta^t neighbours and theta^t(k+1)
  double U_c, U_xp, RU_c, RU_xp, V_c, V_yp, RV_c, RV_yp;
  double om_t, RW, rpp, RTh, Rrho, iT, sU, sV;
};

// ACC: also accumulate the momenta of this substep's continuity equation -- U''new, V''new and beta2 Omega''new + beta1
// Omega''old -- for the transported scalars (Eq. 4 with the stage-time-averaged momenta, L138; k_scalar.cu)
template <int ROWS, int MODE, bool ACC>
__global__ void __launch_bounds__(32 * ROWS, 4) k_acoustic_flat(const AcArgs p) {
  constexpr bool FIRST = (MODE & MODE_FIRST) != 0, LAST = (MODE & MODE_LAST) != 0, ZERO = (MODE & MODE_ZERO) != 0;
  constexpr int BD = 4;
  const int lane = threadIdx.x, row = threadIdx.y;
  const int i = blockIdx.x * 32 + lane, j = blockIdx.y * ROWS + row;
  if (i >= p.nx || j >= p.ny) return;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int im = i == 0 ? nx - 1 : i - 1, ip = i == nx - 1 ? 0 : i + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const size_t plane = (size_t)nx * ny;
  const size_t oc = (size_t)j * nx + i, oxm = (size_t)j * nx + im, oxp = (size_t)j * nx + ip;
  const size_t oym = (size_t)jm * nx + i, oyp = (size_t)jp * nx + i;

  const double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW;
  const double *__restrict__ Rrho = p.Rrho, *__restrict__ RTh = p.RTh;
  const double *__restrict__ theta = p.theta, *__restrict__ pi = p.pi, *__restrict__ iTf = p.iT;
  const double *__restrict__ rdz = p.rdz, *__restrict__ rhwt = p.rhw, *__restrict__ tabB = p.tabB;
  double *__restrict__ cp_scr = p.cp_scr;

  const double dtau = p.dtau, b1 = p.b1, b2 = p.b2, g = p.g, gR = p.gR, beta_d = p.beta_d;
  const double cU = dtau * gR * 0.5 * p.rdx, cV = dtau * gR * 0.5 * p.rdy;
  const double hx = 0.5 * p.rdx, hy = 0.5 * p.rdy;  // face theta = 0.5 (a + b), folded with 1/dx
  const double s = dtau * dtau * b2 * b2;
  const double sg2 = s * g * 0.5;

  // S'' at one point (L581): 0 in RK stage 1, S^n - S^t at the first substep of a stage, else stored
  auto pert = [&](int f, const double *P, size_t a) -> double {
    if (ZERO) return 0.0;
    if (FIRST) return p.Sn[f][a] - p.St[f][a];
    return P[a];
  };
  // Theta''_d (L144) [R:G6]; Theta''_prev = Theta'' at the start of a stage
  auto thd = [&](size_t a) -> double {
    if (ZERO) return 0.0;
    if (FIRST) return p.Sn[TH][a] - p.St[TH][a];
    const double t = p.Pt[a];
    return t + beta_d * (t - p.Ptp[a]);
  };
  auto load_fwd = [&](int k, FwdIn &q) {
    const size_t kk = (size_t)k * plane;
    const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
    if (FIRST) {
      q.T_c = q.d_c = thd(a);
    } else {
      q.T_c = p.Pt[a];
      q.d_c = q.T_c + beta_d * (q.T_c - p.Ptp[a]);
    }
    q.d_xm = thd(axm); q.d_xp = thd(axp); q.d_ym = thd(aym); q.d_yp = thd(ayp);
    q.pi_c = pi[a]; q.pi_xm = pi[axm]; q.pi_xp = pi[axp]; q.pi_ym = pi[aym]; q.pi_yp = pi[ayp];
    q.th_xm = theta[axm]; q.th_xp = theta[axp]; q.th_ym = theta[aym]; q.th_yp = theta[ayp];
    q.U_c = pert(UU, p.Pu, a); q.U_xp = pert(UU, p.Pu, axp); q.RU_c = RU[a]; q.RU_xp = RU[axp];
    q.V_c = pert(VV, p.Pv, a); q.V_yp = pert(VV, p.Pv, ayp); q.RV_c = RV[a]; q.RV_yp = RV[ayp];
    const bool top = k + 1 >= nz;
    q.th_t = top ? 0.0 : theta[a + plane];
    q.om_t = top ? 0.0 : pert(WW, p.Pw, a + plane);
    q.RW = RW[a]; q.rpp = pert(RHO, p.Pr, a); q.RTh = RTh[a]; q.Rrho = Rrho[a]; q.iT = iTf[a];
    q.sU = LAST ? p.St[UU][a] : 0.0;
    q.sV = LAST ? p.St[VV][a] : 0.0;
  };

  // ---------------- forward sweep: k = 0 .. nz-1 ----------------
  double pi_m = 0.0;                 // pi^t at level k-1
  double thf_b = 0.0, thf_bm = 0.0;  // theta^t at w-faces k and k-1
  double iT_m = 0.0, rT_m = 0.0, rhc_m = 0.0;
  double That_m = 0.0, rhat_m = 0.0, cp_m = 0.0, dp_m = 0.0;
  double om_b = 0.0;                 // Omega''(k) = W''(k) at the end of the previous substep (0 on the lid)
  double th_c = theta[oc];           // theta^t(k)
  FwdIn cur;
#pragma unroll 1
  for (int k = 0; k < nz; k++) {
    load_fwd(k, cur);
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
    const double Tpp = cur.T_c, rpp = cur.rpp;
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
      if (p.write_cp) cp_scr[a] = cp_m;  // c' depends on the stage state and dtau only
      p.kW[a] = dp_m;  // parked until the backward sweep
    }
    p.oU[a] = LAST ? cur.sU + Um : Um;
    p.oV[a] = LAST ? cur.sV + Vm : Vm;
    if (ACC) {
      p.sumU[a] += Um;
      p.sumV[a] += Vm;
      if (k >= 1) p.sumOm[a] += b1 * om_b;  // the old-time part of the vertical flux (L591); the new-time part below
    }
    if (FIRST && !LAST && !ZERO) p.oTp[a] = cur.d_c;  // Theta''_prev of the next substep
    p.kT[a] = Ttil;  // parked
    p.kR[a] = rtil;  // parked
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
  }
  // ---------------- backward sweep: k = nz-1 .. 0 ----------------
  struct BwdIn {
    double dp, cp, Ttil, rtil, thm, sW, sT, sR;
  };
  auto load_bwd = [&](int k, BwdIn &q) {
    const size_t a = (size_t)k * plane + oc;
    if (k >= 1) {
      q.dp = p.kW[a];
      q.cp = cp_scr[a];
      q.thm = theta[a - plane];
    } else {
      q.dp = 0.0; q.cp = 0.0; q.thm = 0.0;
    }
    q.Ttil = p.kT[a]; q.rtil = p.kR[a];
    if (LAST) {
      q.sW = p.St[WW][a]; q.sT = p.St[TH][a]; q.sR = p.St[RHO][a];
    } else {
      q.sW = q.sT = q.sR = 0.0;
    }
  };
  double On_t = 0.0;  // Omega''new(k+1); lid: 0
  double thc = theta[(size_t)(nz - 1) * plane + oc];
  double thft = 0.0;  // theta^t at face k+1
  const double cb = dtau * b2;
  if (LAST) p.oW[(size_t)nz * plane + oc] = 0.0;  // flat lid: W = 0 at k = nz
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
        if (ACC && k >= 1) p.sumOm[a] += b2 * On_b;
        if (LAST) {
          p.oW[a] = k >= 1 ? bc.sW + On_b : 0.0;  // L593; flat lid: W = 0 at k = 0
          p.oT[a] = bc.sT + Tnew;
          p.oR[a] = bc.sR + rnew;
        } else {
          if (k >= 1) p.oW[a] = On_b;  // W'' = Omega'' on a flat grid
          p.oT[a] = Tnew;
          p.oR[a] = rnew;
        }
        On_t = On_b;
        thft = thfb;
        thc = bc.thm;
      }
    }
  }
}

template <bool ACC>
static void launch_acc(const AcArgs &p, int mode, cudaStream_t st) {
  constexpr int ROWS = 4;
  dim3 block(32, ROWS), grid((p.nx + 31) / 32, (p.ny + ROWS - 1) / ROWS);
  switch (mode) {
    case 0: k_acoustic_flat<ROWS, 0, ACC><<<grid, block, 0, st>>>(p); break;
    case MODE_FIRST: k_acoustic_flat<ROWS, MODE_FIRST, ACC><<<grid, block, 0, st>>>(p); break;
    case MODE_LAST: k_acoustic_flat<ROWS, MODE_LAST, ACC><<<grid, block, 0, st>>>(p); break;
    case MODE_FIRST | MODE_LAST: k_acoustic_flat<ROWS, MODE_FIRST | MODE_LAST, ACC><<<grid, block, 0, st>>>(p); break;
    default: k_acoustic_flat<ROWS, MODE_FIRST | MODE_LAST | MODE_ZERO, ACC><<<grid, block, 0, st>>>(p); break;
  }
}

void launch_acoustic_flat_one(const AcArgs &p, int mode, cudaStream_t st) {
  if (p.sumU) launch_acc<true>(p, mode, st);
  else launch_acc<false>(p, mode, st);
}

}  // namespace erfb
