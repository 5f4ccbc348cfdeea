// k_acoustic_zc.cu -- one acoustic substep (Appendix A; L138-L144) on flat grids
// with the column tridiagonal solve split into z-chunks, so that NOTHING is parked in HBM between
// the forward and backward sweeps, and with the RK stage combine (L581, L593) folded in.
//
// Mapping.  A CTA owns CW consecutive columns in x of one row j and ALL nz levels.  Thread
// (x, c) owns levels [c*M, c*M+M) of column x ("z-chunk" c; ZC = ceil(nz/M) chunks).  Lanes run
// along x, so every global access is a contiguous 8*CW-byte segment.
//
//   phase A  (all chunks in parallel)  explicit horizontal momenta U'', V'' (L585 rows 1-2) -> HBM;
//            explicit parts Theta~, rho~ of Theta'', rho'' -> shared; rows of the tridiagonal system
//            for Omega'' (S5) of the chunk's interior faces, eliminated upward on the fly
//            with TWO right-hand sides: the true one (y') and the coupling to the chunk's own bottom
//            face (v'), as in the partition method for tridiagonal systems:
//                x_r = y'_r - v'_r * xs_c - c'_r * x_{r+1},   x_M = xs_{c+1}
//            where xs_c = Omega'' at the chunk's bottom face c*M (the "separator" unknowns).
//   phase B  each chunk reduces its separator row with the end values of the chunk below and its own
//            interior to one row of a ZC x ZC tridiagonal system; chunk 0's threads solve it (Thomas).
//   phase C  back-substitution inside each chunk from the separator values, the implicit parts of
//            rho'' and Theta'', stores.
//
// The elimination order differs from a single Thomas sweep only in rounding (the matrix is strictly
// diagonally dominant: off-diagonals ~ (c dtau/dz)^2 b2^2 against 1 + 2 (c dtau/dz)^2 b2^2) [R:G22].
//
// Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev) (L144) [R:G6] is formed at load time from the
// current and the previous Theta'' (three rotating buffers), so a substep reads U'',V'',W'',rho'',
// Theta'',Theta''_prev, the 5 slow tendencies and theta^t, pi^t, 1/Theta^t (14 doubles per cell) and
// writes U'',V'',W'',rho'',Theta'' (5).
//
// Stage combine.  MODE_FIRST: S'' = S^n - S^t is formed at load time (L581) [R:G7] (MODE_ZERO: RK stage 1,
// S'' = 0, nothing is loaded).  MODE_LAST: the kernel writes S^t + S'' (L593) and the flat lids W = 0.
#include "acoustic_args.cuh"

namespace erfb {

template <int CW, int MODE>
__global__ void __launch_bounds__(512, 1) k_acoustic_zc(const AcArgs p) {
  constexpr bool FIRST = (MODE & MODE_FIRST) != 0, LAST = (MODE & MODE_LAST) != 0, ZERO = (MODE & MODE_ZERO) != 0;
  extern __shared__ double sm[];
  const int nx = p.nx, ny = p.ny, nz = p.nz, M = p.M, ZC = p.ZC;
  const int nzp = ZC * M;
  const int x = threadIdx.x % CW, c = threadIdx.x / CW;
  const int i = blockIdx.x * CW + x, j = blockIdx.y;
  const bool act = i < nx;
  double *cpS = sm, *ypS = cpS + nzp * CW, *vpS = ypS + nzp * CW, *TtS = vpS + nzp * CW, *rtS = TtS + nzp * CW,
         *tfS = rtS + nzp * CW;                       // [nzp][CW]: c', y', v', Theta~, rho~, theta at faces
  double *exT = tfS + nzp * CW, *exr = exT + ZC * CW;  // [ZC][CW]: That, rhat of the chunk's top cell
  double *rA = exr + ZC * CW, *rB = rA + ZC * CW, *rC = rB + ZC * CW, *rD = rC + ZC * CW;  // reduced rows
  double *xsS = rD + ZC * CW;                          // [ZC+1][CW] separator values

  const int ic = act ? i : 0;
  const int im = ic == 0 ? nx - 1 : ic - 1, ip = ic == nx - 1 ? 0 : ic + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const size_t plane = (size_t)nx * ny;
  const size_t oc = (size_t)j * nx + ic, oxm = (size_t)j * nx + im, oxp = (size_t)j * nx + ip;
  const size_t oym = (size_t)jm * nx + ic, oyp = (size_t)jp * nx + ic;

  const double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW;
  const double *__restrict__ Rrho = p.Rrho, *__restrict__ RTh = p.RTh;
  const double *__restrict__ theta = p.theta, *__restrict__ pi = p.pi, *__restrict__ iTf = p.iT;
  const double *__restrict__ rdz = p.rdz, *__restrict__ rhwt = p.rhw, *__restrict__ tabB = p.tabB;

  const double dtau = p.dtau, b1 = p.b1, b2 = p.b2, g = p.g, gR = p.gR, beta_d = p.beta_d;
  const double cU = dtau * gR * 0.5 * p.rdx, cV = dtau * gR * 0.5 * p.rdy;
  const double hx = 0.5 * p.rdx, hy = 0.5 * p.rdy;
  const double s = dtau * dtau * b2 * b2;
  const double sg2 = s * g * 0.5;
  const double cb = dtau * b2;

  // S'' at one point (L581): 0 in RK stage 1, S^n - S^t at the first substep of a stage, else stored
  auto pert = [&](int f, const double *__restrict__ P, size_t a) -> double {
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

  const int k0 = c * M;
  // separator row (face k0) pieces, completed after the exchange with the chunk below
  double sA = 0.0, sC = 0.0, sD = 1.0, s_omb = 0.0, s_RW = 0.0, s_c1 = 0.0, s_c2 = 0.0, s_That = 0.0, s_rhat = 0.0,
         s_iT = 0.0, s_iTm = 0.0;
  bool have_sep = false;
  double y1 = 0.0, v1 = 0.0, w1 = 0.0;

  if (act) {
    // ---------------- phase A1: horizontal part, levels independent ----------------
    // explicit horizontal momenta (L585 rows 1-2) at the four faces of the column; their divergences
    // (parked in shared memory for phase A2 together with pi^t and Theta'' of the own cell)
#pragma unroll 1
    for (int r = 0; r < M; r++) {
      const int k = k0 + r;
      if (k >= nz) break;
      const int sa = k * CW + x;
      const size_t kk = (size_t)k * plane;
      const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
      double Tpp, d_c, d_xm, d_xp, d_ym, d_yp, U_c, U_xp, V_c, V_yp;
      if (ZERO) {
        Tpp = d_c = d_xm = d_xp = d_ym = d_yp = U_c = U_xp = V_c = V_yp = 0.0;
      } else if (FIRST) {
        const double *__restrict__ nT = p.Sn[TH], *__restrict__ tT = p.St[TH];
        const double n0 = nT[a], n1 = nT[axm], n2 = nT[axp], n3 = nT[aym], n4 = nT[ayp];
        const double t0 = tT[a], t1 = tT[axm], t2 = tT[axp], t3 = tT[aym], t4 = tT[ayp];
        const double un0 = p.Sn[UU][a], un1 = p.Sn[UU][axp], ut0 = p.St[UU][a], ut1 = p.St[UU][axp];
        const double vn0 = p.Sn[VV][a], vn1 = p.Sn[VV][ayp], vt0 = p.St[VV][a], vt1 = p.St[VV][ayp];
        Tpp = d_c = n0 - t0; d_xm = n1 - t1; d_xp = n2 - t2; d_ym = n3 - t3; d_yp = n4 - t4;
        U_c = un0 - ut0; U_xp = un1 - ut1; V_c = vn0 - vt0; V_yp = vn1 - vt1;
      } else {
        const double *__restrict__ cT = p.Pt, *__restrict__ pT = p.Ptp;
        const double n0 = cT[a], n1 = cT[axm], n2 = cT[axp], n3 = cT[aym], n4 = cT[ayp];
        const double t0 = pT[a], t1 = pT[axm], t2 = pT[axp], t3 = pT[aym], t4 = pT[ayp];
        U_c = p.Pu[a]; U_xp = p.Pu[axp]; V_c = p.Pv[a]; V_yp = p.Pv[ayp];
        Tpp = n0;  // Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev) (L144) [R:G6]
        d_c = n0 + beta_d * (n0 - t0); d_xm = n1 + beta_d * (n1 - t1); d_xp = n2 + beta_d * (n2 - t2);
        d_ym = n3 + beta_d * (n3 - t3); d_yp = n4 + beta_d * (n4 - t4);
      }
      const double pi_c = pi[a], pi_xm = pi[axm], pi_xp = pi[axp], pi_ym = pi[aym], pi_yp = pi[ayp];
      const double th_c = theta[a], th_xm = theta[axm], th_xp = theta[axp], th_ym = theta[aym], th_yp = theta[ayp];
      const double ru_c = RU[a], ru_xp = RU[axp], rv_c = RV[a], rv_yp = RV[ayp];
      double su = 0.0, sv = 0.0;
      if (LAST) { su = p.St[UU][a]; sv = p.St[VV][a]; }
      const double Um = U_c + dtau * ru_c - cU * (pi_xm + pi_c) * (d_c - d_xm);
      const double Up = U_xp + dtau * ru_xp - cU * (pi_c + pi_xp) * (d_xp - d_c);
      const double Vm = V_c + dtau * rv_c - cV * (pi_ym + pi_c) * (d_c - d_ym);
      const double Vp = V_yp + dtau * rv_yp - cV * (pi_c + pi_yp) * (d_yp - d_c);
      const double DhT = (Up * (th_c + th_xp) - Um * (th_xm + th_c)) * hx + (Vp * (th_c + th_yp) - Vm * (th_ym + th_c)) * hy;
      const double Dh = (Up - Um) * p.rdx + (Vp - Vm) * p.rdy;
      p.oU[a] = LAST ? su + Um : Um;
      p.oV[a] = LAST ? sv + Vm : Vm;
      if (FIRST && !LAST && !ZERO) p.oTp[a] = d_c;  // Theta''_prev of the next substep
      TtS[sa] = DhT; rtS[sa] = Dh; cpS[sa] = pi_c; ypS[sa] = Tpp;
    }
    // ---------------- phase A2: vertical part, marching upward through the chunk ----------------
    struct Lv {  // what one level needs from global memory
      double om_t, rpp, RTh, Rrho, RW, iT, th_t, rdz, rhw, tabB;
    };
    auto load_lv = [&](int k, Lv &q) {
      const int kc = min(k, nz - 1);
      const size_t a = (size_t)kc * plane + oc;
      const bool top = kc + 1 >= nz;
      const size_t at = top ? a : a + plane;
      q.om_t = pert(WW, p.Pw, at);
      q.th_t = theta[at];
      q.rpp = pert(RHO, p.Pr, a);
      q.RTh = RTh[a]; q.Rrho = Rrho[a]; q.RW = RW[a]; q.iT = iTf[a];
      q.rdz = rdz[kc]; q.rhw = rhwt[kc]; q.tabB = tabB[kc];
    };
    double th_c = 0.0, thf_b = 0.0, om_b = 0.0;
    double pi_m = 0.0, iT_m = 0.0, rT_m = 0.0, rhc_m = 0.0, That_m = 0.0, rhat_m = 0.0, thf_bm = 0.0;
    double cp_m = 0.0, yp_m = 0.0, vp_m = 0.0;
    Lv cur, nxt;
    if (k0 < nz) {
      load_lv(k0, cur);
      th_c = theta[(size_t)k0 * plane + oc];
      if (k0 >= 1) {
        const size_t am = (size_t)(k0 - 1) * plane + oc;
        const double th_m = theta[am];
        thf_b = 0.5 * (th_m + th_c);
        om_b = pert(WW, p.Pw, am + plane);
        pi_m = pi[am];
        iT_m = iTf[am];
        rhc_m = rdz[k0 - 1];
        rT_m = rhc_m * iT_m;
        thf_bm = k0 >= 2 ? 0.5 * (theta[am - plane] + th_m) : 0.0;
      }
    }
#pragma unroll 1
    for (int r = 0; r < M; r++) {
      const int k = k0 + r;
      const int sa = k * CW + x;
      if (k >= nz) {  // padding levels: identity rows, Omega'' = 0
        cpS[sa] = 0.0; ypS[sa] = 0.0; vpS[sa] = 0.0; TtS[sa] = 0.0; rtS[sa] = 0.0; tfS[sa] = 0.0;
        continue;
      }
      if (r + 1 < M) load_lv(k + 1, nxt);  // software pipeline: the next level's loads fly during this level's math
      const bool top = k + 1 >= nz;
      const double DhT = TtS[sa], Dh = rtS[sa], pi_c = cpS[sa], Tpp = ypS[sa];
      const double om_t = top ? 0.0 : cur.om_t;
      const double rpp = cur.rpp, iT = cur.iT, rhc = cur.rdz;
      // explicit parts of Theta'' and rho'' (L585 rows 4-5 with the old-time part of the Omega'' average)
      const double thf_t = top ? 0.0 : 0.5 * (th_c + cur.th_t);
      const double Ttil = Tpp + dtau * (cur.RTh - DhT - b1 * (thf_t * om_t - thf_b * om_b) * rhc);
      const double rtil = rpp + dtau * (cur.Rrho - Dh - b1 * (om_t - om_b) * rhc);
      const double That = b2 * Ttil + b1 * Tpp, rhat = b2 * rtil + b1 * rpp;
      const double rT = rhc * iT;
      TtS[sa] = Ttil;
      rtS[sa] = rtil;
      tfS[sa] = thf_b;
      if (k >= 1) {
        // row k of the tridiagonal system for Omega''new (S5)
        const double pif = 0.5 * (pi_m + pi_c);
        const double rhw = cur.rhw;
        const double Bf = cur.tabB * pif;
        const double a1 = s * gR * pif * rhw, bB = sg2 * Bf;
        double Cc = thf_t * (bB * rT - a1 * rhc) - sg2 * rhc;
        double Ac = sg2 * rhc_m - thf_bm * (a1 * rhc_m + bB * rT_m);
        const double Dc = 1.0 + thf_b * (a1 * (rhc + rhc_m) - bB * (rT - rT_m)) + sg2 * (rhc - rhc_m);
        if (k == nz - 1) Cc = 0.0;
        if (k == 1) Ac = 0.0;
        const double rw = cur.RW;
        if (r == 0) {  // separator: That, rhat of the cell below arrive through shared memory
          sA = Ac; sC = Cc; sD = Dc; s_omb = om_b; s_RW = rw; s_c1 = gR * pif * rhw; s_c2 = g * Bf * 0.5;
          s_That = That; s_rhat = rhat; s_iT = iT; s_iTm = iT_m;
          have_sep = true;
        } else {
          const double rhs = om_b + dtau * (rw - gR * pif * rhw * (That - That_m) +
                                            g * Bf * 0.5 * (That * iT + That_m * iT_m) - g * 0.5 * (rhat + rhat_m));
          const double minv = 1.0 / (Dc - Ac * cp_m);
          cp_m = Cc * minv;
          yp_m = (rhs - Ac * yp_m) * minv;
          vp_m = (r == 1 ? Ac : -Ac * vp_m) * minv;
          cpS[sa] = cp_m; ypS[sa] = yp_m; vpS[sa] = vp_m;
        }
      }
      if (r == M - 1 || top) {
        exT[c * CW + x] = That;
        exr[c * CW + x] = rhat;
      }
      pi_m = pi_c; th_c = cur.th_t; thf_bm = thf_b; thf_b = thf_t; iT_m = iT; rT_m = rT; rhc_m = rhc;
      That_m = That; rhat_m = rhat; om_b = om_t;
      cur = nxt;
    }
    // interior solution at r = 1 as y1 - v1 xs_c - w1 xs_{c+1} (own shared-memory values only)
    {
      int sa = (k0 + M - 1) * CW + x;
      y1 = ypS[sa]; v1 = vpS[sa]; w1 = cpS[sa];
      for (int r = M - 2; r >= 1; r--) {
        sa -= CW;
        const double cpr = cpS[sa];
        y1 = ypS[sa] - cpr * y1;
        v1 = vpS[sa] - cpr * v1;
        w1 = -cpr * w1;
      }
    }
  }
  __syncthreads();
  // ---------------- phase B: reduced system over the separators ----------------
  if (act) {
    double al = 0.0, be = 1.0, ga = 0.0, de = 0.0;
    if (have_sep) {  // c >= 1 and k0 <= nz-1
      const double That_m = exT[(c - 1) * CW + x], rhat_m = exr[(c - 1) * CW + x];
      const double d_s = s_omb + dtau * (s_RW - s_c1 * (s_That - That_m) + s_c2 * (s_That * s_iT + That_m * s_iTm) -
                                         g * 0.5 * (s_rhat + rhat_m));
      const int se = (k0 - 1) * CW + x;
      const double yE = ypS[se], vE = vpS[se], wE = cpS[se];
      al = -sA * vE;
      be = sD - sA * wE - sC * v1;
      ga = -sC * w1;
      de = d_s - sA * yE - sC * y1;
    }
    rA[c * CW + x] = al; rB[c * CW + x] = be; rC[c * CW + x] = ga; rD[c * CW + x] = de;
  }
  __syncthreads();
  if (act && c == 0) {
    // Thomas over the ZC separator rows (row 0 is the lid: identity)
    double cpm = 0.0, dpm = 0.0;
    for (int q = 0; q < ZC; q++) {
      const int e = q * CW + x;
      const double a_ = rA[e];
      const double minv = 1.0 / (rB[e] - a_ * cpm);
      cpm = rC[e] * minv;
      dpm = (rD[e] - a_ * dpm) * minv;
      rC[e] = cpm;
      rD[e] = dpm;
    }
    double xs = 0.0;
    xsS[ZC * CW + x] = 0.0;
    for (int q = ZC - 1; q >= 0; q--) {
      const int e = q * CW + x;
      xs = rD[e] - rC[e] * xs;
      xsS[e] = xs;
    }
  }
  __syncthreads();
  // ---------------- phase C: back-substitution and the implicit parts ----------------
  if (!act || k0 >= nz) return;
  {
    const double xs_c = xsS[c * CW + x];
    double On_t = xsS[(c + 1) * CW + x];  // Omega''new at the face above the current cell
    const int ktop = min(k0 + M, nz) - 1;
    double thft = (ktop + 1 <= nz - 1) ? tfS[(ktop + 1) * CW + x] : 0.0;
    if (ktop + 1 >= nz) On_t = 0.0;
#pragma unroll 1
    for (int k = ktop; k >= k0; k--) {
      const int sa = k * CW + x;
      const size_t a = (size_t)k * plane + oc;
      const double On_b = (k == k0) ? xs_c : ypS[sa] - vpS[sa] * xs_c - cpS[sa] * On_t;
      const double thfb = tfS[sa];
      const double rhc = rdz[k];
      const double Tnew = TtS[sa] - cb * (thft * On_t - thfb * On_b) * rhc;
      const double rnew = rtS[sa] - cb * (On_t - On_b) * rhc;
      if (LAST) {
        p.oW[a] = k >= 1 ? p.St[WW][a] + On_b : 0.0;  // flat lid: W = 0 at k = 0
        p.oT[a] = p.St[TH][a] + Tnew;
        p.oR[a] = p.St[RHO][a] + rnew;
        if (k == nz - 1) p.oW[a + plane] = 0.0;       // and at k = nz
      } else {
        if (k >= 1) p.oW[a] = On_b;  // W'' = Omega'' on a flat grid
        p.oT[a] = Tnew;
        p.oR[a] = rnew;
      }
      On_t = On_b;
      thft = thfb;
    }
  }
}

// ------------------------------------------------------------------ launch
struct ZcGeom {
  int CW, M, ZC;
  size_t smem;
  bool ok;
};

static ZcGeom zc_geometry(int nz, int variant) {
  ZcGeom gm;
  gm.CW = (variant & 16) ? 32 : 16;
  gm.ok = false;
  for (int M = 8; M <= 32; M *= 2) {
    int ZC = (nz + M - 1) / M;
    while ((ZC * gm.CW) % 32) ZC++;
    if (ZC * gm.CW > 512) continue;
    const size_t smem = ((size_t)6 * ZC * M + 6 * ZC + ZC + 1) * gm.CW * sizeof(double);
    if (smem > 220 * 1024) continue;
    gm.M = M; gm.ZC = ZC; gm.smem = smem; gm.ok = true;
    break;
  }
  return gm;
}

// Which substep kernel: the z-chunked one exposes nz/8 times more parallelism per column, which wins while the grid
// has too few columns to fill the machine with one thread per column (measured on B200: 2.3x faster on 32x32x32,
// 1.8x on 128x128x64, 1.4x slower on 256x256x128 and 1024x1024x128).  Developer knobs: bit 32 forces it, bit 4096
// forces the thread-per-column kernel.
bool acoustic_zc_selected(const erf_ctx *c) {
  if (!c->fz || !c->fz->ok || (c->fz->variant & 4096)) return false;
  if (!zc_geometry(c->nz, c->fz->variant).ok) return false;
  if (c->fz->variant & 32) return true;
  return (long long)c->nx * c->ny <= 32768;
}

template <int CW>
static void zc_launch(const AcArgs &p, int mode, dim3 grid, int threads, size_t smem, cudaStream_t st) {
  void (*kern)(AcArgs) = nullptr;
  switch (mode) {
    case 0: kern = k_acoustic_zc<CW, 0>; break;
    case MODE_FIRST: kern = k_acoustic_zc<CW, MODE_FIRST>; break;
    case MODE_LAST: kern = k_acoustic_zc<CW, MODE_LAST>; break;
    case MODE_FIRST | MODE_LAST: kern = k_acoustic_zc<CW, MODE_FIRST | MODE_LAST>; break;
    default: kern = k_acoustic_zc<CW, MODE_FIRST | MODE_LAST | MODE_ZERO>; break;
  }
  cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  kern<<<grid, threads, smem, st>>>(p);
}

void launch_acoustic_zc_one(const erf_ctx *c, AcArgs &p, int mode, cudaStream_t st) {
  const ZcGeom gm = zc_geometry(c->nz, c->fz->variant);
  p.M = gm.M; p.ZC = gm.ZC;
  dim3 grid((c->nx + gm.CW - 1) / gm.CW, c->ny);
  const int threads = gm.CW * gm.ZC;
  if (gm.CW == 16) zc_launch<16>(p, mode, grid, threads, gm.smem, st);
  else zc_launch<32>(p, mode, grid, threads, gm.smem, st);
}

}  // namespace erfb
