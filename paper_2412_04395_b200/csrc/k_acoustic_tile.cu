// k_acoustic_tile.cu -- one acoustic substep (Appendix A; L138-L144) on flat grids with the
// column scratch kept on chip: no HBM round trip between the elimination and the back-substitution.
//
// Mapping.  A CTA owns a tile of 32 consecutive columns in x (one 256-byte row per level and field) and ALL levels.
// Its NW warps split the levels into contiguous chunks; lane = column.  Three phases, separated by CTA barriers:
//
//   1. all warps, levels in parallel: the explicit horizontal momenta U'', V'' (L585 rows 1-2; the +x / +y
//      neighbours' values recomputed, no exchange), the explicit parts Theta~, rho~ of Theta'' and rho'' (rows 4-5),
//      and row k of the tridiagonal system for Omega'' (row 3), already divided by its pivot:
//          e_k = A_k / (D_k - A_k c'_{k-1}),   r_k = rhs_k / (D_k - A_k c'_{k-1})
//      with the Thomas factor c' of the stage read from HBM (it depends on the stage state and dtau only, so the
//      first substep of a stage -- template flag WCP -- computes and stores it).  e, r and c' go to shared memory;
//      Theta~ and rho~ are parked in the output arrays, which the same thread re-reads in phase 3 while the lines
//      are still in L2 (a tile's footprint is 64 KB and it lives for some ten microseconds).
//   2. one warp: d_k = r_k - e_k d_{k-1} upward, Omega''_k = d_k - c'_k Omega''_{k+1} downward: two chains of one
//      dependent fused multiply-add per level, operands from shared memory.
//   3. all warps, levels in parallel: back-substitution of Theta'' and rho'' (rows 4-5 with the new Omega''),
//      the RK stage result S^t + S'' where the launch is the last substep of a stage (L593), the flat lids.
//
// A warp's first level needs the time-weighted Theta^, rho^ of the level below, which another warp computes: the
// row is finished after the first barrier from a two-value exchange slot per warp.
//
// Stage combine (MODE bits), Theta''_d at load time and the buffer roles are those of k_fused_acoustic.cu, whose
// driver (k_fused.cu) serves both kernels.
//
// Algorithmic HBM traffic per cell per substep: reads U'', V'', W'', rho'', Theta'', Theta''_prev, the five slow
// tendencies, theta^t, pi^t, 1/Theta^t, c' (15); writes U'', V'', W'', rho'', Theta'' (5).
#include "acoustic_args.cuh"

namespace erfb {
namespace actile {

constexpr int NW = 8;      // warps per CTA
constexpr int CW = 32;     // columns per CTA

__host__ __device__ constexpr size_t smem_bytes(int nz) { return ((size_t)3 * nz * CW + 2 * NW * CW) * sizeof(double); }
constexpr size_t MAX_SMEM = 226 * 1024;  // dynamic shared memory the kernels opt in to

// right-hand side of row k (S5): c1 = gamma Rd pi_f / hw, Bf = B_f(k), (.)_m = level k-1
__device__ __forceinline__ double row_rhs(double om_b, double RW, double c1, double Bf, double That, double That_m,
                                          double iT, double iT_m, double rhat, double rhat_m, double dtau, double g) {
  return om_b + dtau * (RW - c1 * (That - That_m) + g * Bf * 0.5 * (That * iT + That_m * iT_m) - g * 0.5 * (rhat + rhat_m));
}

template <int MODE, bool WCP>
__global__ void __launch_bounds__(32 * NW, 2) k_acoustic_tile(const AcArgs p, const int chunk) {
  constexpr bool FIRST = (MODE & MODE_FIRST) != 0, LAST = (MODE & MODE_LAST) != 0, ZERO = (MODE & MODE_ZERO) != 0;
  extern __shared__ __align__(16) double sm[];
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  double *const s_e = sm, *const s_r = sm + (size_t)nz * CW, *const s_c = sm + (size_t)2 * nz * CW;
  double *const s_x = sm + (size_t)3 * nz * CW;  // [NW][2][CW] exchange of (Theta^, rho^) across chunk boundaries

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int i = blockIdx.x * CW + lane, j = blockIdx.y;
  const bool act = i < nx;
  const int ii = act ? i : nx - 1;
  const int im = ii == 0 ? nx - 1 : ii - 1, ip = ii == nx - 1 ? 0 : ii + 1;
  const int jm = j == 0 ? ny - 1 : j - 1, jp = j == ny - 1 ? 0 : j + 1;
  const size_t plane = (size_t)nx * ny;
  const size_t oc = (size_t)j * nx + ii, oxm = (size_t)j * nx + im, oxp = (size_t)j * nx + ip;
  const size_t oym = (size_t)jm * nx + ii, oyp = (size_t)jp * nx + ii;

  const double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW;
  const double *__restrict__ Rrho = p.Rrho, *__restrict__ RTh = p.RTh;
  const double *__restrict__ theta = p.theta, *__restrict__ pi = p.pi, *__restrict__ iTf = p.iT;
  const double *__restrict__ rdz = p.rdz, *__restrict__ rhwt = p.rhw, *__restrict__ tabB = p.tabB;

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

  const int k0 = w * chunk, k1 = min(nz, k0 + chunk);
  const bool work = act && k0 < nz;

  // ------------------------------------------------------------------ phase 1: explicit parts and scaled rows
  // first row of the chunk, finished after the exchange
  double f_om = 0.0, f_RW = 0.0, f_c1 = 0.0, f_Bf = 0.0, f_That = 0.0, f_iT = 0.0, f_iTm = 0.0, f_rhat = 0.0, f_scale = 0.0;
  if (work) {
    double pi_m = 0.0;                 // pi^t at level k-1
    double thf_b = 0.0, thf_bm = 0.0;  // theta^t at w-faces k and k-1
    double iT_m = 0.0, rT_m = 0.0, rhc_m = 0.0;
    double That_m = 0.0, rhat_m = 0.0;
    double om_b = 0.0;                 // Omega''(k) = W''(k) at the end of the previous substep (0 on the lid)
    double th_c = theta[(size_t)k0 * plane + oc];
    if (k0 >= 1) {
      const size_t am = (size_t)(k0 - 1) * plane + oc;
      pi_m = pi[am];
      iT_m = iTf[am];
      rhc_m = rdz[k0 - 1];
      rT_m = rhc_m * iT_m;
      const double th_m = theta[am];
      thf_b = 0.5 * (th_m + th_c);
      if (k0 >= 2) thf_bm = 0.5 * (theta[am - plane] + th_m);
      om_b = pert(WW, p.Pw, am + plane);
    }
    struct In {
      double T_c, d_c, d_xm, d_xp, d_ym, d_yp, pi_c, pi_xm, pi_xp, pi_ym, pi_yp, th_xm, th_xp, th_ym, th_yp;
      double U_c, U_xp, RU_c, RU_xp, V_c, V_yp, RV_c, RV_yp, th_t, om_t, RW_c, rpp, RTh_c, Rrho_c, iT, cpm, sU, sV;
    };
    auto load = [&](int k, In &q) {
      const size_t kk = (size_t)k * plane;
      const size_t a = kk + oc, axm = kk + oxm, axp = kk + oxp, aym = kk + oym, ayp = kk + oyp;
      const bool top = k + 1 >= nz;
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
      q.th_t = top ? 0.0 : theta[a + plane];
      q.om_t = top ? 0.0 : pert(WW, p.Pw, a + plane);
      q.RW_c = RW[a]; q.rpp = pert(RHO, p.Pr, a); q.RTh_c = RTh[a]; q.Rrho_c = Rrho[a]; q.iT = iTf[a];
      q.cpm = (!WCP && k >= 2) ? p.cp_scr[a - plane] : 0.0;  // c'_{k-1}
      q.sU = LAST ? p.St[UU][a] : 0.0;
      q.sV = LAST ? p.St[VV][a] : 0.0;
    };
    In cur;
#pragma unroll 1
    for (int k = k0; k < k1; k++) {
      load(k, cur);
      const size_t a = (size_t)k * plane + oc;
      const bool top = k + 1 >= nz;
      const double T_c = cur.T_c, d_c = cur.d_c, d_xm = cur.d_xm, d_xp = cur.d_xp, d_ym = cur.d_ym, d_yp = cur.d_yp;
      const double pi_c = cur.pi_c, pi_xm = cur.pi_xm, pi_xp = cur.pi_xp, pi_ym = cur.pi_ym, pi_yp = cur.pi_yp;
      const double th_xm = cur.th_xm, th_xp = cur.th_xp, th_ym = cur.th_ym, th_yp = cur.th_yp;
      const double U_c = cur.U_c, U_xp = cur.U_xp, RU_c = cur.RU_c, RU_xp = cur.RU_xp;
      const double V_c = cur.V_c, V_yp = cur.V_yp, RV_c = cur.RV_c, RV_yp = cur.RV_yp;
      const double th_t = cur.th_t, om_t = cur.om_t, RW_c = cur.RW_c, rpp = cur.rpp, RTh_c = cur.RTh_c, Rrho_c = cur.Rrho_c;
      const double iT = cur.iT, cpm = cur.cpm;
      // explicit horizontal momenta (L585 rows 1-2) at the four faces of the column
      const double Um = U_c + dtau * RU_c - cU * (pi_xm + pi_c) * (d_c - d_xm);
      const double Up = U_xp + dtau * RU_xp - cU * (pi_c + pi_xp) * (d_xp - d_c);
      const double Vm = V_c + dtau * RV_c - cV * (pi_ym + pi_c) * (d_c - d_ym);
      const double Vp = V_yp + dtau * RV_yp - cV * (pi_c + pi_yp) * (d_yp - d_c);
      p.oU[a] = LAST ? cur.sU + Um : Um;
      p.oV[a] = LAST ? cur.sV + Vm : Vm;
      if (FIRST && !LAST && !ZERO) p.oTp[a] = d_c;  // Theta''_prev of the next substep
      // explicit parts of Theta'' and rho'' (L585 rows 4-5 with the old-time part of the W'' average)
      const double thf_t = top ? 0.0 : 0.5 * (th_c + th_t);
      const double rhc = rdz[k];
      const double DhT = (Up * (th_c + th_xp) - Um * (th_xm + th_c)) * hx + (Vp * (th_c + th_yp) - Vm * (th_ym + th_c)) * hy;
      const double Dh = (Up - Um) * p.rdx + (Vp - Vm) * p.rdy;
      const double Ttil = T_c + dtau * (RTh_c - DhT - b1 * (thf_t * om_t - thf_b * om_b) * rhc);
      const double rtil = rpp + dtau * (Rrho_c - Dh - b1 * (om_t - om_b) * rhc);
      const double That = b2 * Ttil + b1 * T_c, rhat = b2 * rtil + b1 * rpp;
      p.kT[a] = Ttil;  // parked (L2) until phase 3
      p.kR[a] = rtil;
      const double rT = rhc * iT;
      if (k >= 1) {
        // row k of the tridiagonal system for Omega''new (S5)
        const double pif = 0.5 * (pi_m + pi_c);
        const double rhw = rhwt[k];
        const double Bf = tabB[k] * pif;
        const double c1 = gR * pif * rhw;
        const double a1 = s * c1, bB = sg2 * Bf;
        double Ac = sg2 * rhc_m - thf_bm * (a1 * rhc_m + bB * rT_m);
        const double Dc = 1.0 + thf_b * (a1 * (rhc + rhc_m) - bB * (rT - rT_m)) + sg2 * (rhc - rhc_m);
        if (k == 1) Ac = 0.0;
        double scale = 1.0;
        if (WCP) {
          double Cc = thf_t * (bB * rT - a1 * rhc) - sg2 * rhc;
          if (k == nz - 1) Cc = 0.0;
          s_e[k * CW + lane] = Ac;
          s_c[k * CW + lane] = Dc;
          p.cp_scr[a] = Cc;  // parked; the solving warp replaces it by c'_k
        } else {
          scale = 1.0 / (Dc - Ac * cpm);
          s_e[k * CW + lane] = Ac * scale;
          s_c[(k - 1) * CW + lane] = cpm;
        }
        if (k == k0) {
          f_om = om_b; f_RW = RW_c; f_c1 = c1; f_Bf = Bf; f_That = That; f_iT = iT; f_iTm = iT_m; f_rhat = rhat;
          f_scale = scale;
        } else {
          s_r[k * CW + lane] = scale * row_rhs(om_b, RW_c, c1, Bf, That, That_m, iT, iT_m, rhat, rhat_m, dtau, g);
        }
      }
      pi_m = pi_c;
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
    s_x[(w * 2 + 0) * CW + lane] = That_m;
    s_x[(w * 2 + 1) * CW + lane] = rhat_m;
  }
  __syncthreads();
  if (work && k0 >= 1) {
    const double That_m = s_x[((w - 1) * 2 + 0) * CW + lane], rhat_m = s_x[((w - 1) * 2 + 1) * CW + lane];
    s_r[k0 * CW + lane] = f_scale * row_rhs(f_om, f_RW, f_c1, f_Bf, f_That, That_m, f_iT, f_iTm, f_rhat, rhat_m, dtau, g);
  }
  __syncthreads();

  // ------------------------------------------------------------------ phase 2: the two recurrences, one warp
  if (w == 0 && act) {
    double d = 0.0;
    if (WCP) {
      double cp = 0.0;
#pragma unroll 4
      for (int k = 1; k < nz; k++) {
        const size_t a = (size_t)k * plane + oc;
        const double Ac = s_e[k * CW + lane];
        const double minv = 1.0 / (s_c[k * CW + lane] - Ac * cp);
        cp = p.cp_scr[a] * minv;
        d = (s_r[k * CW + lane] - Ac * d) * minv;
        s_r[k * CW + lane] = d;
        s_c[k * CW + lane] = cp;
        p.cp_scr[a] = cp;
      }
    } else {
#pragma unroll 8
      for (int k = 1; k < nz; k++) {
        d = fma(-s_e[k * CW + lane], d, s_r[k * CW + lane]);
        s_r[k * CW + lane] = d;
      }
    }
    // Omega''_{nz-1} = d_{nz-1} (Omega''_nz = 0 on the lid)
    double On = d;
#pragma unroll 8
    for (int k = nz - 2; k >= 1; k--) {
      On = fma(-s_c[k * CW + lane], On, s_r[k * CW + lane]);
      s_r[k * CW + lane] = On;
    }
  }
  __syncthreads();

  // ------------------------------------------------------------------ phase 3: back-substitution, stage result
  if (work) {
    const double cb = dtau * b2;
    double th_m = k0 >= 1 ? theta[(size_t)(k0 - 1) * plane + oc] : 0.0;
    double th_c = theta[(size_t)k0 * plane + oc];
    double On_b = k0 >= 1 ? s_r[k0 * CW + lane] : 0.0;
    double thfb = k0 >= 1 ? 0.5 * (th_m + th_c) : 0.0;
#pragma unroll 2
    for (int k = k0; k < k1; k++) {
      const size_t a = (size_t)k * plane + oc;
      const bool top = k + 1 >= nz;
      const double th_t = top ? 0.0 : theta[a + plane];
      const double On_t = top ? 0.0 : s_r[(k + 1) * CW + lane];
      const double thft = top ? 0.0 : 0.5 * (th_c + th_t);
      const double rhc = rdz[k];
      const double Tnew = p.kT[a] - cb * (thft * On_t - thfb * On_b) * rhc;
      const double rnew = p.kR[a] - cb * (On_t - On_b) * rhc;
      if (LAST) {
        p.oW[a] = k >= 1 ? p.St[WW][a] + On_b : 0.0;  // L593; flat lid: W = 0 at k = 0
        p.oT[a] = p.St[TH][a] + Tnew;
        p.oR[a] = p.St[RHO][a] + rnew;
        if (top) p.oW[a + plane] = 0.0;               // and at k = nz
      } else {
        if (k >= 1) p.oW[a] = On_b;  // W'' = Omega'' on a flat grid
        p.oT[a] = Tnew;
        p.oR[a] = rnew;
      }
      th_c = th_t;
      thfb = thft;
      On_b = On_t;
    }
  }
}

template <int MODE>
static void launch_mode(const AcArgs &p, dim3 grid, int chunk, size_t smem, cudaStream_t st) {
  void (*kern)(AcArgs, int) = p.write_cp ? k_acoustic_tile<MODE, true> : k_acoustic_tile<MODE, false>;
  static OncePerDevice once;  // the opt-in covers every nz acoustic_tile_selected admits; the launch asks for what it uses
  once.run([] {
    cudaFuncSetAttribute(k_acoustic_tile<MODE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MAX_SMEM);
    cudaFuncSetAttribute(k_acoustic_tile<MODE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)MAX_SMEM);
  });
  kern<<<grid, 32 * NW, smem, st>>>(p, chunk);
}

}  // namespace actile

// Which substep kernel.  Splitting the levels of a column over the warps of a CTA exposes nz / 16 times more parallelism
// per column than one thread per column, which wins while the grid has too few columns to fill the machine (measured on
// B200, substeps per RK3 step: 32x32x32 0.15 against 0.39 ms, 128x128x64 0.74 against 1.44 ms).  On large grids the
// thread-per-column kernel is faster (256x256x128: 3.9 against 6.6 ms; 1024x1024x128: 59.1 against 104.6 ms per step)
// although it moves 27 % more bytes: both kernels are bound by load latency at 16 warps per SM, and the tile kernel adds
// two barriers, a single-warp phase and a second pass over its levels (profiles/r2_substep_experiments.md; addressing the
// fields as [j][k][i] instead of [k][j][i] does not change its time, so the layout is not the reason).
// Developer knobs: ERF_VARIANT_FORCE_TILE / _FORCE_COLUMN.
bool acoustic_tile_selected(const erf_ctx *c) {
  if (!c->fz || !c->fz->ok || (c->fz->variant & ERF_VARIANT_FORCE_COLUMN)) return false;
  if (actile::smem_bytes(c->nz) > actile::MAX_SMEM) return false;  // 3 nz rows of 32 columns: nz <= 290
  if (c->fz->variant & ERF_VARIANT_FORCE_TILE) return true;
  return (long long)c->nx * c->ny <= 32768;
}

void launch_acoustic_tile_one(const AcArgs &p, int mode, cudaStream_t st) {
  using namespace actile;
  dim3 grid((p.nx + CW - 1) / CW, p.ny);
  const int chunk = (p.nz + NW - 1) / NW;
  const size_t smem = smem_bytes(p.nz);
  switch (mode) {
    case 0: launch_mode<0>(p, grid, chunk, smem, st); break;
    case MODE_FIRST: launch_mode<MODE_FIRST>(p, grid, chunk, smem, st); break;
    case MODE_LAST: launch_mode<MODE_LAST>(p, grid, chunk, smem, st); break;
    case MODE_FIRST | MODE_LAST: launch_mode<MODE_FIRST | MODE_LAST>(p, grid, chunk, smem, st); break;
    default: launch_mode<MODE_FIRST | MODE_LAST | MODE_ZERO>(p, grid, chunk, smem, st); break;
  }
}

}  // namespace erfb
