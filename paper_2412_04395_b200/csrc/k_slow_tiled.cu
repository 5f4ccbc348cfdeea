// k_slow_tiled.cu -- the two heavy slow-RHS kernels on flat grids, staged through shared memory.
//
//   k_adv_tiled   advection of (rho, u, v, w, theta) by Eq. 17-21 + pressure
//                 gradient + buoyancy (L84)                                   -> R (5 fields)
//   k_diff_tiled  R_U,V,W -= div(tau), R_Theta -= div(F)  (Eq. 2-3, Eq. 9)
//
// A CTA of 32 x 8 threads owns 32 x 8 columns and a range of levels; each thread marches its column
// upward.  Vertical stencils live in per-thread register windows, vertical face fluxes are computed
// once and carried to the cell above; everything a thread needs from its horizontal neighbours at
// level k comes from shared-memory plane tiles (tiles.cuh) that cp.async fills one level ahead of the
// arithmetic (three stages: level k in use, k+1 and k+2 in flight; one __syncthreads per level).  The thread's own column values for the
// levels above (k+3, k+4) are loaded straight from global memory one iteration before first use.
//
// Level ranges (grid.z chunks) let small grids fill the machine: a chunk starting at k0 > 0 first runs
// iteration k0-1 with its stores switched off to build the values carried from the level below.
#include "slow_flat.cuh"
#include "tiles.cuh"

namespace erfb {

using GB = TileG<4, 3>;  // halo 3 (x padded to 4): advected quantities
using GS = TileG<2, 1>;  // halo 1 (x padded to 2)

// ------------------------------------------------------------------ advection + PG + buoyancy
constexpr int NSTAGE = 3;                            // pipeline depth: level k in use, k+1 and k+2 in flight
// doubles per pipeline stage: one halo-3 tile per advected field of the launch, then the U, V, W, p' tiles
// (W tile only with U or V, p' tile with U, V or W)
__host__ __device__ constexpr int adv_stage(int fm) {
  return ((fm & 1) + ((fm >> 1) & 1) + ((fm >> 2) & 1) + ((fm >> 3) & 1)) * GB::SZ +
         (2 + ((fm & 6) ? 1 : 0) + ((fm & 14) ? 1 : 0)) * GS::SZ;
}

// FM = field mask: which tendencies this launch computes.  One launch with all four bits computes everything;
// splitting by field trades re-reading the mass-flux tiles for much lower register pressure per launch.
enum { F_T = 1, F_U = 2, F_V = 4, F_W = 8, F_ALL = 15 };  // F_T: rho and rho*theta; F_W: rho*w with PG_z + buoyancy

template <int OH, int FM>
__global__ void __launch_bounds__(NTHR, FM == F_ALL ? 2 : 3) k_adv_tiled(const SlowFlat p, const int kchunk) {
  constexpr bool DO_T = (FM & F_T) != 0, DO_U = (FM & F_U) != 0, DO_V = (FM & F_V) != 0, DO_W = (FM & F_W) != 0;
  constexpr int ADV_STAGE = adv_stage(FM);
  constexpr int OFF_U = DO_T * GB::SZ, OFF_V = OFF_U + DO_U * GB::SZ, OFF_W = OFF_V + DO_V * GB::SZ, OFF_S = OFF_W + DO_W * GB::SZ;
  constexpr int OFF_MW = OFF_S + 2 * GS::SZ, OFF_MP = OFF_MW + ((DO_U || DO_V) ? GS::SZ : 0);
  extern __shared__ __align__(16) double sm[];
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
  const int nx = p.nx, ny = p.ny, nz = p.nz, ov = p.ov;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + tx, j = y0 + ty;
  const bool act = i < nx && j < ny;
  const size_t plane = (size_t)nx * ny;
  const int k0 = blockIdx.z * kchunk, k1 = min(nz, k0 + kchunk);  // this CTA's cells [k0, k1)
  const int kb = max(k0 - 1, 0);                                  // first iteration (warm-up if k0 > 0)
  const int ke = k1;                                              // last iteration: finishes cell k1-1
  const int kl = min(ke, nz - 1);                                 // last plane that is staged

  ChunkSet<4, 3, FM != F_ALL> cb;
  ChunkSet<2, 1, FM != F_ALL> cs;
  int *tabs = reinterpret_cast<int *>(sm + NSTAGE * ADV_STAGE);
  cb.init(tabs, tid, x0, y0, nx, ny);
  cs.init(tabs + ChunkSet<4, 3>::TAB, tid, x0, y0, nx, ny);
  const double *__restrict__ U = p.U, *__restrict__ V = p.V, *__restrict__ W = p.W, *__restrict__ rho = p.rho;
  const double *__restrict__ th = p.theta, *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w;
  const double *__restrict__ pp = p.pp;
  auto stage_in = [&](int k, int st) {
    double *b = sm + st * ADV_STAGE;
    const size_t kk = (size_t)k * plane;
    if (DO_T) cb.issue(b, th + kk);
    if (DO_U) cb.issue(b + OFF_U, u + kk);
    if (DO_V) cb.issue(b + OFF_V, v + kk);
    if (DO_W) cb.issue(b + OFF_W, w + kk);
    double *s = b + OFF_S;
    cs.issue(s, U + kk);
    cs.issue(s + GS::SZ, V + kk);
    if (DO_U || DO_V) cs.issue(b + OFF_MW, W + kk);
    if (DO_U || DO_V || DO_W) cs.issue(b + OFF_MP, pp + kk);
  };
  stage_in(kb, 0);
  cp_async_commit();
  if (kb + 1 <= kl) stage_in(kb + 1, 1);
  cp_async_commit();

  double *__restrict__ Rrho = p.Rrho, *__restrict__ RU = p.RU, *__restrict__ RV = p.RV;
  double *__restrict__ RW = p.RW, *__restrict__ RTh = p.RTh;
  const double rdx = p.rdx, rdy = p.rdy;
  const size_t oc = act ? (size_t)j * nx + i : 0;
  const int cB = GB::centre(tx, ty), cS = GS::centre(tx, ty);
  constexpr int WB = GB::W, WS = GS::W;

  // vertical register windows at iteration k: cells k-3..k+2 (theta,u,v), faces k-2..k+3 (w)
  double wt[6], wu[6], wv[6], ww[6];
#pragma unroll
  for (int n = 0; n < 6; n++) {
    const int kc = kb + n - 3, kf = kb + n - 2;
    const bool okc = act && kc >= 0 && kc < nz, okf = act && kf >= 0 && kf <= nz;
    const size_t ac = (size_t)(okc ? kc : 0) * plane + oc, af = (size_t)(okf ? kf : 0) * plane + oc;
    wt[n] = (DO_T && okc) ? th[ac] : 0.0;
    wu[n] = (DO_U && okc) ? u[ac] : 0.0;
    wv[n] = (DO_V && okc) ? v[ac] : 0.0;
    ww[n] = (DO_W && okf) ? w[af] : 0.0;
  }
  double fT_b = 0.0, fU_b = 0.0, fV_b = 0.0, om_b = 0.0;  // face fluxes at the bottom of the previous cell
  double HT = 0.0, HU = 0.0, HV = 0.0, Hr = 0.0;          // horizontal parts of the previous cell
  double Gz_m = 0.0;                                      // w flux at centre k-1
  double U_cm = 0.0, U_pm = 0.0, V_cm = 0.0, V_pm = 0.0;  // dz*U(i), dz*U(i+1), dz*V(j), dz*V(j+1) at level k-1
  double pp_m = 0.0, rp_m = 0.0;                          // p', rho' at level k-1
  double om_c = (act && kb >= 1) ? W[(size_t)kb * plane + oc] : 0.0;  // Omega at face k (lid: 0)
  // prefetched one iteration ahead: Omega at face k+1, rho at cell k
  double om_n = (act && kb + 1 <= nz - 1) ? W[(size_t)(kb + 1) * plane + oc] : 0.0;
  double rho_n = (DO_W && act) ? rho[(size_t)kb * plane + oc] : 0.0;

#pragma unroll 1
  for (int k = kb; k <= ke; k++) {
    const int st = (k - kb) % NSTAGE;
    cp_async_wait_but_one();  // level k has landed; level k+1 may still be in flight
    __syncthreads();
    if (k + 2 <= kl) stage_in(k + 2, (k + 2 - kb) % NSTAGE);
    cp_async_commit();
    if (!act) continue;
    const double *__restrict__ sT = sm + st * ADV_STAGE, *__restrict__ sU = sT + OFF_U,
                               *__restrict__ sV = sT + OFF_V, *__restrict__ sW = sT + OFF_W;
    const double *__restrict__ mU = sT + OFF_S, *__restrict__ mV = mU + GS::SZ,
                               *__restrict__ mW = sT + OFF_MW, *__restrict__ mP = sT + OFF_MP;
    const size_t kk = (size_t)k * plane;
    // own-column values for the next iteration (window tops, Omega at face k+2, rho at cell k+1)
    double nt = 0.0, nu_ = 0.0, nv = 0.0, nw = 0.0, om_nn = 0.0, rho_nn = 0.0;
    {
      const int kc = k + 3, kf = k + 4;
      if (kc < nz) {
        const size_t ac = (size_t)kc * plane + oc;
        if (DO_T) nt = th[ac];
        if (DO_U) nu_ = u[ac];
        if (DO_V) nv = v[ac];
      }
      if (DO_W && kf <= nz) nw = w[(size_t)kf * plane + oc];
      if (k + 2 <= nz - 1) om_nn = W[(size_t)(k + 2) * plane + oc];
      if (DO_W && k + 1 < nz) rho_nn = rho[(size_t)(k + 1) * plane + oc];
    }
    // ---- face k: vertical fluxes of theta, u, v (zero on the lids)
    double fT = 0.0, fU = 0.0, fV = 0.0;
    if (k >= 1 && k <= nz - 1) {
      const int ord = vorder(ov, min(k, nz - k));
      if (DO_T) fT = flux_rt(ord, om_c, wt);
      if (DO_U) fU = flux_rt(ord, 0.5 * (mW[cS - 1] + om_c), wu);
      if (DO_V) fV = flux_rt(ord, 0.5 * (mW[cS - WS] + om_c), wv);
    }
    // ---- finish cell k-1
    if (k - 1 >= k0) {
      const size_t am = kk - plane + oc;
      const double rdzm = p.rdz[k - 1];
      if (DO_T) {
        Rrho[am] = -(Hr + (om_c - om_b) * rdzm);
        RTh[am] = -(HT + (fT - fT_b) * rdzm);
      }
      if (DO_U) RU[am] = -(HU + (fU - fU_b) * rdzm);
      if (DO_V) RV[am] = -(HV + (fV - fV_b) * rdzm);
    }
    if (k == nz) {
      if (DO_W) RW[kk + oc] = 0.0;
      continue;
    }
    if (k == ke) continue;  // the cell above belongs to the next chunk
    fT_b = fT; fU_b = fU; fV_b = fV; om_b = om_c;
    // ---- cell k: horizontal flux divergences
    const double U_m1 = mU[cS - 1], U_c = mU[cS], U_p1 = mU[cS + 1];
    const double U_ym = mU[cS - WS], U_pym = mU[cS - WS + 1];
    const double V_m1 = mV[cS - WS], V_c = mV[cS], V_p1 = mV[cS + WS];
    const double V_xm = mV[cS - 1], V_xmp = mV[cS + WS - 1];
    if (DO_T) Hr = (U_p1 - U_c) * rdx + (V_p1 - V_c) * rdy;
    if (DO_T) {
      double q[7];
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sT[cB + n - 3];
      HT = (flux_c<OH>(U_p1, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(U_c, q[0], q[1], q[2], q[3], q[4], q[5])) * rdx;
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sT[cB + (n - 3) * WB];
      HT += (flux_c<OH>(V_p1, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(V_c, q[0], q[1], q[2], q[3], q[4], q[5])) * rdy;
    }
    const double pp_c = (DO_U || DO_V || DO_W) ? mP[cS] : 0.0;
    if (DO_U) {
      double q[7];
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sU[cB + n - 3];
      HU = (flux_c<OH>(0.5 * (U_c + U_p1), q[1], q[2], q[3], q[4], q[5], q[6]) -
            flux_c<OH>(0.5 * (U_m1 + U_c), q[0], q[1], q[2], q[3], q[4], q[5])) * rdx;
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sU[cB + (n - 3) * WB];
      HU += (flux_c<OH>(0.5 * (V_xmp + V_p1), q[1], q[2], q[3], q[4], q[5], q[6]) -
             flux_c<OH>(0.5 * (V_xm + V_c), q[0], q[1], q[2], q[3], q[4], q[5])) * rdy;
      HU += (pp_c - mP[cS - 1]) * rdx;
    }
    if (DO_V) {
      double q[7];
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sV[cB + n - 3];
      HV = (flux_c<OH>(0.5 * (U_pym + U_p1), q[1], q[2], q[3], q[4], q[5], q[6]) -
            flux_c<OH>(0.5 * (U_ym + U_c), q[0], q[1], q[2], q[3], q[4], q[5])) * rdx;
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sV[cB + (n - 3) * WB];
      HV += (flux_c<OH>(0.5 * (V_c + V_p1), q[1], q[2], q[3], q[4], q[5], q[6]) -
             flux_c<OH>(0.5 * (V_m1 + V_c), q[0], q[1], q[2], q[3], q[4], q[5])) * rdy;
      HV += (pp_c - mP[cS - WS]) * rdy;
    }
    // ---- w equation at face k; vertical flux at centre k
    const double om_t = om_n;
    if (DO_W) {
    const double Gz = flux_rt(vorder(ov, min(k + 1, nz - k)), 0.5 * (om_c + om_t), ww);
    const double dzk = p.dz[k];
    const double U_cd = dzk * U_c, U_pd = dzk * U_p1, V_cd = dzk * V_c, V_pd = dzk * V_p1;
    const double rp_c = rho_n - p.rho0[k];
    if (k >= 1) {
      const double rhw = p.rhw[k];
      double q[7];
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sW[cB + n - 3];
      double adv = (flux_c<OH>(0.5 * (U_pm + U_pd), q[1], q[2], q[3], q[4], q[5], q[6]) -
                    flux_c<OH>(0.5 * (U_cm + U_cd), q[0], q[1], q[2], q[3], q[4], q[5])) * rdx;
#pragma unroll
      for (int n = 0; n < 7; n++) q[n] = sW[cB + (n - 3) * WB];
      adv += (flux_c<OH>(0.5 * (V_pm + V_pd), q[1], q[2], q[3], q[4], q[5], q[6]) -
              flux_c<OH>(0.5 * (V_cm + V_cd), q[0], q[1], q[2], q[3], q[4], q[5])) * rdy;
      adv += Gz - Gz_m;
      if (k >= k0) RW[kk + oc] = -adv * rhw - ((pp_c - pp_m) * rhw + p.g * 0.5 * (rp_m + rp_c));
    } else if (k >= k0) {
      RW[kk + oc] = 0.0;
    }
    Gz_m = Gz;
    U_cm = U_cd; U_pm = U_pd; V_cm = V_cd; V_pm = V_pd;
    pp_m = pp_c; rp_m = rp_c;
    }
    om_c = om_t;
    om_n = om_nn;
    rho_n = rho_nn;
    // ---- shift the vertical windows: bring in cell k+3 and face k+4
#pragma unroll
    for (int n = 0; n < 5; n++) {
      if (DO_T) wt[n] = wt[n + 1];
      if (DO_U) wu[n] = wu[n + 1];
      if (DO_V) wv[n] = wv[n + 1];
      if (DO_W) ww[n] = ww[n + 1];
    }
    wt[5] = nt; wu[5] = nu_; wv[5] = nv; ww[5] = nw;
  }
}

// ------------------------------------------------------------------ diffusion
// R_U,V,W -= div(tau), tau = -2 mu (S - 1/3 div u I) (Eq. 9); R_Theta -= div(-K grad theta) (Eq. 3);
// free-slip lids: tau13 = tau23 = 0 and no scalar flux at k = 0, nz (Table C1 "Slip Wall").
__host__ __device__ constexpr int diff_stage(int part) { return ((part & 1) ? 4 : 0) * GS::SZ + ((part & 2) ? 2 : 0) * GS::SZ; }

// PART bits: 1 = momentum (tiles u, v, w, mu), 2 = scalar (tiles theta, K); the two parts share no tile, so
// splitting them costs no traffic and lets the scalar part run at high occupancy.
template <int PART>
__global__ void __launch_bounds__(NTHR, PART == 2 ? 4 : 2) k_diff_tiled(const SlowFlat p, const int kchunk) {
  constexpr bool DO_M = (PART & 1) != 0, DO_S = (PART & 2) != 0;
  constexpr int DIFF_STAGE = diff_stage(PART), OFF_TH = DO_M ? 4 * GS::SZ : 0, OFF_K = OFF_TH + GS::SZ;
  extern __shared__ __align__(16) double sm[];
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + tx, j = y0 + ty;
  const bool act = i < nx && j < ny;
  const size_t plane = (size_t)nx * ny;
  const int k0 = blockIdx.z * kchunk, k1 = min(nz, k0 + kchunk);
  const int kb = max(k0 - 1, 0), ke = k1, kl = min(ke, nz - 1);

  ChunkSet<2, 1> cs;
  cs.init(reinterpret_cast<int *>(sm + NSTAGE * DIFF_STAGE), tid, x0, y0, nx, ny);
  const double *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w, *__restrict__ th = p.theta;
  const double *__restrict__ mu = p.mu, *__restrict__ Kf = p.K;
  auto stage_in = [&](int k, int st) {
    double *b = sm + st * DIFF_STAGE;
    const size_t kk = (size_t)k * plane;
    if (DO_M) {
      cs.issue(b, u + kk);
      cs.issue(b + GS::SZ, v + kk);
      cs.issue(b + 2 * GS::SZ, w + kk + plane);  // w at face k+1
      cs.issue(b + 3 * GS::SZ, mu + kk);
    }
    if (DO_S) {
      cs.issue(b + OFF_TH, th + kk);
      cs.issue(b + OFF_K, Kf + kk);
    }
  };
  stage_in(kb, 0);
  cp_async_commit();
  if (kb + 1 <= kl) stage_in(kb + 1, 1);
  cp_async_commit();

  double *__restrict__ RU = p.RU, *__restrict__ RV = p.RV, *__restrict__ RW = p.RW, *__restrict__ RTh = p.RTh;
  const double rdx = p.rdx, rdy = p.rdy;
  constexpr int WS = GS::W;
  const int c = GS::centre(tx, ty);
  const size_t oc = act ? (size_t)j * nx + i : 0;

  // carried from level k-1 / face k
  double u_cm = 0, u_pm = 0, v_cm = 0, v_pm = 0;                     // u(i), u(i+1), v(j), v(j+1) at k-1
  double mu_cm = 0, mu_xmm = 0, mu_xpm = 0, mu_ymm = 0, mu_ypm = 0;  // mu at k-1: c, xm, xp, ym, yp
  double K_m = 0, th_m = 0, t33_m = 0;
  double t13_b = 0, t23_b = 0, Fz_b = 0;  // bottom face of the previous cell
  double HU = 0, HV = 0, HT = 0;
  // w at face k: c, xm, xp, ym, yp
  double w_c = 0, w_xm = 0, w_xp = 0, w_ym = 0, w_yp = 0;
  if (DO_M && act) {
    const size_t kk = (size_t)kb * plane;
    const int im = pmod(i - 1, nx), ip = pmod(i + 1, nx), jm = pmod(j - 1, ny), jp = pmod(j + 1, ny);
    w_c = w[kk + oc];
    w_xm = w[kk + (size_t)j * nx + im];
    w_xp = w[kk + (size_t)j * nx + ip];
    w_ym = w[kk + (size_t)jm * nx + i];
    w_yp = w[kk + (size_t)jp * nx + i];
  }
  // tendencies of cell k-1 (read one iteration before they are updated) and of face k
  double rU = 0, rV = 0, rT = 0, rW = (DO_M && act && kb >= 1) ? RW[(size_t)kb * plane + oc] : 0.0;

#pragma unroll 1
  for (int k = kb; k <= ke; k++) {
    const int st = (k - kb) % NSTAGE;
    cp_async_wait_but_one();
    __syncthreads();
    if (k + 2 <= kl) stage_in(k + 2, (k + 2 - kb) % NSTAGE);
    cp_async_commit();
    if (!act) continue;
    const double *__restrict__ su = sm + st * DIFF_STAGE, *__restrict__ sv = su + GS::SZ,
                               *__restrict__ sw = su + 2 * GS::SZ, *__restrict__ smu = su + 3 * GS::SZ,
                               *__restrict__ sth = su + OFF_TH, *__restrict__ sK = su + OFF_K;
    const size_t kk = (size_t)k * plane;
    const bool cell = k < nz && k < ke, inner = k >= 1 && k <= nz - 1;
    // tendencies this thread updates in the next iteration
    double rU_n = 0, rV_n = 0, rT_n = 0, rW_n = 0;
    if (cell) {
      if (DO_M) {
        rU_n = RU[kk + oc];
        rV_n = RV[kk + oc];
        if (k + 1 <= nz - 1) rW_n = RW[kk + plane + oc];
      }
      if (DO_S) rT_n = RTh[kk + oc];
    }
    double u_c = 0, u_p = 0, v_c = 0, v_p = 0, mu_c = 0, mu_xm = 0, mu_xp = 0, mu_ym = 0, mu_yp = 0, K_c = 0, th_c = 0;
    if (k < nz) {
      if (DO_M) {
        u_c = su[c]; u_p = su[c + 1]; v_c = sv[c]; v_p = sv[c + WS];
        mu_c = smu[c]; mu_xm = smu[c - 1]; mu_xp = smu[c + 1]; mu_ym = smu[c - WS]; mu_yp = smu[c + WS];
      }
      if (DO_S) { K_c = sK[c]; th_c = sth[c]; }
    }
    // ---- face k: tau13 at (i,k) and (i+1,k), tau23 at (j,k) and (j+1,k), vertical scalar flux
    double t13 = 0, t13p = 0, t23 = 0, t23p = 0, Fz = 0;
    if (inner) {
      const double rhw = p.rhw[k];
      if (DO_S) Fz = -0.5 * (K_m + K_c) * ((th_c - th_m) * rhw);
      if (DO_M) {
      const double S13 = 0.5 * ((u_c - u_cm) * rhw + (w_c - w_xm) * rdx);
      const double S13p = 0.5 * ((u_p - u_pm) * rhw + (w_xp - w_c) * rdx);
      const double S23 = 0.5 * ((v_c - v_cm) * rhw + (w_c - w_ym) * rdy);
      const double S23p = 0.5 * ((v_p - v_pm) * rhw + (w_yp - w_c) * rdy);
      t13 = -2.0 * (0.25 * (mu_xmm + mu_cm + mu_xm + mu_c)) * S13;
      t13p = -2.0 * (0.25 * (mu_cm + mu_xpm + mu_c + mu_xp)) * S13p;
      t23 = -2.0 * (0.25 * (mu_ymm + mu_cm + mu_ym + mu_c)) * S23;
      t23p = -2.0 * (0.25 * (mu_cm + mu_ypm + mu_c + mu_yp)) * S23p;
      }
    }
    // ---- finish cell k-1
    if (k - 1 >= k0) {
      const size_t am = kk - plane + oc;
      const double rdzm = p.rdz[k - 1];
      if (DO_M) {
        RU[am] = rU - (HU + (t13 - t13_b) * rdzm);
        RV[am] = rV - (HV + (t23 - t23_b) * rdzm);
      }
      if (DO_S) RTh[am] = rT - (HT + (Fz - Fz_b) * rdzm);
    }
    if (!cell) continue;
    t13_b = t13; t23_b = t23; Fz_b = Fz;
    // ---- cell k
    if (DO_S) {
      // scalar fluxes through the x- and y-faces
      const double th_xm = sth[c - 1], th_xp = sth[c + 1], th_ym = sth[c - WS], th_yp = sth[c + WS];
      const double K_xm = sK[c - 1], K_xp = sK[c + 1], K_ym = sK[c - WS], K_yp = sK[c + WS];
      const double Fx = -0.5 * (K_xm + K_c) * ((th_c - th_xm) * rdx), Fxp = -0.5 * (K_c + K_xp) * ((th_xp - th_c) * rdx);
      const double Fy = -0.5 * (K_ym + K_c) * ((th_c - th_ym) * rdy), Fyp = -0.5 * (K_c + K_yp) * ((th_yp - th_c) * rdy);
      HT = (Fxp - Fx) * rdx + (Fyp - Fy) * rdy;
      K_m = K_c; th_m = th_c; rT = rT_n;
    }
    if (!DO_M) continue;
    const double u_m = su[c - 1], u_ym = su[c - WS], u_pym = su[c - WS + 1], u_yp = su[c + WS];
    const double v_m = sv[c - WS], v_xm = sv[c - 1], v_xmp = sv[c + WS - 1], v_xp = sv[c + 1];
    const double wt_c = sw[c], wt_xm = sw[c - 1], wt_xp = sw[c + 1], wt_ym = sw[c - WS], wt_yp = sw[c + WS];
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
    const double mu_xmym = smu[c - WS - 1], mu_xpym = smu[c - WS + 1], mu_xmyp = smu[c + WS - 1];
    const double S12 = 0.5 * ((u_c - u_ym) * rdy + (v_c - v_xm) * rdx);
    const double S12yp = 0.5 * ((u_yp - u_c) * rdy + (v_p - v_xmp) * rdx);
    const double S12xp = 0.5 * ((u_p - u_pym) * rdy + (v_xp - v_c) * rdx);
    const double t12 = -2.0 * (0.25 * (mu_xmym + mu_ym + mu_xm + mu_c)) * S12;
    const double t12yp = -2.0 * (0.25 * (mu_xm + mu_c + mu_xmyp + mu_yp)) * S12yp;
    const double t12xp = -2.0 * (0.25 * (mu_ym + mu_xpym + mu_c + mu_xp)) * S12xp;
    HU = (t11c - t11x) * rdx + (t12yp - t12) * rdy;
    HV = (t12xp - t12) * rdx + (t22c - t22y) * rdy;
    if (k >= 1 && k >= k0) RW[kk + oc] = rW - ((t13p - t13) * rdx + (t23p - t23) * rdy + (t33c - t33_m) * p.rhw[k]);
    // carry
    u_cm = u_c; u_pm = u_p; v_cm = v_c; v_pm = v_p;
    mu_cm = mu_c; mu_xmm = mu_xm; mu_xpm = mu_xp; mu_ymm = mu_ym; mu_ypm = mu_yp;
    t33_m = t33c;
    w_c = wt_c; w_xm = wt_xm; w_xp = wt_xp; w_ym = wt_ym; w_yp = wt_yp;
    rU = rU_n; rV = rV_n; rW = rW_n;
  }
}

// ------------------------------------------------------------------ Smagorinsky viscosity
// mu = rho nu + mu_t, K = rho alpha + mu_t / Pr_t; mu_t = rho (Cs Delta)^2 |S| (Eq. 9) [R:G9,G10].
// Cell k needs u, v of levels k-1, k, k+1 and w of faces k, k+1 with a halo of one column: a ring of five
// stages (stage L = u(L), v(L), w(face L+1)) holds levels k-1..k+1 while k+2 and k+3 are in flight.
constexpr int VISC_NST = 5, VISC_STAGE = 3 * GS::SZ;

__global__ void __launch_bounds__(NTHR, 4) k_visc_tiled(const SlowFlat p, const int kchunk) {
  extern __shared__ __align__(16) double sm[];
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * TX + tx;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + tx, j = y0 + ty;
  const bool act = i < nx && j < ny;
  const size_t plane = (size_t)nx * ny;
  const int k0 = blockIdx.z * kchunk, k1 = min(nz, k0 + kchunk);  // this CTA's cells [k0, k1)
  const int Lb = k0 - 1, Le = min(k1, nz - 1);                    // stages Lb .. Le are needed

  ChunkSet<2, 1> cs;
  cs.init(reinterpret_cast<int *>(sm + VISC_NST * VISC_STAGE), tid, x0, y0, nx, ny);
  const double *__restrict__ u = p.u, *__restrict__ v = p.v, *__restrict__ w = p.w, *__restrict__ rho = p.rho;
  auto slot = [&](int L) { return sm + ((L - Lb) % VISC_NST) * VISC_STAGE; };
  auto stage_in = [&](int L) {
    if (L > Le) return;
    double *b = slot(L);
    if (L >= 0) {
      cs.issue(b, u + (size_t)L * plane);
      cs.issue(b + GS::SZ, v + (size_t)L * plane);
    }
    cs.issue(b + 2 * GS::SZ, w + (size_t)(L + 1) * plane);  // face L+1 (L = -1: the lower lid)
  };
#pragma unroll
  for (int n = 0; n < 4; n++) {
    stage_in(Lb + n);
    cp_async_commit();
  }
  constexpr int WS = GS::W;
  const int c = GS::centre(tx, ty);
  const size_t oc = act ? (size_t)j * nx + i : 0;
  const double rdx = p.rdx, rdy = p.rdy;
  double rho_n = act ? rho[(size_t)k0 * plane + oc] : 0.0;

#pragma unroll 1
  for (int k = k0; k < k1; k++) {
    cp_async_wait_but_one();  // stages up to k+1 have landed; k+2 may still be in flight
    __syncthreads();
    stage_in(k + 3);          // into the slot of stage k-2, which every thread has finished reading
    cp_async_commit();
    if (!act) continue;
    const double rc = rho_n;
    if (k + 1 < k1) rho_n = rho[(size_t)(k + 1) * plane + oc];
    double mu = rc * p.nu, K = rc * p.alpha;
    if (p.diffusion == 2) {
      const double *__restrict__ su = slot(k), *__restrict__ sv = su + GS::SZ, *__restrict__ swt = su + 2 * GS::SZ;
      const double *__restrict__ sm1 = slot(k - 1), *__restrict__ sp1 = slot(k + 1);
      const double *__restrict__ swb = sm1 + 2 * GS::SZ;  // w at face k
      const double u_c = su[c], u_p = su[c + 1], v_c = sv[c], v_p = sv[c + WS];
      const double S11 = (u_p - u_c) * rdx, S22 = (v_p - v_c) * rdy;
      const double w_c = swb[c], w_t = swt[c];
      const double S33 = (w_t - w_c) * p.rdz[k];
      // S12 at the four xy-edges around the centre
      const double u_jm = su[c - WS], u_jp = su[c + WS], u_pjm = su[c + 1 - WS], u_pjp = su[c + 1 + WS];
      const double v_im = sv[c - 1], v_ip = sv[c + 1], v_imp = sv[c - 1 + WS], v_ipp = sv[c + 1 + WS];
      const double e00 = 0.5 * ((u_c - u_jm) * rdy + (v_c - v_im) * rdx);
      const double e10 = 0.5 * ((u_p - u_pjm) * rdy + (v_ip - v_c) * rdx);
      const double e01 = 0.5 * ((u_jp - u_c) * rdy + (v_p - v_imp) * rdx);
      const double e11 = 0.5 * ((u_pjp - u_p) * rdy + (v_ipp - v_p) * rdx);
      const double s12 = 0.25 * (e00 + e10 + e01 + e11);
      // S13 at (i,k), (i+1,k), (i,k+1), (i+1,k+1); S23 likewise; zero on the lids
      double s13 = 0.0, s23 = 0.0;
      if (k >= 1) {
        const double rhw = p.rhw[k];
        const double *__restrict__ um = sm1, *__restrict__ vm = sm1 + GS::SZ;
        s13 += 0.5 * ((u_c - um[c]) * rhw + (w_c - swb[c - 1]) * rdx) +
               0.5 * ((u_p - um[c + 1]) * rhw + (swb[c + 1] - w_c) * rdx);
        s23 += 0.5 * ((v_c - vm[c]) * rhw + (w_c - swb[c - WS]) * rdy) +
               0.5 * ((v_p - vm[c + WS]) * rhw + (swb[c + WS] - w_c) * rdy);
      }
      if (k + 1 <= nz - 1) {
        const double rhw = p.rhw[k + 1];
        const double *__restrict__ up = sp1, *__restrict__ vp = sp1 + GS::SZ;
        s13 += 0.5 * ((up[c] - u_c) * rhw + (w_t - swt[c - 1]) * rdx) +
               0.5 * ((up[c + 1] - u_p) * rhw + (swt[c + 1] - w_t) * rdx);
        s23 += 0.5 * ((vp[c] - v_c) * rhw + (w_t - swt[c - WS]) * rdy) +
               0.5 * ((vp[c + WS] - v_p) * rhw + (swt[c + WS] - w_t) * rdy);
      }
      s13 *= 0.25;
      s23 *= 0.25;
      const double ss = 2.0 * (S11 * S11 + S22 * S22 + S33 * S33) + 4.0 * (s12 * s12 + s13 * s13 + s23 * s23);
      const double mut = rc * p.csd2[k] * sqrt(ss);
      mu += mut;
      K += mut * p.rPrt;
    }
    p.mu[(size_t)k * plane + oc] = mu;
    p.K[(size_t)k * plane + oc] = K;
  }
}

// number of level chunks so that a small grid still fills the machine (2 CTAs x 148 SMs, twice over)
static int level_chunks(const erf_ctx *c, int *kchunk) {
  const int tiles = ((c->nx + TX - 1) / TX) * ((c->ny + TY - 1) / TY);
  int nch = (592 + tiles - 1) / tiles;
  const int maxch = c->nz / 8 > 1 ? c->nz / 8 : 1;
  if (nch > maxch) nch = maxch;
  if (nch < 1) nch = 1;
  *kchunk = (c->nz + nch - 1) / nch;
  return (c->nz + *kchunk - 1) / *kchunk;
}

template <int OH, int FM>
static void launch_adv_mask(const SlowFlat &p, dim3 grid, int kchunk, cudaStream_t st) {
  const size_t smem = NSTAGE * adv_stage(FM) * sizeof(double) + (ChunkSet<4, 3>::TAB + ChunkSet<2, 1>::TAB) * sizeof(int);
  static OncePerDevice once;
  once.run([smem] { cudaFuncSetAttribute(k_adv_tiled<OH, FM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
  k_adv_tiled<OH, FM><<<grid, dim3(TX, TY), smem, st>>>(p, kchunk);
}

// split: 0 = one launch for all five tendencies; 1 = (rho, Theta, W) + (U, V); 2 = (rho, Theta) + (U, V) + (W)
// (the default: measured fastest on B200 -- 3 CTAs per SM without spills beat re-reading the U, V, W, p' tiles);
// 3 = one launch per field
template <int OH>
static int launch_adv_tiled(const SlowFlat &p, dim3 grid, int kchunk, int split, cudaStream_t st) {
  if (split == 1) {
    launch_adv_mask<OH, F_T | F_W>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_U | F_V>(p, grid, kchunk, st);
    return 2;
  }
  if (split == 2) {
    launch_adv_mask<OH, F_T>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_U | F_V>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_W>(p, grid, kchunk, st);
    return 3;
  }
  if (split == 3) {
    launch_adv_mask<OH, F_T>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_U>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_V>(p, grid, kchunk, st);
    launch_adv_mask<OH, F_W>(p, grid, kchunk, st);
    return 4;
  }
  launch_adv_mask<OH, F_ALL>(p, grid, kchunk, st);
  return 1;
}

void launch_adv_diff_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st) {
  int kchunk = 0;
  const int nch = level_chunks(c, &kchunk);
  dim3 grid((c->nx + TX - 1) / TX, (c->ny + TY - 1) / TY, nch);
  const int knob = (c->fz->variant >> 6) & 3;  // developer knob: 0 default, 1 fused, 2 two-way, 3 four-way
  const int split = knob == 0 ? 2 : (knob == 1 ? 0 : (knob == 2 ? 1 : 3));
  int n = 1;
  switch (c->p.adv_order_h) {
    case 2: n = launch_adv_tiled<2>(p, grid, kchunk, split, st); break;
    case 3: n = launch_adv_tiled<3>(p, grid, kchunk, split, st); break;
    case 4: n = launch_adv_tiled<4>(p, grid, kchunk, split, st); break;
    case 5: n = launch_adv_tiled<5>(p, grid, kchunk, split, st); break;
    default: n = launch_adv_tiled<6>(p, grid, kchunk, split, st); break;
  }
  c->launches += n;
}

void launch_visc_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st) {
  int kchunk = 0;
  const int nch = level_chunks(c, &kchunk);
  dim3 grid((c->nx + TX - 1) / TX, (c->ny + TY - 1) / TY, nch);
  const size_t smem = VISC_NST * VISC_STAGE * sizeof(double) + ChunkSet<2, 1>::TAB * sizeof(int);
  static OncePerDevice once;
  once.run([smem] { cudaFuncSetAttribute(k_visc_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
  k_visc_tiled<<<grid, dim3(TX, TY), smem, st>>>(p, kchunk);
  c->launches++;
}

template <int PART>
static void launch_diff_part(const SlowFlat &p, dim3 grid, int kchunk, cudaStream_t st) {
  const size_t smem = NSTAGE * diff_stage(PART) * sizeof(double) + ChunkSet<2, 1>::TAB * sizeof(int);
  static OncePerDevice once;
  once.run([smem] { cudaFuncSetAttribute(k_diff_tiled<PART>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); });
  k_diff_tiled<PART><<<grid, dim3(TX, TY), smem, st>>>(p, kchunk);
}

void launch_diff_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st) {
  int kchunk = 0;
  const int nch = level_chunks(c, &kchunk);
  dim3 grid((c->nx + TX - 1) / TX, (c->ny + TY - 1) / TY, nch);
  if (c->fz->variant & 1024) {  // developer knob: one launch per part (measured slower: 3.47 + 0.96 ms against 3.64 ms)
    launch_diff_part<1>(p, grid, kchunk, st);
    launch_diff_part<2>(p, grid, kchunk, st);
    c->launches += 2;
  } else {
    launch_diff_part<3>(p, grid, kchunk, st);
    c->launches++;
  }
}

}  // namespace erfb
