// k_slow_adv.cu -- flat grids: primitive variables, advection, pressure gradient and buoyancy of the slow
// right-hand side f(S) in ONE kernel.
//
//   S = (rho, U, V, W, Theta)  ->  R_rho, R_U, R_V, R_W, R_Theta (advective + pressure/buoyancy part)
//                                  and the stage constants theta^t, pi^t, 1/Theta^t of the acoustic substeps
//
//   Eq. 7   theta = Theta/rho, p' = p0 [(Theta/Theta0)^gamma - 1], pi       [R:S1]
//   L196                        advected primitive = momentum / face density (two-point mean)     [R:G11]
//   Eq. 17-21 (L196-L215)       flux-form advection, flux = M q_even - |M| q_odd                  [R:G1]
//   Eq. 2 (L65), L84            -grad p' and B = -(rho - rho0) g
//
// Layout of the work.  A CTA owns 32 x 8 columns (and a range of levels on small grids) and marches upward.  For
// every level the five state planes arrive as halo tiles through cp.async.bulk row copies (bulk.cuh; ring of NS
// stages, filled two levels ahead, periodic wrap in the source address).  All 512 threads first turn the newly
// landed level into primitive tiles theta, u, v, w (halo 3) and p' (halo 1) in shared memory -- each primitive is
// computed once per tile point instead of once per consumer -- and write theta^t, pi^t, 1/Theta^t of the interior.
// Then two groups of 256 threads (warp-uniform roles) each handle one column per thread:
//     group 0: rho, rho*theta and rho*w (+ vertical pressure gradient and buoyancy),   group 1: rho*u and rho*v.
// The two roles carry about the same arithmetic; splitting by field halves the per-thread state (vertical windows,
// FIFOs) while the tiles are loaded and the primitives computed once for both.
//
// Vertical stencils.  The horizontal work of a thread runs at the "front" level L (the plane that is resident with
// its halo); its horizontal divergences are parked in a three-deep register FIFO.  The value of the own column at
// level L enters a six-deep register window, which is what the vertical flux at face L-2 (cells L-5 .. L) needs;
// cell L-3 is finished in the same iteration.  So no plane other than the front one is ever read, and nothing is
// re-loaded from global memory.
#include <cstring>

#include "bulk.cuh"
#include "slow_flat.cuh"

namespace erfb {
namespace sadv {

constexpr int TX = 32, TY = 8, HX = 4, HY = 4;
constexpr int TW = TX + 2 * HX, TH = TY + 2 * HY, TSZ = TW * TH;  // 40 x 16 tile (rho: all rows; others rows 1..14)
constexpr int NS = 5;                                             // raw ring: levels P-2 .. P+2
constexpr int NPB = 3;                                            // primitive buffers
constexpr int PW = 36, PH = 10, PSZ = PW * PH;                    // p' tile: x in [-2, 33], y in [-1, 8]
constexpr int RAW = 5 * TSZ, PB = 4 * TSZ + PSZ;
constexpr int NTH = 512, NCOL = TX * TY;
constexpr int NCOPY = TH + 4 * (TH - 2);                          // row copies per level: 16 + 4 * 14
constexpr int NTAB = 8;                                           // per-level tables staged in shared memory
constexpr int MAXLEV = 320;                                       // nz + 1 <= MAXLEV (shared-memory budget)
constexpr size_t smem_bytes(int nlev) {
  return (size_t)(NS * RAW + NPB * PB + NTAB * nlev) * sizeof(double) + (NS + 1) * sizeof(uint64_t);
}

struct Maps {
  CUtensorMap m[5];  // rho, U, V, W, Theta: (TW x TH x 1) boxes
};

struct Poly {
  double c[12];  // (1+x)^kappa - 1 = x (c0 + c1 x + ... + c11 x^11), kappa = Rd/cv
  double xmax;   // series used for |x| < xmax
};

// 1/a to within an ulp: hardware seed (relative error 2^-23) and two Newton steps; a is a density, never 0 / inf / nan
__device__ __forceinline__ double rcp(double a) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));
  double e = fma(-a, r, 1.0);
  r = fma(r, e, r);
  e = fma(-a, r, 1.0);
  return fma(r, e, r);
}

template <int OVT>
__device__ __forceinline__ double vflux(int ov, int r, double M, const double *w) {
  const int ord = vorder(ov, r);
  if (OVT > 0 && ord == OVT) return flux_c<OVT>(M, w[0], w[1], w[2], w[3], w[4], w[5]);
  return flux_rt(ord, M, w);
}

template <int OH>
__device__ __forceinline__ double hdiv_x(const double *__restrict__ s, int c, double Mm, double Mp) {
  double q[7];
#pragma unroll
  for (int n = 0; n < 7; n++) q[n] = s[c + n - 3];
  return flux_c<OH>(Mp, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(Mm, q[0], q[1], q[2], q[3], q[4], q[5]);
}
template <int OH>
__device__ __forceinline__ double hdiv_y(const double *__restrict__ s, int c, double Mm, double Mp) {
  double q[7];
#pragma unroll
  for (int n = 0; n < 7; n++) q[n] = s[c + (n - 3) * TW];
  return flux_c<OH>(Mp, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(Mm, q[0], q[1], q[2], q[3], q[4], q[5]);
}

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 1, %0;\n" ::"n"(NTH) : "memory"); }

// the whole march of one thread; GRP (warp-uniform) selects the fields it advances, so that each role keeps only
// its own vertical windows and FIFOs in registers
template <int OH, int OVT, int GRP>
__device__ __forceinline__ void march(const SlowFlat &p, const Poly &poly, const Maps &maps, const int kchunk, double *sm) {
  double *const raw = sm;
  double *const prim = raw + NS * RAW;
  double *const tab = prim + NPB * PB;

  const int tid = threadIdx.x, t = tid & 255, tx = t & 31, ty = t >> 5;
  const int nx = p.nx, ny = p.ny, nz = p.nz, ov = p.ov;
  const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
  const int i = x0 + tx, j = y0 + ty;
  const bool act = i < nx && j < ny;
  const size_t plane = (size_t)nx * ny;
  const int k0 = blockIdx.z * kchunk, k1 = min(nz, k0 + kchunk);  // this CTA finishes cells / faces [k0, k1)
  const int Ls = max(k0 - 3, 0);                                  // first front level
  const int Ld = min(k1 + 2, nz);                                 // last level with data (nz: the W lid only)
  const int Lf = k1 + 2;                                          // last front level (flushes the FIFOs)
  const int nlev = nz + 1;
  uint64_t *const full = reinterpret_cast<uint64_t *>(tab + NTAB * nlev);
  // per-level tables: shared memory instead of a dependent global load per level
  const double *const t_dz = tab, *const t_rdz = tab + nlev, *const t_rhw = tab + 2 * nlev, *const t_rho0 = tab + 3 * nlev;
  const double *const t_Th0 = tab + 4 * nlev, *const t_rTh0 = tab + 5 * nlev, *const t_p0 = tab + 6 * nlev,
                      *const t_pi0 = tab + 7 * nlev;
  for (int n = tid; n < nlev; n += NTH) {
    tab[n] = p.dz[n]; tab[nlev + n] = p.rdz[n]; tab[2 * nlev + n] = p.rhw[n]; tab[3 * nlev + n] = p.rho0[n];
    tab[4 * nlev + n] = p.Th0[n]; tab[5 * nlev + n] = p.rTh0[n]; tab[6 * nlev + n] = p.p0[n]; tab[7 * nlev + n] = p.pi0[n];
  }

  if (GRP == 0 && tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; s++) mbar_init(&full[s], 1);
    mbar_init(&full[NS], NTH);  // "everybody has finished the previous iteration"
    mbar_fence_init();
  }
  cta_sync();

  // ---- producer: one level = 72 row copies (rho: 16 rows, U, V, W, Theta: 14 rows)
  int cp_f = -1, cp_off = 0, cp_gy = 0;
  const double *cp_src = nullptr;
  // (the copies are spread over all 16 warps, five lanes each: a warp issues its bulk copies one lane at a time)
  const int cpn = (tid & 31) < 5 ? (tid >> 5) * 5 + (tid & 31) : NCOPY;
  if (cpn < NCOPY) {
    int row;
    if (cpn < TH) { cp_f = 0; row = cpn; }
    else { cp_f = 1 + (cpn - TH) / (TH - 2); row = 1 + (cpn - TH) % (TH - 2); }
    cp_gy = pmodi(y0 - HY + row, ny);
    cp_off = cp_f * TSZ + row * TW;
    cp_src = cp_f == 0 ? p.rho : cp_f == 1 ? p.U : cp_f == 2 ? p.V : cp_f == 3 ? p.W : p.Th;
  }
  const int gxs = pmodi(x0 - HX, nx);
  // a CTA whose halo tile lies inside the domain gets each field plane with ONE tensor copy
  const bool inside = p.use_tma && x0 >= HX && x0 + TX + HX <= nx && y0 >= HY && y0 + TY + HY <= ny;
  auto issue = [&](int lv, int slot) {
    uint64_t *bar = &full[slot];
    if (inside) {
      if (tid == 0) {
        double *st = raw + slot * RAW;
        if (lv < nz) {
          mbar_arrive_expect_tx(bar, (unsigned)(5 * TSZ * 8));
#pragma unroll
          for (int f = 0; f < 5; f++) tma_tile_g2s(st + f * TSZ, &maps.m[f], x0 - HX, y0 - HY, lv, bar);
        } else {
          mbar_arrive_expect_tx(bar, (unsigned)(TSZ * 8));
          tma_tile_g2s(st + 3 * TSZ, &maps.m[3], x0 - HX, y0 - HY, lv, bar);
        }
      }
      return;
    }
    if (tid == 0) mbar_arrive_expect_tx(bar, (unsigned)((lv < nz ? NCOPY : TH - 2) * TW * 8));
    if (cp_f >= 0 && (lv < nz || cp_f == 3))
      bulk_row(raw + slot * RAW + cp_off, cp_src + (size_t)lv * plane, cp_gy, gxs, TW, nx, bar);
  };
  unsigned phase = 0;
  auto wait_slot = [&](int s) {
    mbar_wait(&full[s], (phase >> s) & 1u);
    phase ^= 1u << s;
  };

  // ---- primitives of level P (raw tile r, the level below in rm) into primitive buffer q.  The stencils never
  // touch the corners of the halo, so the points needed form a cross: rows 4..11 x columns 1..38 and rows 1..3,
  // 12..14 x columns 4..35 -- 496 points, one per thread in a single pass.
  int ppx, ppy;
  if (tid < 8 * 38) { ppy = HY + tid / 38; ppx = 1 + tid % 38; }
  else { const int t2 = tid - 8 * 38, rr = t2 >> 5; ppy = rr < 3 ? 1 + rr : 9 + rr; ppx = HX + (t2 & 31); }
  const bool p_on = tid < 8 * 38 + 6 * 32;
  const int ppt = ppy * TW + ppx;
  const bool p_pp = p_on && ppx >= 3 && ppx <= TX + HX - 1 && ppy >= 3 && ppy <= TY + HY - 1;  // p' region
  const int p_gi = x0 + ppx - HX, p_gj = y0 + ppy - HY;
  const bool p_int = p_pp && ppx >= HX && ppy >= HY && p_gi < nx && p_gj < ny;
  const size_t p_oc = p_int ? (size_t)p_gj * nx + p_gi : 0;
  auto prim_phase = [&](int P, const double *__restrict__ r, const double *__restrict__ rm, double *__restrict__ q) {
    if (!p_on) return;
    const double W = r[3 * TSZ + ppt];
    if (P < nz) {
      const double rc = r[ppt], Th = r[4 * TSZ + ppt];
      const double th = Th * rcp(rc);
      const double u = r[TSZ + ppt] * rcp(0.5 * (r[ppt - 1] + rc));
      const double v = r[2 * TSZ + ppt] * rcp(0.5 * (r[ppt - TW] + rc));
      const double w = W * rcp(P == 0 ? rc : 0.5 * (rm[ppt] + rc));
      q[ppt] = th;
      q[TSZ + ppt] = u;
      q[2 * TSZ + ppt] = v;
      q[3 * TSZ + ppt] = w;
      if (p_pp) {
        // x = Theta/Theta0 - 1, e = (1+x)^(Rd/cv) - 1: p' = p0 (x + e + x e), pi = pi0 (1 + e)   [R:S1]
        const double x = (Th - t_Th0[P]) * t_rTh0[P];
        double e;
        if (fabs(x) < poly.xmax) {
          e = poly.c[11];
#pragma unroll
          for (int n = 10; n >= 0; n--) e = fma(e, x, poly.c[n]);
          e *= x;
        } else {
          e = expm1(p.rdocv * log1p(x));
        }
        q[4 * TSZ + (ppy - 3) * PW + ppx - 2] = t_p0[P] * (x + e + x * e);
        if (p_int && P >= k0 && P < k1) {
          const size_t a = (size_t)P * plane + p_oc;
          p.theta[a] = th;
          p.pi[a] = t_pi0[P] * (1.0 + e);
          p.iT[a] = rcp(Th);
          if (p.diffusion != 0) {  // the diffusion kernels still read u, v, w from HBM
            p.u[a] = u;
            p.v[a] = v;
            p.w[a] = w;
          }
        }
      }
    } else {
      const double w = W * rcp(rm[ppt]);  // face nz: rho_w = rho(nz-1)
      q[3 * TSZ + ppt] = w;
      if (p_int && k1 == nz && p.diffusion != 0) p.w[(size_t)P * plane + p_oc] = w;
    }
  };

  // ---- prologue: levels Ls-1 (for rho below the first face) .. Ls+1
  int sP = Ls % NS;  // raw slot of level P
  {
    const int lo = max(Ls - 1, 0);
    for (int lv = lo; lv <= min(Ls + 1, Ld); lv++) issue(lv, lv % NS);
    if (Ls >= 1) wait_slot((Ls - 1) % NS);
  }
  int bP = Ls % NPB;  // primitive buffer of level P
  cta_sync();         // the tables

  const double rdx = p.rdx, rdy = p.rdy;
  const size_t oc = act ? (size_t)j * nx + i : 0;
  const int c = (ty + HY) * TW + tx + HX;           // own column in a TW x TH tile
  const int cP = (ty + 1) * PW + tx + 2;            // own column in the p' tile

  // per-thread state
  double win[6] = {0, 0, 0, 0, 0, 0}, win2[6] = {0, 0, 0, 0, 0, 0};  // vertical windows: (theta, w) or (u, v)
  double omw[4] = {0, 0, 0, 0};                                      // Omega at faces L-3 .. L (group 1: averaged to the u-point)
  double omv[3] = {0, 0, 0};                                         // group 1: Omega averaged to the v-point, faces L-2 .. L
  double f0[3] = {0, 0, 0}, f1[3] = {0, 0, 0}, f2[3] = {0, 0, 0};    // parked horizontal parts of levels L-3 .. L-1
  double fb0 = 0.0, fb1 = 0.0;                                       // vertical fluxes carried from the face below
  double U_cm = 0.0, U_pm = 0.0, V_cm = 0.0, V_pm = 0.0, pp_m = 0.0, rp_m = 0.0;  // group 0, rho*w: level L-1

  // One iteration = the column work of the front level L = P-2 (its primitives were finished two iterations ago),
  // then the primitives of level P, which has landed in the meantime.  The only synchronisation is a split
  // barrier: every thread ARRIVES at the end of its iteration and WAITS for the others only between its own column
  // work and the primitives (the first point where it overwrites something the others may still read), so warps
  // drift up to half an iteration apart instead of stopping together at every level.  Behind that wait thread 0
  // refills the raw slot that the previous iteration released (level P+2 takes the slot of level P-3).
  uint64_t *const done = &full[NS];
  unsigned done_phase = 0;
#pragma unroll 1
  for (int P = Ls; P <= Lf + 2; P++) {
    const int sM = sP == 0 ? NS - 1 : sP - 1;        // raw slot of level P-1
    const int sL = sM == 0 ? NS - 1 : sM - 1;        // raw slot of level P-2 (= the front level L)
    const int bL = bP == NPB - 1 ? 0 : bP + 1;       // (P-2) % 3 == (P+1) % 3
    const int L = P - 2;
    if (L >= Ls && act) {
    const double *__restrict__ r = raw + sL * RAW;
    const double *__restrict__ q = prim + bL * PB;
    const double *__restrict__ mU = r + TSZ, *__restrict__ mV = r + 2 * TSZ, *__restrict__ mW = r + 3 * TSZ;
    const bool cell = L < nz;                        // a cell level with data
    const bool inner = L >= 1 && L <= nz - 1;        // an interior w-face
    const int kf = L - 2, kc = L - 3;                // face whose vertical flux is formed, cell that is finished
    const bool fin = kc >= k0 && kc < k1;

    if (GRP == 0) {
      // ------------------------------------------------ rho, rho*theta; rho*w at face L with PG_z and buoyancy
      const double *__restrict__ sW = q + 3 * TSZ, *__restrict__ sPp = q + 4 * TSZ;
      double Hr = 0.0, HT = 0.0, X = 0.0, th = 0.0, wc = 0.0;
      if (L <= nz) wc = sW[c];
      if (cell) {
        const double U_c = mU[c], U_p = mU[c + 1], V_c = mV[c], V_p = mV[c + TW];
        Hr = (U_p - U_c) * rdx + (V_p - V_c) * rdy;
        HT = hdiv_x<OH>(q, c, U_c, U_p) * rdx + hdiv_y<OH>(q, c, V_c, V_p) * rdy;
        th = q[c];
        const double dzk = t_dz[L];
        const double U_cd = dzk * U_c, U_pd = dzk * U_p, V_cd = dzk * V_c, V_pd = dzk * V_p;
        const double pp_c = sPp[cP], rp_c = r[c] - t_rho0[L];
        if (L >= 1) {
          const double rhw = t_rhw[L];
          const double adv = hdiv_x<OH>(sW, c, 0.5 * (U_cm + U_cd), 0.5 * (U_pm + U_pd)) * rdx +
                             hdiv_y<OH>(sW, c, 0.5 * (V_cm + V_cd), 0.5 * (V_pm + V_pd)) * rdy;
          X = -adv * rhw - ((pp_c - pp_m) * rhw + p.g * 0.5 * (rp_m + rp_c));
        }
        U_cm = U_cd; U_pm = U_pd; V_cm = V_cd; V_pm = V_pd;
        pp_m = pp_c; rp_m = rp_c;
      }
#pragma unroll
      for (int n = 0; n < 5; n++) { win[n] = win[n + 1]; win2[n] = win2[n + 1]; }
      win[5] = th;                                   // cells L-5 .. L
      win2[5] = wc;                                  // faces L-5 .. L
      omw[0] = omw[1]; omw[1] = omw[2]; omw[2] = omw[3];
      omw[3] = inner ? mW[c] : 0.0;                  // Omega = W on a flat grid; 0 on the lids
      double fT = 0.0, Gz = 0.0;
      if (kf >= 1 && kf <= nz - 1) fT = vflux<OVT>(ov, min(kf, nz - kf), omw[1], win);
      // vertical flux of w at centre kc (between faces kc and kc+1)
      if (kc >= 0 && kc <= nz - 1) Gz = vflux<OVT>(ov, min(kc + 1, nz - kc), 0.5 * (omw[0] + omw[1]), win2);
      if (fin) {
        const double rdzc = t_rdz[kc];
        const size_t a = (size_t)kc * plane + oc;
        p.Rrho[a] = -(f0[0] + (omw[1] - omw[0]) * rdzc);
        p.RTh[a] = -(f1[0] + (fT - fb0) * rdzc);
        p.RW[a] = kc >= 1 ? f2[0] - (Gz - fb1) * t_rhw[kc] : 0.0;
        if (kc == nz - 1) p.RW[a + plane] = 0.0;     // upper lid
      }
      fb0 = fT;
      fb1 = Gz;
      f0[0] = f0[1]; f0[1] = f0[2]; f0[2] = Hr;
      f1[0] = f1[1]; f1[1] = f1[2]; f1[2] = HT;
      f2[0] = f2[1]; f2[1] = f2[2]; f2[2] = X;
    } else {
      // ------------------------------------------------ rho*u, rho*v
      const double *__restrict__ sU = q + TSZ, *__restrict__ sV = q + 2 * TSZ, *__restrict__ sPp = q + 4 * TSZ;
      double HU = 0.0, HV = 0.0, uc = 0.0, vc = 0.0;
      if (cell) {
        const double U_m = mU[c - 1], U_c = mU[c], U_p = mU[c + 1], U_ym = mU[c - TW], U_pym = mU[c - TW + 1];
        const double V_m = mV[c - TW], V_c = mV[c], V_p = mV[c + TW], V_xm = mV[c - 1], V_xmp = mV[c + TW - 1];
        const double pp_c = sPp[cP];
        HU = hdiv_x<OH>(sU, c, 0.5 * (U_m + U_c), 0.5 * (U_c + U_p)) * rdx +
             hdiv_y<OH>(sU, c, 0.5 * (V_xm + V_c), 0.5 * (V_xmp + V_p)) * rdy + (pp_c - sPp[cP - 1]) * rdx;
        HV = hdiv_x<OH>(sV, c, 0.5 * (U_ym + U_c), 0.5 * (U_pym + U_p)) * rdx +
             hdiv_y<OH>(sV, c, 0.5 * (V_m + V_c), 0.5 * (V_c + V_p)) * rdy + (pp_c - sPp[cP - PW]) * rdy;
        uc = sU[c];
        vc = sV[c];
      }
#pragma unroll
      for (int n = 0; n < 5; n++) { win[n] = win[n + 1]; win2[n] = win2[n + 1]; }
      win[5] = uc;
      win2[5] = vc;
      omw[0] = omw[1]; omw[1] = omw[2];
      omv[0] = omv[1]; omv[1] = omv[2];
      if (inner) {
        const double w_c = mW[c];
        omw[2] = 0.5 * (mW[c - 1] + w_c);            // Omega averaged to (i-1/2, face L)
        omv[2] = 0.5 * (mW[c - TW] + w_c);           // ... and to (j-1/2, face L)
      } else {
        omw[2] = omv[2] = 0.0;
      }
      double fU = 0.0, fV = 0.0;
      if (kf >= 1 && kf <= nz - 1) {
        const int rr = min(kf, nz - kf);
        fU = vflux<OVT>(ov, rr, omw[0], win);
        fV = vflux<OVT>(ov, rr, omv[0], win2);
      }
      if (fin) {
        const double rdzc = t_rdz[kc];
        const size_t a = (size_t)kc * plane + oc;
        p.RU[a] = -(f0[0] + (fU - fb0) * rdzc);
        p.RV[a] = -(f1[0] + (fV - fb1) * rdzc);
      }
      fb0 = fU;
      fb1 = fV;
      f0[0] = f0[1]; f0[1] = f0[2]; f0[2] = HU;
      f1[0] = f1[1]; f1[1] = f1[2]; f1[2] = HV;
    }
    }
    if (P > Ls) {                                    // everybody has finished iteration P-1
      mbar_wait(done, done_phase);
      done_phase ^= 1u;
    }
    if (P + 2 <= Ld) issue(P + 2, sL == 0 ? NS - 1 : sL - 1);  // level P+2 takes the slot of level P-3
    if (P <= Ld) {
      wait_slot(sP);
      prim_phase(P, raw + sP * RAW, raw + sM * RAW, prim + bP * PB);
    }
    mbar_arrive(done);
    sP = sP == NS - 1 ? 0 : sP + 1;
    bP = bL;
  }
}

template <int OH, int OVT>
__global__ void __launch_bounds__(NTH, 1)
    k_slow_adv(const SlowFlat p, const Poly poly, const __grid_constant__ Maps maps, const int kchunk) {
  extern __shared__ __align__(128) double sm[];
  if (threadIdx.x < NCOL) march<OH, OVT, 0>(p, poly, maps, kchunk, sm);
  else march<OH, OVT, 1>(p, poly, maps, kchunk, sm);
}

}  // namespace sadv

// (1+x)^kappa - 1 = sum_{n>=1} binom(kappa, n) x^n
static sadv::Poly make_poly(double kappa) {
  sadv::Poly P;
  long double c = 1.0L;
  for (int n = 1; n <= 12; n++) {
    c *= ((long double)kappa - (n - 1)) / n;
    P.c[n - 1] = (double)c;
  }
  P.xmax = 1.0 / 32.0;  // |c13| x^12 < 1e-20 there
  return P;
}

bool slow_adv_available(const erf_ctx *c) { return (c->nx % 2) == 0 && c->nz + 1 <= sadv::MAXLEV; }

template <int OH, int OVT>
static void launch_one(const SlowFlat &p, const sadv::Poly &poly, const sadv::Maps &maps, dim3 grid, int kchunk,
                       cudaStream_t st) {
  static OncePerDevice once;
  once.run([] {
    cudaFuncSetAttribute(sadv::k_slow_adv<OH, OVT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)sadv::smem_bytes(sadv::MAXLEV));
  });
  sadv::k_slow_adv<OH, OVT><<<grid, sadv::NTH, sadv::smem_bytes(p.nz + 1), st>>>(p, poly, maps, kchunk);
}

void launch_slow_adv(erf_ctx *c, const SlowFlat &pin, cudaStream_t st) {
  using namespace sadv;
  const int gx = (c->nx + TX - 1) / TX, gy = (c->ny + TY - 1) / TY;
  // level chunks so that a small grid still gives every SM a CTA (each chunk recomputes 6 levels)
  int nch = (2 * 148 + gx * gy - 1) / (gx * gy);
  const int maxch = c->nz / 4 > 1 ? c->nz / 4 : 1;
  if (nch > maxch) nch = maxch;
  const int kchunk = (c->nz + nch - 1) / nch;
  dim3 grid(gx, gy, (c->nz + kchunk - 1) / kchunk);
  const Poly poly = make_poly(c->v.rdocv);
  // tensor maps of the five input fields (cached per buffer: the state buffers rotate between steps)
  SlowFlat p = pin;
  Maps maps;
  memset(&maps, 0, sizeof(maps));
  p.use_tma = 1;
  const double *src[5] = {p.rho, p.U, p.V, p.W, p.Th};
  for (int f = 0; f < 5 && p.use_tma; f++) {
    auto it = c->fz->tmaps.find(src[f]);
    if (it == c->fz->tmaps.end()) {
      CUtensorMap m;
      if (!make_tile_map(&m, src[f], c->nx, c->ny, c->nz + 1, sadv::TW, sadv::TH)) { p.use_tma = 0; break; }
      it = c->fz->tmaps.emplace(src[f], m).first;
    }
    maps.m[f] = it->second;
  }
  const bool same = c->p.adv_order_h == c->p.adv_order_v;
  switch (c->p.adv_order_h) {
    case 2: same ? launch_one<2, 2>(p, poly, maps, grid, kchunk, st) : launch_one<2, 0>(p, poly, maps, grid, kchunk, st); break;
    case 3: same ? launch_one<3, 3>(p, poly, maps, grid, kchunk, st) : launch_one<3, 0>(p, poly, maps, grid, kchunk, st); break;
    case 4: same ? launch_one<4, 4>(p, poly, maps, grid, kchunk, st) : launch_one<4, 0>(p, poly, maps, grid, kchunk, st); break;
    case 5: same ? launch_one<5, 5>(p, poly, maps, grid, kchunk, st) : launch_one<5, 0>(p, poly, maps, grid, kchunk, st); break;
    default: same ? launch_one<6, 6>(p, poly, maps, grid, kchunk, st) : launch_one<6, 0>(p, poly, maps, grid, kchunk, st); break;
  }
  c->launches++;
}

}  // namespace erfb
