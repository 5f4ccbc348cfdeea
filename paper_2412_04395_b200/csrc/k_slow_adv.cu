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
// stages, filled two levels ahead, periodic wrap in the source address).  All 768 threads first turn the newly
// landed level into primitive tiles theta, u, v, w (halo 3) and p' (halo 1) in shared memory -- each primitive is
// computed once per tile point instead of once per consumer -- and write theta^t, pi^t, 1/Theta^t of the interior.
// Then three groups of 256 threads (warp-uniform roles) each handle one column per thread:
//     group 0: rho and rho*theta,   group 1: rho*u and rho*v,   group 2: rho*w (+ vertical PG and buoyancy).
// Splitting by field keeps every thread under 85 registers (768 threads per SM) while the tiles are loaded and the
// primitives computed once for all three.
//
// Vertical stencils.  The horizontal work of a thread runs at the "front" level L (the plane that is resident with
// its halo); its horizontal divergences are parked in a three-deep FIFO (registers; shared memory for group 1).
// The value of the own column at level L enters a six-deep register window, which is what the vertical flux at
// face L-2 (cells L-5 .. L) needs; cell L-3 is finished in the same iteration.  So no plane other than the front
// one is ever read, and nothing is re-loaded from global memory.
#include "bulk.cuh"
#include "slow_flat.cuh"

namespace erfb {
namespace sadv {

constexpr int TX = 32, TY = 8, HX = 4, HY = 4;
constexpr int TW = TX + 2 * HX, TH = TY + 2 * HY, TSZ = TW * TH;  // 40 x 16 tile (rho: all rows; others rows 1..14)
constexpr int NS = 4;                                             // raw ring: levels P-1 .. P+2
constexpr int NPB = 3;                                            // primitive buffers
constexpr int PW = 36, PH = 10, PSZ = PW * PH;                    // p' tile: x in [-2, 33], y in [-1, 8]
constexpr int RAW = 5 * TSZ, PB = 4 * TSZ + PSZ;
constexpr int NTH = 768, NCOL = TX * TY;
constexpr int NCOPY = TH + 4 * (TH - 2);                          // row copies per level: 16 + 4 * 14
constexpr size_t SMEM = (size_t)(NS * RAW + NPB * PB + NCOL * 4 * 2) * sizeof(double) + NS * sizeof(uint64_t);

struct Poly {
  double c[12];  // (1+x)^kappa - 1 = x (c0 + c1 x + ... + c11 x^11), kappa = Rd/cv
  double xmax;   // series used for |x| < xmax
};

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
__device__ __forceinline__ void march(const SlowFlat &p, const Poly &poly, const int kchunk, double *sm) {
  double *const raw = sm;
  double *const prim = raw + NS * RAW;
  double *const fifo = prim + NPB * PB;
  uint64_t *const full = reinterpret_cast<uint64_t *>(fifo + NCOL * 4 * 2);

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

  if (GRP == 0 && tid == 0) {
#pragma unroll
    for (int s = 0; s < NS; s++) mbar_init(&full[s], 1);
    mbar_fence_init();
  }
  cta_sync();

  // ---- producer: one level = 72 row copies (rho: 16 rows, U, V, W, Theta: 14 rows), one per thread
  const int gxs = pmodi(x0 - HX, nx);
  int cp_f = -1, cp_row = 0, cp_gy = 0;
  if (tid < NCOPY) {
    if (tid < TH) { cp_f = 0; cp_row = tid; }
    else { cp_f = 1 + (tid - TH) / (TH - 2); cp_row = 1 + (tid - TH) % (TH - 2); }
    cp_gy = pmodi(y0 - HY + cp_row, ny);
  }
  auto issue = [&](int lv) {
    double *st = raw + (lv % NS) * RAW;
    uint64_t *bar = &full[lv % NS];
    if (tid == 0) mbar_arrive_expect_tx(bar, (unsigned)((lv < nz ? NCOPY : TH - 2) * TW * 8));
    if (cp_f >= 0 && (lv < nz || cp_f == 3)) {
      const double *src = cp_f == 0 ? p.rho : cp_f == 1 ? p.U : cp_f == 2 ? p.V : cp_f == 3 ? p.W : p.Th;
      bulk_row(st + cp_f * TSZ + cp_row * TW, src + (size_t)lv * plane, cp_gy, gxs, TW, nx, bar);
    }
  };
  unsigned phase = 0;
  auto wait_level = [&](int lv) {
    const int s = lv % NS;
    mbar_wait(&full[s], (phase >> s) & 1u);
    phase ^= 1u << s;
  };

  // ---- primitives of level P into buffer P % NPB (every thread: one tile point)
  const int ppt = tid, ppy = ppt / TW, ppx = ppt - ppy * TW;
  const bool p_on = ppt < TSZ && ppy >= 1 && ppy <= TH - 2;
  const bool p_pp = p_on && ppx >= 3 && ppx <= TX + HX - 1 && ppy >= 3 && ppy <= TY + HY - 1;    // p' region
  const int p_gi = x0 + ppx - HX, p_gj = y0 + ppy - HY;
  const bool p_int = p_on && ppx >= HX && ppx < HX + TX && ppy >= HY && ppy < HY + TY && p_gi < nx && p_gj < ny;
  auto prim_phase = [&](int P) {
    if (!p_on) return;
    const double *__restrict__ r = raw + (P % NS) * RAW;
    double *__restrict__ q = prim + (P % NPB) * PB;
    const double W = r[3 * TSZ + ppt];
    if (P < nz) {
      const double rc = r[ppt], Th = r[4 * TSZ + ppt];
      q[ppt] = Th / rc;
      if (ppx >= 1) q[TSZ + ppt] = r[TSZ + ppt] / (0.5 * (r[ppt - 1] + rc));
      q[2 * TSZ + ppt] = r[2 * TSZ + ppt] / (0.5 * (r[ppt - TW] + rc));
      const double rw = P == 0 ? rc : 0.5 * (raw[((P - 1) % NS) * RAW + ppt] + rc);
      q[3 * TSZ + ppt] = W / rw;
      if (p_pp) {
        // x = Theta/Theta0 - 1, e = (1+x)^(Rd/cv) - 1: p' = p0 (x + e + x e), pi = pi0 (1 + e)   [R:S1]
        const double x = (Th - p.Th0[P]) * p.rTh0[P];
        double e;
        if (fabs(x) < poly.xmax) {
          e = poly.c[11];
#pragma unroll
          for (int n = 10; n >= 0; n--) e = fma(e, x, poly.c[n]);
          e *= x;
        } else {
          e = expm1(p.rdocv * log1p(x));
        }
        q[4 * TSZ + (ppy - 3) * PW + ppx - 2] = p.p0[P] * (x + e + x * e);
        if (p_int && P >= k0 && P < k1) {
          const size_t a = (size_t)P * plane + (size_t)p_gj * nx + p_gi;
          p.theta[a] = q[ppt];
          p.pi[a] = p.pi0[P] * (1.0 + e);
          p.iT[a] = 1.0 / Th;
          if (p.diffusion != 0) {  // the diffusion kernels still read u, v, w from HBM
            p.u[a] = q[TSZ + ppt];
            p.v[a] = q[2 * TSZ + ppt];
            p.w[a] = q[3 * TSZ + ppt];
          }
        }
      }
    } else {
      const double wl = W / raw[((P - 1) % NS) * RAW + ppt];  // face nz: rho_w = rho(nz-1)
      q[3 * TSZ + ppt] = wl;
      if (p_int && k1 == nz && p.diffusion != 0) p.w[(size_t)P * plane + (size_t)p_gj * nx + p_gi] = wl;
    }
  };

  // ---- prologue: levels Ls-1 (for rho below the first face), Ls, Ls+1
  for (int lv = max(Ls - 1, 0); lv <= min(Ls + 1, Ld); lv++) issue(lv);
  if (Ls >= 1) wait_level(Ls - 1);

  const double rdx = p.rdx, rdy = p.rdy;
  const size_t oc = act ? (size_t)j * nx + i : 0;
  const int c = (ty + HY) * TW + tx + HX;           // own column in a TW x TH tile
  const int cP = (ty + 1) * PW + tx + 2;            // own column in the p' tile
  double *const myfifo = fifo + t;                  // group 1: [(slot * 2 + f) * NCOL]

  // per-thread state (each group uses its own subset; the compiler drops the rest per branch)
  double win[6] = {0, 0, 0, 0, 0, 0}, win2[6] = {0, 0, 0, 0, 0, 0};  // vertical windows
  double omw[4] = {0, 0, 0, 0};                                      // Omega at faces L-3 .. L (own column / averaged)
  double omv[3] = {0, 0, 0};                                         // group 1: Mz for v at faces L-2 .. L
  double f0[3] = {0, 0, 0}, f1[3] = {0, 0, 0};                       // parked horizontal parts of cells L-3 .. L-1
  double fb0 = 0.0, fb1 = 0.0;                                       // vertical flux at the bottom face of the cell being finished
  double U_cm = 0.0, U_pm = 0.0, V_cm = 0.0, V_pm = 0.0, pp_m = 0.0, rp_m = 0.0;  // group 2: level L-1

#pragma unroll 1
  for (int P = Ls; P <= Lf + 1; P++) {
    if (P <= Ld) {
      wait_level(P);
      prim_phase(P);
    }
    cta_sync();
    if (P + 2 <= Ld) issue(P + 2);
    const int L = P - 1;
    if (L < Ls || !act) continue;
    const double *__restrict__ r = raw + (L % NS) * RAW;
    const double *__restrict__ q = prim + (L % NPB) * PB;
    const double *__restrict__ mU = r + TSZ, *__restrict__ mV = r + 2 * TSZ, *__restrict__ mW = r + 3 * TSZ;
    const bool cell = L < nz;                        // a cell level with data
    const bool inner = L >= 1 && L <= nz - 1;        // an interior w-face
    const int kf = L - 2, kc = L - 3;                // face whose vertical flux is formed, cell that is finished
    const bool fin = kc >= k0 && kc < k1;

    if (GRP == 0) {
      // ------------------------------------------------ rho, rho*theta
      double Hr = 0.0, HT = 0.0, th = 0.0;
      if (cell) {
        const double U_c = mU[c], U_p = mU[c + 1], V_c = mV[c], V_p = mV[c + TW];
        Hr = (U_p - U_c) * rdx + (V_p - V_c) * rdy;
        HT = hdiv_x<OH>(q, c, U_c, U_p) * rdx + hdiv_y<OH>(q, c, V_c, V_p) * rdy;
        th = q[c];
      }
#pragma unroll
      for (int n = 0; n < 5; n++) win[n] = win[n + 1];
      win[5] = th;
      omw[0] = omw[1]; omw[1] = omw[2]; omw[2] = omw[3];
      omw[3] = inner ? mW[c] : 0.0;                  // Omega = W on a flat grid; 0 on the lids
      double fT = 0.0;
      if (kf >= 1 && kf <= nz - 1) fT = vflux<OVT>(ov, min(kf, nz - kf), omw[1], win);
      if (fin) {
        const double rdzc = p.rdz[kc];
        const size_t a = (size_t)kc * plane + oc;
        p.Rrho[a] = -(f0[0] + (omw[1] - omw[0]) * rdzc);
        p.RTh[a] = -(f1[0] + (fT - fb0) * rdzc);
      }
      fb0 = fT;
      f0[0] = f0[1]; f0[1] = f0[2]; f0[2] = Hr;
      f1[0] = f1[1]; f1[1] = f1[2]; f1[2] = HT;
    } else if (GRP == 1) {
      // ------------------------------------------------ rho*u, rho*v
      const double *__restrict__ sU = q + TSZ, *__restrict__ sV = q + 2 * TSZ, *__restrict__ sP = q + 4 * TSZ;
      double uc = 0.0, vc = 0.0;
      if (cell) {
        const double U_m = mU[c - 1], U_c = mU[c], U_p = mU[c + 1], U_ym = mU[c - TW], U_pym = mU[c - TW + 1];
        const double V_m = mV[c - TW], V_c = mV[c], V_p = mV[c + TW], V_xm = mV[c - 1], V_xmp = mV[c + TW - 1];
        const double pp_c = sP[cP];
        const double HU = hdiv_x<OH>(sU, c, 0.5 * (U_m + U_c), 0.5 * (U_c + U_p)) * rdx +
                          hdiv_y<OH>(sU, c, 0.5 * (V_xm + V_c), 0.5 * (V_xmp + V_p)) * rdy + (pp_c - sP[cP - 1]) * rdx;
        const double HV = hdiv_x<OH>(sV, c, 0.5 * (U_ym + U_c), 0.5 * (U_pym + U_p)) * rdx +
                          hdiv_y<OH>(sV, c, 0.5 * (V_m + V_c), 0.5 * (V_c + V_p)) * rdy + (pp_c - sP[cP - PW]) * rdy;
        myfifo[((L & 3) * 2) * NCOL] = HU;
        myfifo[((L & 3) * 2 + 1) * NCOL] = HV;
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
        const double rdzc = p.rdz[kc];
        const size_t a = (size_t)kc * plane + oc;
        p.RU[a] = -(myfifo[((kc & 3) * 2) * NCOL] + (fU - fb0) * rdzc);
        p.RV[a] = -(myfifo[((kc & 3) * 2 + 1) * NCOL] + (fV - fb1) * rdzc);
      }
      fb0 = fU;
      fb1 = fV;
    } else {
      // ------------------------------------------------ rho*w at face L, pressure gradient and buoyancy
      const double *__restrict__ sW = q + 3 * TSZ, *__restrict__ sP = q + 4 * TSZ;
      double X = 0.0, wc = 0.0;
      if (L <= nz) wc = sW[c];
      if (cell) {
        const double dzk = p.dz[L];
        const double U_cd = dzk * mU[c], U_pd = dzk * mU[c + 1], V_cd = dzk * mV[c], V_pd = dzk * mV[c + TW];
        const double pp_c = sP[cP], rp_c = r[c] - p.rho0[L];
        if (L >= 1) {
          const double rhw = p.rhw[L];
          const double adv = hdiv_x<OH>(sW, c, 0.5 * (U_cm + U_cd), 0.5 * (U_pm + U_pd)) * rdx +
                             hdiv_y<OH>(sW, c, 0.5 * (V_cm + V_cd), 0.5 * (V_pm + V_pd)) * rdy;
          X = -adv * rhw - ((pp_c - pp_m) * rhw + p.g * 0.5 * (rp_m + rp_c));
        }
        U_cm = U_cd; U_pm = U_pd; V_cm = V_cd; V_pm = V_pd;
        pp_m = pp_c; rp_m = rp_c;
      }
#pragma unroll
      for (int n = 0; n < 5; n++) win[n] = win[n + 1];
      win[5] = wc;                                   // faces L-5 .. L
      omw[0] = omw[1]; omw[1] = omw[2]; omw[2] = omw[3];
      omw[3] = inner ? mW[c] : 0.0;
      // vertical flux of w at centre kc (between faces kc and kc+1)
      double Gz = 0.0;
      if (kc >= 0 && kc <= nz - 1) Gz = vflux<OVT>(ov, min(kc + 1, nz - kc), 0.5 * (omw[0] + omw[1]), win);
      if (fin) {
        const size_t a = (size_t)kc * plane + oc;
        p.RW[a] = kc >= 1 ? f0[0] - (Gz - fb0) * p.rhw[kc] : 0.0;
        if (kc == nz - 1) p.RW[a + plane] = 0.0;     // upper lid
      }
      fb0 = Gz;
      f0[0] = f0[1]; f0[1] = f0[2]; f0[2] = X;
    }
  }
}

template <int OH, int OVT>
__global__ void __launch_bounds__(NTH, 1) k_slow_adv(const SlowFlat p, const Poly poly, const int kchunk) {
  extern __shared__ __align__(128) double sm[];
  const int grp = threadIdx.x >> 8;
  if (grp == 0) march<OH, OVT, 0>(p, poly, kchunk, sm);
  else if (grp == 1) march<OH, OVT, 1>(p, poly, kchunk, sm);
  else march<OH, OVT, 2>(p, poly, kchunk, sm);
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

bool slow_adv_available(const erf_ctx *c) { return (c->nx % 2) == 0; }

template <int OH, int OVT>
static void launch_one(const SlowFlat &p, const sadv::Poly &poly, dim3 grid, int kchunk, cudaStream_t st) {
  static bool once = false;
  if (!once) {
    cudaFuncSetAttribute(sadv::k_slow_adv<OH, OVT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sadv::SMEM);
    once = true;
  }
  sadv::k_slow_adv<OH, OVT><<<grid, sadv::NTH, sadv::SMEM, st>>>(p, poly, kchunk);
}

void launch_slow_adv(erf_ctx *c, const SlowFlat &p, cudaStream_t st) {
  using namespace sadv;
  const int gx = (c->nx + TX - 1) / TX, gy = (c->ny + TY - 1) / TY;
  // level chunks so that a small grid still gives every SM a CTA (each chunk recomputes 6 levels)
  int nch = (2 * 148 + gx * gy - 1) / (gx * gy);
  const int maxch = c->nz / 16 > 1 ? c->nz / 16 : 1;
  if (nch > maxch) nch = maxch;
  const int kchunk = (c->nz + nch - 1) / nch;
  dim3 grid(gx, gy, (c->nz + kchunk - 1) / kchunk);
  const Poly poly = make_poly(c->v.rdocv);
  const bool same = c->p.adv_order_h == c->p.adv_order_v;
  switch (c->p.adv_order_h) {
    case 2: same ? launch_one<2, 2>(p, poly, grid, kchunk, st) : launch_one<2, 0>(p, poly, grid, kchunk, st); break;
    case 3: same ? launch_one<3, 3>(p, poly, grid, kchunk, st) : launch_one<3, 0>(p, poly, grid, kchunk, st); break;
    case 4: same ? launch_one<4, 4>(p, poly, grid, kchunk, st) : launch_one<4, 0>(p, poly, grid, kchunk, st); break;
    case 5: same ? launch_one<5, 5>(p, poly, grid, kchunk, st) : launch_one<5, 0>(p, poly, grid, kchunk, st); break;
    default: same ? launch_one<6, 6>(p, poly, grid, kchunk, st) : launch_one<6, 0>(p, poly, grid, kchunk, st); break;
  }
  c->launches++;
}

}  // namespace erfb
