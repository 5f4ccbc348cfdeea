// k_terrain_slow.cu -- terrain-following grids: the advective part of the slow right-hand side f(S) for all five
// prognostic fields in ONE kernel.
//
//   R_rho, R_Theta, R_U, R_V at cell (i,j,k) and R_W at its lower face, from the mass fluxes hx U, hy V and the
//   contravariant vertical flux Omega ("rho Omega ... normal to the face"), the advected primitives
//   theta, u, v, w (L196) and the stencils of Eq. 17-21 (L198-L211) in the branch-free form
//   flux = M q_even - |M| q_odd [R:G1], vertical order reduced next to the lids [R:G13].
//
// One thread per cell, one level per CTA (so the vertical order is uniform over a CTA).  The seven column
// offsets in x and in y are wrapped (periodic) or clamped (open boundary) once per thread; every stencil value is then one load at
// level base + row offset + column offset, served by L1/L2 (neighbouring threads share all but one point).  This
// replaces the two terrain-general advection passes (general_cells.cuh advect_cell / advect_wface: a run-time
// order, a wrapped index per stencil point), which stay as the ERF_PATH_GENERAL cross-check.
#include "erf_ctx.cuh"
#include "slow_flat.cuh"

namespace erfb {
namespace tslow {

struct Args {
  const double *U, *V, *Om;              // momenta of the stage state, contravariant flux
  const double *th, *u, *v, *w;          // advected primitives
  const double *hx, *hy, *hc, *hu, *hv, *hw;
  double *Rrho, *RU, *RV, *RW, *RTh;
  int nx, ny, nz, ov, perx, pery;
  double rdx, rdy;
};

template <int OH>
__device__ __forceinline__ double hdiv(const double *q, double Mm, double Mp) {
  return flux_c<OH>(Mp, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(Mm, q[0], q[1], q[2], q[3], q[4], q[5]);
}

template <int OH>
__global__ void __launch_bounds__(256) k_adv_terrain(const Args p) {
  // levels fastest in the launch order: the CTAs resident at one time share their +-3 level windows through L2
  const int i = blockIdx.y * 32 + threadIdx.x, j = blockIdx.z * 8 + threadIdx.y, k = blockIdx.x;
  const int nx = p.nx, ny = p.ny, nz = p.nz;
  if (i >= nx || j >= ny) return;
  const size_t plane = (size_t)nx * ny, kb = (size_t)k * plane;
  int xo[7];
  size_t yo[7];
#pragma unroll
  for (int n = 0; n < 7; n++) {
    xo[n] = lati(i + n - 3, nx, p.perx);
    yo[n] = (size_t)lati(j + n - 3, ny, p.pery) * nx;
  }
  const size_t oc = yo[3] + xo[3], a = kb + oc;
  const bool low = k >= 1, up = k + 1 <= nz - 1;
  // levels k-3 .. k+3 clamped to the valid range (clamped values sit outside the reduced stencils)
  size_t zc[7], zf[7];
#pragma unroll
  for (int n = 0; n < 7; n++) {
    const int kk = k + n - 3;
    zc[n] = (size_t)min(max(kk, 0), nz - 1) * plane + oc;
    zf[n] = (size_t)min(max(kk, 0), nz) * plane + oc;
  }
  // mass fluxes through the faces of the cell and of its neighbours
  auto FX = [&](size_t b) { return p.hx[b] * p.U[b]; };
  auto FY = [&](size_t b) { return p.hy[b] * p.V[b]; };
  const size_t axm = kb + yo[3] + xo[2], axp = kb + yo[3] + xo[4], aym = kb + yo[2] + xo[3], ayp = kb + yo[4] + xo[3];
  const double fxmm = FX(axm), fxm = FX(a), fxp = FX(axp);
  const double fymm = FY(aym), fym = FY(a), fyp = FY(ayp);
  const double omm = p.Om[a], omp = p.Om[a + plane];
  const double rdx = p.rdx, rdy = p.rdy;
  const int ov = p.ov;
  const int oc_m = vorder(ov, min(k, nz - k)), oc_p = vorder(ov, min(k + 1, nz - k - 1));  // cell fields: faces k, k+1

  double q[7];
  // ---- rho, Theta
  {
    const double rhc = 1.0 / p.hc[a];
    p.Rrho[a] = -((fxp - fxm) * rdx + (fyp - fym) * rdy + (omp - omm)) * rhc;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.th[kb + yo[3] + xo[n]];
    double acc = hdiv<OH>(q, fxm, fxp) * rdx;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.th[kb + yo[n] + xo[3]];
    acc += hdiv<OH>(q, fym, fyp) * rdy;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.th[zc[n]];
    acc += (up ? flux_rt(oc_p, omp, q + 1) : 0.0) - (low ? flux_rt(oc_m, omm, q) : 0.0);
    p.RTh[a] = -acc * rhc;
  }
  // ---- rho*u at (i-1/2, j, k): mass fluxes averaged to the faces of its control volume (L196) [R:G11]
  {
    const double Mxm = 0.5 * (fxmm + fxm), Mxp = 0.5 * (fxm + fxp);
    const double Mym = 0.5 * (FY(kb + yo[3] + xo[2]) + fym), Myp = 0.5 * (FY(kb + yo[4] + xo[2]) + fyp);
    const double Mzm = 0.5 * (p.Om[axm] + omm), Mzp = 0.5 * (p.Om[axm + plane] + omp);
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.u[kb + yo[3] + xo[n]];
    double acc = hdiv<OH>(q, Mxm, Mxp) * rdx;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.u[kb + yo[n] + xo[3]];
    acc += hdiv<OH>(q, Mym, Myp) * rdy;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.u[zc[n]];
    acc += (up ? flux_rt(oc_p, Mzp, q + 1) : 0.0) - (low ? flux_rt(oc_m, Mzm, q) : 0.0);
    p.RU[a] = -acc / p.hu[a];
  }
  // ---- rho*v at (i, j-1/2, k)
  {
    const double Mxm = 0.5 * (FX(kb + yo[2] + xo[3]) + fxm), Mxp = 0.5 * (FX(kb + yo[2] + xo[4]) + fxp);
    const double Mym = 0.5 * (fymm + fym), Myp = 0.5 * (fym + fyp);
    const double Mzm = 0.5 * (p.Om[aym] + omm), Mzp = 0.5 * (p.Om[aym + plane] + omp);
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.v[kb + yo[3] + xo[n]];
    double acc = hdiv<OH>(q, Mxm, Mxp) * rdx;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.v[kb + yo[n] + xo[3]];
    acc += hdiv<OH>(q, Mym, Myp) * rdy;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.v[zc[n]];
    acc += (up ? flux_rt(oc_p, Mzp, q + 1) : 0.0) - (low ? flux_rt(oc_m, Mzm, q) : 0.0);
    p.RV[a] = -acc / p.hv[a];
  }
  // ---- rho*w at face (i, j, k-1/2): zero on the lids
  if (!low) {
    p.RW[a] = 0.0;
  } else {
    const size_t b = a - plane;
    const double Mxm = 0.5 * (FX(b) + fxm), Mxp = 0.5 * (FX(axp - plane) + fxp);
    const double Mym = 0.5 * (FY(b) + fym), Myp = 0.5 * (FY(ayp - plane) + fyp);
    const double Mzm = 0.5 * (p.Om[b] + omm), Mzp = 0.5 * (omm + omp);
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.w[kb + yo[3] + xo[n]];
    double acc = hdiv<OH>(q, Mxm, Mxp) * rdx;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.w[kb + yo[n] + xo[3]];
    acc += hdiv<OH>(q, Mym, Myp) * rdy;
#pragma unroll
    for (int n = 0; n < 7; n++) q[n] = p.w[zf[n]];
    // w-faces 0 .. nz are all valid points: between faces k-1, k and k, k+1
    acc += flux_rt(vorder(ov, min(k + 1, nz - k)), Mzp, q + 1) - flux_rt(vorder(ov, min(k, nz - k + 1)), Mzm, q);
    p.RW[a] = -acc / p.hw[a];
  }
  if (k == nz - 1) p.RW[a + plane] = 0.0;
}

}  // namespace tslow

// Eq. 17-21 only (the WENO scalars keep the general kernels)
bool terrain_advection_available(const erf_ctx *c) { return c->v.osh == c->v.oh && c->v.osv == c->v.ov; }

void launch_terrain_advection(erf_ctx *c, const F5 &S, cudaStream_t st) {
  tslow::Args p;
  const View &v = c->v;
  p.U = S.f[UU]; p.V = S.f[VV]; p.Om = c->Om_slow;
  p.th = c->prim.theta; p.u = c->prim.u; p.v = c->prim.v; p.w = c->prim.w;
  p.hx = v.hx; p.hy = v.hy; p.hc = v.hc; p.hu = v.hu; p.hv = v.hv; p.hw = v.hw;
  p.Rrho = c->R.f[RHO]; p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.RTh = c->R.f[TH];
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.ov = v.ov; p.perx = v.perx; p.pery = v.pery;
  p.rdx = 1.0 / v.dx; p.rdy = 1.0 / v.dy;
  dim3 block(32, 8), grid(c->nz, (c->nx + 31) / 32, (c->ny + 7) / 8);
  switch (v.oh) {
    case 2: tslow::k_adv_terrain<2><<<grid, block, 0, st>>>(p); break;
    case 3: tslow::k_adv_terrain<3><<<grid, block, 0, st>>>(p); break;
    case 4: tslow::k_adv_terrain<4><<<grid, block, 0, st>>>(p); break;
    case 5: tslow::k_adv_terrain<5><<<grid, block, 0, st>>>(p); break;
    default: tslow::k_adv_terrain<6><<<grid, block, 0, st>>>(p); break;
  }
  c->launches++;
}

}  // namespace erfb
