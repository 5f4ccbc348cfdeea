// k_fused_slow.cu -- the slow right-hand side f(S) of PAPER.md Eq. 1-3 on flat grids: the primitive-variable
// kernel and the launch sequence.
//
// Six launches per evaluation:
//   k_prim_flat          S -> theta, u, v, w, p', pi^t, 1/Theta^t               (Eq. 7; L196)
//   k_adv_tiled x 3      advection (Eq. 17-21) + pressure gradient + buoyancy (L84) -> R,
//                        one launch each for (rho, Theta), (U, V), (W)                     (k_slow_tiled.cu)
//   k_visc_tiled         u, v, w, rho -> mu, K          (Eq. 9; Smagorinsky [R:G9])  (k_slow_tiled.cu)
//   k_diff_tiled         R -= div(tau), R_Theta -= div(F)                (Eq. 2-3, Eq. 9)      (k_slow_tiled.cu)
// On a flat grid all metric terms are per-level constants (tables), Omega = W, and every horizontal slope term
// of D0 vanishes identically.
#include "slow_flat.cuh"

namespace erfb {

// ------------------------------------------------------------------ primitives
__global__ void __launch_bounds__(256) k_prim_flat(const SlowFlat p) {
  const size_t plane = (size_t)p.nx * p.ny;
  const size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= plane * (p.nz + 1)) return;
  const int k = (int)(a / plane);
  const size_t r = a - (size_t)k * plane;
  const int j = (int)(r / p.nx), i = (int)(r - (size_t)j * p.nx);
  const double *__restrict__ rho = p.rho;
  if (k < p.nz) {
    const double rc = rho[a], Th = p.Th[a];
    const int im = i == 0 ? p.nx - 1 : i - 1, jm = j == 0 ? p.ny - 1 : j - 1;
    const size_t kk = (size_t)k * plane;
    p.theta[a] = Th / rc;
    // x = Theta/Theta0 - 1.  gamma = 1 + Rd/cv, so with e = (1+x)^(Rd/cv) - 1 = expm1((Rd/cv) log1p(x)):
    //   pi = pi0 (1 + e)                     pi = pi0 (Theta/Theta0)^(Rd/cv)
    //   p' = p0 [(1+x)(1+e) - 1] = p0 (x + e + x e)   p' = p0 [(Theta/Theta0)^gamma - 1]   [R:S1]
    // one log1p and one expm1 per cell, no cancellation (x, e are small and enter linearly)
    const double x = (Th - p.Th0[k]) * p.rTh0[k];
    const double e = expm1(p.rdocv * log1p(x));
    p.pp[a] = p.p0[k] * (x + e + x * e);
    p.pi[a] = p.pi0[k] * (1.0 + e);
    p.iT[a] = 1.0 / Th;
    p.u[a] = p.U[a] / (0.5 * (rho[kk + (size_t)j * p.nx + im] + rc));
    p.v[a] = p.V[a] / (0.5 * (rho[kk + (size_t)jm * p.nx + i] + rc));
    const double rw = k == 0 ? rc : 0.5 * (rho[a - plane] + rc);
    p.w[a] = p.W[a] / rw;
  } else {
    p.w[a] = p.W[a] / rho[a - plane];
  }
}

// Rayleigh damping layer (L219, L622) [R:G28] on the levels k0 .. nz-1 that the layer reaches: relaxation of the masked
// primitives towards (u_ref, v_ref, 0, theta0); the rates are per-level tables on a flat grid
__global__ void __launch_bounds__(256) k_rayleigh_flat(const SlowFlat p, const double *__restrict__ tauc,
                                                       const double *__restrict__ tauw, int k0, int fields,
                                                       double uref, double vref) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = k0 + blockIdx.z;
  if (i >= p.nx || j >= p.ny) return;
  const size_t kk = (size_t)k * p.nx * p.ny, a = kk + (size_t)j * p.nx + i;
  const double tc = tauc[k], rc = p.rho[a];
  if (fields & 1) p.RU[a] -= tc * (p.U[a] - 0.5 * (p.rho[kk + (size_t)j * p.nx + (i == 0 ? p.nx - 1 : i - 1)] + rc) * uref);
  if (fields & 2) p.RV[a] -= tc * (p.V[a] - 0.5 * (p.rho[kk + (size_t)(j == 0 ? p.ny - 1 : j - 1) * p.nx + i] + rc) * vref);
  if ((fields & 4) && k >= 1) p.RW[a] -= tauw[k] * p.W[a];
  if (fields & 8) p.RTh[a] -= tc * (p.Th[a] - rc * p.Th0[k] / p.rho0[k]);
}

void launch_slow_flat(erf_ctx *c, const F5 &S, cudaStream_t st) {
  Timed t(c, T_SLOW_FUSED, st);
  FusedState *z = c->fz;
  SlowFlat p;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz; p.ov = c->p.adv_order_v;
  p.rdx = 1.0 / c->v.dx; p.rdy = 1.0 / c->v.dy; p.g = c->v.g;
  p.rho = S.f[RHO]; p.U = S.f[UU]; p.V = S.f[VV]; p.W = S.f[WW]; p.Th = S.f[TH];
  p.theta = c->theta_t; p.pi = c->pi_t; p.iT = z->iT;
  p.u = c->prim.u; p.v = c->prim.v; p.w = c->prim.w; p.pp = c->prim.pp;
  p.Rrho = c->R.f[RHO]; p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.RTh = c->R.f[TH];
  p.mu = z->mu; p.K = z->Kd;
  p.dz = z->tab.dz; p.rdz = z->tab.rdz; p.rhw = z->tab.rhw; p.rho0 = z->tab.rho0; p.Th0 = z->tab.Th0;
  p.rTh0 = z->tab.rTh0; p.p0 = z->tab.p0; p.pi0 = z->tab.pi0; p.csd2 = z->tab.csd2;
  p.gam = c->v.gam; p.rdocv = c->v.rdocv; p.nu = c->v.nu; p.alpha = c->v.alpha;
  p.rPrt = c->p.diffusion == 2 ? 1.0 / c->v.Prt : 0.0;
  p.diffusion = c->p.diffusion;
  p.use_tma = 0;
  if (slow_adv_available(c) && !(z->variant & ERF_VARIANT_SPLIT_SLOW_RHS)) {
    launch_slow_adv(c, p, st);
  } else {
    const size_t plane = (size_t)c->nx * c->ny;
    k_prim_flat<<<(unsigned)((plane * (c->nz + 1) + 255) / 256), 256, 0, st>>>(p);
    c->launches++;
    launch_adv_diff_tiled(c, p, st);
  }
  if (c->p.diffusion != 0) {
    launch_visc_tiled(c, p, st);
    launch_diff_tiled(c, p, st);
  }
  if (z->ray_k0 < c->nz) {
    dim3 block(32, 8), grid((c->nx + 31) / 32, (c->ny + 7) / 8, c->nz - z->ray_k0);
    k_rayleigh_flat<<<grid, block, 0, st>>>(p, z->tab.tauc, z->tab.tauw, z->ray_k0, c->v.ray_fields, c->v.ray_uref,
                                            c->v.ray_vref);
    c->launches++;
  }
}

}  // namespace erfb
