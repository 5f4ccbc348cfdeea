// k_fused.cu -- set-up and RK3 driver of the fused flat-grid path.
#include <cstdlib>
#include <cstring>

#include "acoustic_args.cuh"
#include "slow_flat.cuh"

namespace erfb {

// per-level tables from column (0,0) of the 3-D geometry / base-state fields
__global__ void k_level_tables(View v, double *dz, double *rdz, double *rhw, double *tabB, double *rho0,
                               double *Th0, double *rTh0, double *p0, double *pi0, double *csd2, double *tauc,
                               double *tauw) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > v.nz) return;
  size_t a = (size_t)k * v.ny * v.nx;
  {  // Rayleigh damping rates (L622) [R:G28]
    const double ztop = v.zw[(size_t)v.nz * v.ny * v.nx];
    const bool on = v.ray_fields != 0;
    tauw[k] = on ? gen::rayleigh_tau(v.ray_depth, v.ray_coef, v.zw[a], ztop) : 0.0;
    tauc[k] = on && k < v.nz ? gen::rayleigh_tau(v.ray_depth, v.ray_coef, v.zc[a], ztop) : 0.0;
  }
  if (k < v.nz) {
    dz[k] = v.hc[a];
    rdz[k] = 1.0 / v.hc[a];
    rho0[k] = v.rho0[a];
    Th0[k] = v.Th0[a];
    rTh0[k] = 1.0 / v.Th0[a];
    p0[k] = v.p0[a];
    pi0[k] = v.pi0[a];
    const double cd = v.Cs * cbrt(v.dx * v.dy * v.hc[a]);
    csd2[k] = cd * cd;
  } else {
    dz[k] = rdz[k] = rho0[k] = Th0[k] = rTh0[k] = p0[k] = pi0[k] = csd2[k] = 0.0;
  }
  if (k >= 1 && k < v.nz) {
    size_t b = (size_t)(k - 1) * v.ny * v.nx;
    rhw[k] = 1.0 / v.hw[a];
    double pi0f = 0.5 * (v.pi0[b] + v.pi0[a]);
    double rho0f = 0.5 * (v.rho0[b] + v.rho0[a]);
    tabB[k] = rho0f * v.rdocv / pi0f;
  } else {
    rhw[k] = 0.0;
    tabB[k] = 0.0;
  }
}

int fused_setup(erf_ctx *c, const erf_metrics *m, cudaStream_t st) {
  FusedState *z = new FusedState();  // value-initialised: every pointer null
  c->fz = z;
  // (the fused kernels carry the stencils of Eq. 17-21 only: WENO scalars run the terrain-general kernels)
  // ... and periodic boundaries only: open grids run the terrain-general kernels, whose index helper clamps
  z->ok = c->v.flat && m->base_is_1d && c->p.substep_mode == 1 && c->p.scalar_adv == 0 && c->v.perx && c->v.pery;
  z->variant = 0;  // kernel-variant mask, erf_set_option(ERF_OPT_VARIANT)
  if (!z->ok) return ERF_OK;
  const int nl = c->nz + 1;
  // Per-level tables.  They come from the SAME geometry / base-state routines as the 3-D arrays of the general
  // path, run on a one-column periodic grid (on a flat grid every column is that column), so both paths see
  // bit-identical metric terms without the 3-D arrays ever being allocated here.
  View vc = c->v;
  vc.nx = vc.ny = 1;
  double *col[18];
  for (auto &p : col) {
    p = c->alloc(nl);
    if (!p) return c->status;
  }
  double *zxf = col[0], *zyf = col[1], *zw = col[2], *hx = col[3], *hy = col[4], *hc = col[5], *zc = col[6];
  double *hw = col[7], *hu = col[8], *hv = col[9], *sxu = col[10], *syv = col[11], *sxw = col[12], *syw = col[13];
  double *rho0 = col[14], *Th0 = col[15], *p0 = col[16], *pi0 = col[17];
  vc.hc = hc; vc.hw = hw; vc.rho0 = rho0; vc.Th0 = Th0; vc.p0 = p0; vc.pi0 = pi0; vc.zw = zw; vc.zc = zc;
  gen::NodeH Z;
  Z.zn = nullptr; Z.zl = c->zl_dev; Z.nx = 1; Z.ny = 1;
  const double *r0in = c->base1d_r0, *t0in = c->base1d_T0;
  const int nz = c->nz;
  View vv = vc;
  auto column = [&](int nlev, auto f) {
    k_cells<<<dim3(1, 1, nlev), dim3(32, 8), 0, st>>>(1, 1, nlev, f);
    c->launches++;
  };
  column(nz + 1, [=] __device__(int i, int j, int k) { gen::geo_faces(vv, Z, zxf, zyf, zw, i, j, k); });
  column(nz, [=] __device__(int i, int j, int k) { gen::geo_cells(vv, zxf, zyf, zw, hx, hy, hc, zc, i, j, k); });
  column(nz + 1, [=] __device__(int i, int j, int k) {
    gen::geo_derived(vv, zxf, zyf, hc, zc, hw, hu, hv, sxu, syv, sxw, syw, i, j, k);
  });
  column(nz, [=] __device__(int i, int j, int k) { gen::base_state(vv, r0in, t0in, 1, rho0, Th0, p0, pi0, i, j, k); });
  double *t[12];
  for (auto &p : t) {
    p = c->alloc(nl);
    if (!p) return c->status;
  }
  k_level_tables<<<(nl + 127) / 128, 128, 0, st>>>(vc, t[0], t[1], t[2], t[3], t[4], t[5], t[6], t[7], t[8], t[9], t[10],
                                                   t[11]);
  c->launches++;
  z->tab = LevelTables{t[0], t[1], t[2], t[3], t[4], t[5], t[6], t[7], t[8], t[9], t[10], t[11]};
  // the layer's first level, from the host copy of the level heights (the rates themselves come from the device)
  z->ray_k0 = c->nz;
  if (c->v.ray_fields && m->z_levels) {
    const double zb = m->z_levels[c->nz] - c->v.ray_depth;
    int k0 = 0;
    while (k0 < c->nz && m->z_levels[k0 + 1] <= zb) k0++;  // cell k0 is the first whose top face lies above z_b
    z->ray_k0 = k0;
  }
  double **arr[] = {&z->iT, &z->U2, &z->V2, &z->Thd[0], &z->Thd[1], &z->cp_scr};
  for (auto p : arr) {
    *p = c->alloc(c->NW);
    if (!*p) return c->status;
  }
  if (c->p.diffusion != 0) {
    z->mu = c->alloc(c->NW);
    z->Kd = c->alloc(c->NW);
    if (!z->mu || !z->Kd) return c->status;
    if (!ensure_prim(c, false)) return c->status;  // u, v, w for the diffusion kernels
  }
  // wherever the round-1 slow-RHS kernels run instead of k_slow_adv (odd nx, nz + 1 beyond its level tables): k_prim_flat
  // writes u, v, w, p' whether or not diffusion reads them
  if (!slow_adv_available(c) && !ensure_prim(c, false)) return c->status;
  return ERF_OK;
}

void fused_buffer_roles(const erf_ctx *c, std::vector<const void *> &r) {
  const FusedState *z = c->fz;
  r.push_back(z->U2); r.push_back(z->V2); r.push_back(z->Thd[0]); r.push_back(z->Thd[1]);
}

void fused_set_buffer_roles(erf_ctx *c, const std::vector<const void *> &r, size_t n) {
  FusedState *z = c->fz;
  z->U2 = (double *)r[n]; z->V2 = (double *)r[n + 1]; z->Thd[0] = (double *)r[n + 2]; z->Thd[1] = (double *)r[n + 3];
}

void fused_release(erf_ctx *c) {
  delete c->fz;
  c->fz = nullptr;
}

bool fused_available(const erf_ctx *c) { return c->fz && c->fz->ok; }

void fused_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st) { launch_slow_flat(c, S, st); }

// n acoustic substeps of size dtau (Appendix A), one kernel each, with the RK stage combine folded in.
//   stage 0: S'' in/out in c->P about the stage state c->S (erf_acoustic);
//   stage 1: RK stage 1: S^t = S^n = c->S, S'' = 0, the stage result goes to c->St;
//   stage 2, 3: S'' = c->S - c->St at the first substep (L581) [R:G7], c->St += S'' at the last (L593).
// U'', V'' ping-pong between c->P and (U2, V2); Theta'' rotates through three buffers so that
// Theta''_d = Theta'' + beta_d (Theta'' - Theta''_prev) (L144) [R:G6] can be formed at load time.
static void acoustic_substeps(erf_ctx *c, double dtau, int n, int stage, cudaStream_t st) {
  FusedState *z = c->fz;
  if (n <= 0) return;
  const bool acc = c->sc_Q != nullptr && stage >= 1;  // transported scalar: accumulate the averaged momenta (L138)
  const bool tile = acoustic_tile_selected(c) && !acc;
  AcArgs p;
  p.nx = c->nx; p.ny = c->ny; p.nz = c->nz;
  p.dtau = dtau; p.rdx = 1.0 / c->v.dx; p.rdy = 1.0 / c->v.dy;
  p.b1 = 0.5 * (1.0 - c->v.beta_s); p.b2 = 0.5 * (1.0 + c->v.beta_s);  // L589
  p.beta_d = c->v.beta_d; p.g = c->v.g; p.gR = c->v.gam * c->v.Rd;
  p.RU = c->R.f[UU]; p.RV = c->R.f[VV]; p.RW = c->R.f[WW]; p.Rrho = c->R.f[RHO]; p.RTh = c->R.f[TH];
  p.theta = c->theta_t; p.pi = c->pi_t; p.iT = z->iT;
  p.rdz = z->tab.rdz; p.rhw = z->tab.rhw; p.tabB = z->tab.tabB;
  p.cp_scr = z->cp_scr;
  p.sumU = acc ? c->sc_sum[0] : nullptr; p.sumV = acc ? c->sc_sum[1] : nullptr; p.sumOm = acc ? c->sc_sum[2] : nullptr;

  double *cur = c->P.f[TH], *prev = c->P.f[TH], *fr[2] = {z->Thd[0], z->Thd[1]};  // the three Theta'' buffers
  int nfree = 2;
  bool rotated = false;
  for (int sidx = 0; sidx < n; sidx++) {
    Timed t(c, T_ACOUSTIC_FUSED, st);
    const bool first = stage >= 1 && sidx == 0, last = stage >= 1 && sidx == n - 1;
    int mode = (first ? MODE_FIRST : 0) | (last ? MODE_LAST : 0);
    if (stage == 1) mode |= MODE_ZERO;
    for (int f = 0; f < 5; f++) {
      p.Sn[f] = c->S.f[f];
      p.St[f] = stage == 1 ? c->S.f[f] : c->St.f[f];
    }
    p.Pu = c->P.f[UU]; p.Pv = c->P.f[VV]; p.Pw = c->P.f[WW]; p.Pr = c->P.f[RHO]; p.Pt = cur; p.Ptp = prev;
    p.oTp = nullptr;
    p.write_cp = sidx == 0;
    bool swap_uv = false, swap_stage = false;
    if (last) {
      if (stage == 1) {  // out of place: S^n -> S^t buffers
        p.oU = c->St.f[UU]; p.oV = c->St.f[VV]; p.oW = c->St.f[WW]; p.oR = c->St.f[RHO]; p.oT = c->St.f[TH];
      } else if (first) {  // neighbours still read S^t: write the stage result to the S'' buffers, then swap
        p.oU = c->P.f[UU]; p.oV = c->P.f[VV]; p.oW = c->P.f[WW]; p.oR = c->P.f[RHO]; p.oT = c->P.f[TH];
        swap_stage = true;
      } else {  // in place (own cells only)
        p.oU = c->St.f[UU]; p.oV = c->St.f[VV]; p.oW = c->St.f[WW]; p.oR = c->St.f[RHO]; p.oT = c->St.f[TH];
      }
    } else if (first) {
      p.oU = c->P.f[UU]; p.oV = c->P.f[VV]; p.oW = c->P.f[WW]; p.oR = c->P.f[RHO];
      p.oTp = c->P.f[TH];  // initial Theta'' = Theta''_prev of the next substep
      p.oT = fr[--nfree];
      rotated = true;
    } else {
      p.oU = z->U2; p.oV = z->V2; p.oW = c->P.f[WW]; p.oR = c->P.f[RHO];
      p.oT = fr[--nfree];
      rotated = true;
      swap_uv = true;
    }
    // column scratch of the thread-per-column kernel: the outputs themselves, except where the output buffer
    // still holds the stage state that is added at the end (in-place LAST): then the consumed S'' buffers
    if (last && !first) { p.kW = c->P.f[WW]; p.kR = c->P.f[RHO]; p.kT = fr[nfree - 1]; }
    else { p.kW = p.oW; p.kR = p.oR; p.kT = p.oT; }
    if (tile) launch_acoustic_tile_one(p, mode, st);
    else launch_acoustic_flat_one(p, mode, st);
    c->launches++;
    if (swap_uv) {
      double *t1 = c->P.f[UU]; c->P.f[UU] = z->U2; z->U2 = t1;
      double *t2 = c->P.f[VV]; c->P.f[VV] = z->V2; z->V2 = t2;
    }
    if (swap_stage)
      for (int f = 0; f < 5; f++) { double *t1 = c->St.f[f]; c->St.f[f] = c->P.f[f]; c->P.f[f] = t1; }
    if (!last) {
      if (first) {
        prev = c->P.f[TH];
      } else {
        if (prev != cur) fr[nfree++] = prev;
        prev = cur;
      }
      cur = p.oT;
    }
  }
  // keep three distinct Theta'' buffers: the live one in c->P
  if (rotated && cur != c->P.f[TH]) {
    double *others[2];
    int m = 0;
    if (prev != cur) others[m++] = prev;
    for (int q = 0; q < nfree && m < 2; q++) others[m++] = fr[q];
    c->P.f[TH] = cur; z->Thd[0] = others[0]; z->Thd[1] = others[1];
  }
}

void fused_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st) {
  (void)St;
  acoustic_substeps(c, dtau, n, 0, st);
}

void fused_rk3_step(erf_ctx *c, double dt, int ns, cudaStream_t st) {
  if (c->sc_Q) cudaMemcpyAsync(c->sc_Qt, c->sc_Q, c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  for (int stage = 1; stage <= 3; stage++) {
    int nsub = stage == 1 ? 1 : (stage == 2 ? ns / 2 : ns);  // L170
    double dtau = stage == 1 ? dt / 3.0 : dt / ns;
    const double dts = stage == 1 ? dt / 3.0 : (stage == 2 ? dt / 2.0 : dt);
    // f(S^t) every stage (L140) (also theta^t, pi^t, 1/Theta^t); S^t = S^n in stage 1
    const F5 &Sstage = stage == 1 ? c->S : c->St;
    launch_slow_flat(c, Sstage, st);
    if (c->sc_Q) scalar_prepare_fused(c, Sstage, c->sc_Qt, nsub, st);  // before the last substep overwrites S^t
    acoustic_substeps(c, dtau, nsub, stage, st);
    if (c->sc_Q) {  // Eq. 4 after the substeps of the stage (L138)
      scalar_stage(c, c->St, c->sc_Qt, c->sc_Q, c->sc_Qnew, nsub, dts, st, true);
      double *t = c->sc_Qt; c->sc_Qt = c->sc_Qnew; c->sc_Qnew = t;
    }
  }
  if (c->sc_Q) { double *t = c->sc_Q; c->sc_Q = c->sc_Qt; c->sc_Qt = t; }
  for (int f = 0; f < 5; f++) {
    double *t = c->S.f[f];
    c->S.f[f] = c->St.f[f];
    c->St.f[f] = t;
  }
}

}  // namespace erfb
