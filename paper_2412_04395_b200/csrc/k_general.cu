// k_general.cu -- the GENERAL path: one kernel per operator pass, all intermediates in HBM.
// Serves terrain-following grids and cross-checks the fused kernels on the device.
#include "erf_ctx.cuh"

namespace erfb {

static bool ensure_diff(erf_ctx *c) {
  if (c->diff_alloc) return true;
  gen::Diff &d = c->diff;
  double **all[] = {&d.mu, &d.K, &d.S11, &d.S22, &d.S33, &d.S12, &d.S13, &d.S23, &d.qu, &d.qv,
                    &d.t11, &d.t22, &d.t33, &d.t12, &d.t13, &d.t23, &d.q11, &d.q22, &d.q12,
                    &d.q13, &d.q23, &d.qth, &d.ze12, &d.Fx, &d.Fy, &d.Fz};
  for (auto p : all) {
    *p = c->alloc(c->NW);
    if (!*p) return false;
  }
  c->diff_alloc = true;
  return true;
}

// u, v, w, p' (and theta, pi with `all`) work arrays: the general path and the round-1 fused slow-RHS kernels use them
bool ensure_prim(erf_ctx *c, bool all) {
  double **need[] = {&c->prim.u, &c->prim.v, &c->prim.w, &c->prim.pp, &c->prim.theta, &c->prim.pi};
  for (int n = 0; n < (all ? 6 : 4); n++)
    if (!*need[n]) {
      *need[n] = c->alloc(c->NW);
      if (!*need[n]) return false;
    }
  return true;
}

// the 3-D metric terms (S0) from the node heights, the 3-D base state with p0, pi0 from Eq. 7, and the
// unfused path's intermediates
int build_general(erf_ctx *c, const gen::NodeH &Z, const double *r0in, const double *t0in, int b1d, cudaStream_t st) {
  if (c->gen_ready) return c->status;
  double **geo[] = {&c->zxf, &c->zyf, &c->zw, &c->hx, &c->hy, &c->hc, &c->zc, &c->hw, &c->hu, &c->hv,
                    &c->sxw, &c->syw, &c->sxu, &c->syv, &c->rho0, &c->Th0, &c->p0, &c->pi0,
                    &c->Om_slow, &c->ac.Om, &c->ac.Th_prev, &c->ac.Thd,
                    &c->ac.om, &c->ac.Ttil, &c->ac.rtil, &c->ac.cpr, &c->ac.dpr};
  for (auto pp : geo) {
    *pp = c->alloc(c->NW);
    if (!*pp) return c->status;
  }
  if (!ensure_prim(c, true)) return c->status;
  View &v = c->v;
  v.zw = c->zw; v.hx = c->hx; v.hy = c->hy; v.hc = c->hc; v.zc = c->zc; v.hw = c->hw;
  v.hu = c->hu; v.hv = c->hv; v.sxw = c->sxw; v.syw = c->syw; v.sxu = c->sxu; v.syv = c->syv;
  v.rho0 = c->rho0; v.Th0 = c->Th0; v.p0 = c->p0; v.pi0 = c->pi0;
  View vv = v;
  double *zxf = c->zxf, *zyf = c->zyf, *zw = c->zw, *hx = c->hx, *hy = c->hy, *hc = c->hc, *zc = c->zc;
  double *hw = c->hw, *hu = c->hu, *hv = c->hv, *sxu = c->sxu, *syv = c->syv, *sxw = c->sxw, *syw = c->syw;
  double *rho0 = c->rho0, *Th0 = c->Th0, *p0 = c->p0, *pi0 = c->pi0;
  const int nz = c->nz;
  launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) { gen::geo_faces(vv, Z, zxf, zyf, zw, i, j, k); });
  launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::geo_cells(vv, zxf, zyf, zw, hx, hy, hc, zc, i, j, k); });
  launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) {
    gen::geo_derived(vv, zxf, zyf, hc, zc, hw, hu, hv, sxu, syv, sxw, syw, i, j, k);
  });
  launch_cells(c, st, nz, [=] __device__(int i, int j, int k) {
    gen::base_state(vv, r0in, t0in, b1d, rho0, Th0, p0, pi0, i, j, k);
  });
  c->gen_ready = true;
  return c->status;
}

// flat grids with a 1-D base state build the general arrays only when that path is first used
int ensure_general(erf_ctx *c, cudaStream_t st) {
  if (c->gen_ready) return c->status;
  if (!c->zl_dev || !c->base1d_r0) return c->status = ERF_EINVAL;
  gen::NodeH Z;
  Z.zn = nullptr; Z.zl = c->zl_dev; Z.nx = c->nx; Z.ny = c->ny;
  return build_general(c, Z, c->base1d_r0, c->base1d_T0, 1, st);
}

// kinematic W on the lids [R:G15]; on a flat grid the slopes vanish identically: W = 0
void impose_lids(erf_ctx *c, const F5 &S, cudaStream_t st) {
  if (c->gen_ready) {
    general_lids(c, S, st);
    return;
  }
  double *W = S.f[WW];
  const size_t plane = (size_t)c->nx * c->ny, top = plane * c->nz;
  const int nx = c->nx;
  launch_columns(c, st, [=] __device__(int i, int j) {
    const size_t a = (size_t)j * nx + i;
    W[a] = 0.0;
    W[top + a] = 0.0;
  });
}

void general_lids(erf_ctx *c, const F5 &S, cudaStream_t st) {
  View v = c->v;
  const double *U = S.f[UU], *V = S.f[VV];
  double *W = S.f[WW];
  launch_columns(c, st, [=] __device__(int i, int j) { gen::lids(v, U, V, W, i, j); });
}

// ---- per-cell passes as functors over the view type: CTAs whose 32 x 8 tile lies at least MARGIN columns inside the
// domain run the body on a ViewNW (no wrap / clamp in the index helper), the others on the View
namespace {
struct FPrim {
  F5 S; gen::Prim q;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const { gen::primitives(v, S.f, q, i, j, k); }
};
struct FOmega {
  F5 S; double *Om;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    Om[IX(v, i, j, k)] = gen::omega_at(v, S.f[UU], S.f[VV], S.f[WW], i, j, k);
  }
};
template <int PASS>
struct FDiff {
  gen::Prim q; gen::Diff d; F5 R; const double *rho;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    if (PASS == 1) gen::diff_pass1(v, q, d, i, j, k);
    if (PASS == 2) gen::diff_pass2(v, q, d, i, j, k);
    if (PASS == 3) gen::diff_pass3(v, rho, d, i, j, k);
    if (PASS == 4) gen::diff_pass4(v, d, i, j, k);
    if (PASS == 5) gen::diff_pass5(v, q, d, i, j, k);
    if (PASS == 6) gen::diff_pass6(v, q, d, R.f, i, j, k);
    if (PASS == 7) gen::diff_pass7(v, d, i, j, k);
    if (PASS == 8) gen::diff_pass8(v, d, R.f, i, j, k);
  }
};
struct FPgBuoy {
  F5 S, R; gen::Prim q; const double *pan;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    if (pan) gen::anel_pgbuoy_cell(v, q, pan, R.f, i, j, k);  // anelastic mode: p' of the projection, buoyancy from theta
    else gen::pgbuoy_cell(v, S.f, q, R.f, i, j, k);
  }
};
}  // namespace

// ---- inflow boundary [R:G30]: the first column (row) of cells is a Dirichlet column held at the values of erf_set_state
__global__ void k_inflow(F5 S, double *in_x, double *in_y, int nx, int ny, int nz, bool store) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y, f = blockIdx.z;
  const size_t plane = (size_t)nx * ny;
  if (in_x && t < ny) {
    const size_t a = (size_t)k * plane + (size_t)t * nx, b = ((size_t)f * (nz + 1) + k) * ny + t;
    if (store) in_x[b] = S.f[f][a]; else S.f[f][a] = in_x[b];
  }
  if (in_y && t < nx) {
    const size_t a = (size_t)k * plane + t, b = ((size_t)f * (nz + 1) + k) * nx + t;
    if (store) in_y[b] = S.f[f][a]; else S.f[f][a] = in_y[b];
  }
}

static void inflow_launch(erf_ctx *c, const F5 &S, bool store, cudaStream_t st) {
  const int n = c->nx > c->ny ? c->nx : c->ny;
  dim3 grid((n + 127) / 128, c->nz + 1, 5);
  if (!store && c->in_x && c->in_y) {  // x first, then y (the corner holds the same stored value either way)
    k_inflow<<<grid, 128, 0, st>>>(S, c->in_x, nullptr, c->nx, c->ny, c->nz, false);
    k_inflow<<<grid, 128, 0, st>>>(S, nullptr, c->in_y, c->nx, c->ny, c->nz, false);
    c->launches += 2;
    return;
  }
  k_inflow<<<grid, 128, 0, st>>>(S, c->in_x, c->in_y, c->nx, c->ny, c->nz, store);
  c->launches++;
}

void inflow_store(erf_ctx *c, cudaStream_t st) {
  if (!c->inx && !c->iny) return;
  if (c->inx && !c->in_x) c->in_x = c->alloc((size_t)5 * (c->nz + 1) * c->ny);
  if (c->iny && !c->in_y) c->in_y = c->alloc((size_t)5 * (c->nz + 1) * c->nx);
  if (c->status != ERF_OK) return;
  inflow_launch(c, c->S, true, st);
}

void inflow_impose(erf_ctx *c, const F5 &S, cudaStream_t st) {
  if ((c->inx && c->in_x) || (c->iny && c->in_y)) inflow_launch(c, S, false, st);
}

void general_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st, const double *pan) {
  View v = c->v;
  const int nz = c->nz;
  gen::Prim q = c->prim;
  F5 Sv = S, R = c->R;
  double *Om = c->Om_slow;
  launch_cells_v(c, st, nz + 1, FPrim{Sv, q});
  launch_cells_v(c, st, nz + 1, FOmega{Sv, Om});
  if (c->path == ERF_PATH_AUTO && terrain_advection_available(c)) {
    launch_terrain_advection(c, S, st);  // all five advective tendencies in one kernel (k_terrain_slow.cu)
  } else {
    launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::advect_cell(v, Sv.f, Om, q, R.f, i, j, k); });
    launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) { gen::advect_wface(v, Sv.f, Om, q, R.f, i, j, k); });
  }
  if (c->p.diffusion != 0) {
    if (!ensure_diff(c)) return;
    gen::Diff d = c->diff;
    const double *rho = S.f[RHO];
    launch_cells_v(c, st, nz + 1, FDiff<1>{q, d, R, rho});
    launch_cells_v(c, st, nz + 1, FDiff<2>{q, d, R, rho});
    launch_cells_v(c, st, nz, FDiff<3>{q, d, R, rho});
    launch_cells_v(c, st, nz + 1, FDiff<4>{q, d, R, rho});
    launch_cells_v(c, st, nz, FDiff<5>{q, d, R, rho});
    launch_cells_v(c, st, nz, FDiff<6>{q, d, R, rho});
    launch_cells_v(c, st, nz + 1, FDiff<7>{q, d, R, rho});
    launch_cells_v(c, st, nz, FDiff<8>{q, d, R, rho});
  }
  launch_cells_v(c, st, nz, FPgBuoy{Sv, R, q, pan});
  if (v.ray_fields)  // Rayleigh damping layer (L219, L622)
    launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::rayleigh_cell(v, Sv.f, R.f, i, j, k); });
  // stage constants for the substeps: theta^t, pi^t
  cudaMemcpyAsync(c->theta_t, q.theta, c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(c->pi_t, q.pi, c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
}

void general_stage_init(erf_ctx *c, cudaStream_t st) {
  F5 S = c->S, St = c->St, P = c->P;
  View v = c->v;
  launch_cells(c, st, c->nz + 1, [=] __device__(int i, int j, int k) {
    size_t a = IX(v, i, j, k);
    if (k < v.nz) {
      P.f[RHO][a] = S.f[RHO][a] - St.f[RHO][a];
      P.f[UU][a] = S.f[UU][a] - St.f[UU][a];
      P.f[VV][a] = S.f[VV][a] - St.f[VV][a];
      P.f[TH][a] = S.f[TH][a] - St.f[TH][a];
    }
    P.f[WW][a] = S.f[WW][a] - St.f[WW][a];
  });
}

void general_stage_finish(erf_ctx *c, cudaStream_t st) {
  F5 St = c->St, P = c->P;
  View v = c->v;
  launch_cells(c, st, c->nz + 1, [=] __device__(int i, int j, int k) {
    size_t a = IX(v, i, j, k);
    if (k < v.nz) {
      St.f[RHO][a] += P.f[RHO][a];
      St.f[UU][a] += P.f[UU][a];
      St.f[VV][a] += P.f[VV][a];
      St.f[TH][a] += P.f[TH][a];
    }
    St.f[WW][a] += P.f[WW][a];
  });
  inflow_impose(c, c->St, st);
  general_lids(c, c->St, st);
}

// n substeps of size dtau about the stage state St (theta_t, pi_t, R, P set by the caller)
void general_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st) {
  View v = c->v;
  const int nz = c->nz;
  gen::Acou A = c->ac;
  A.theta_t = c->theta_t;
  A.pi_t = c->pi_t;
  A.Th_t = St.f[TH];
  for (int m = 0; m < 5; m++) {
    A.R[m] = c->R.f[m];
    A.P[m] = c->P.f[m];
  }
  A.Usum = A.Vsum = A.Omsum = nullptr;
  if (c->sc_Q) {
    A.Usum = c->sc_sum[0]; A.Vsum = c->sc_sum[1]; A.Omsum = c->sc_sum[2];
    for (int m = 0; m < 3; m++) cudaMemsetAsync(c->sc_sum[m], 0, c->NW * sizeof(double), st);
  }
  // Omega'' of the initial S''; Theta''_prev = Theta''
  launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) {
    size_t a = IX(v, i, j, k);
    A.Om[a] = gen::omega_at(v, A.P[UU], A.P[VV], A.P[WW], i, j, k);
    if (k < v.nz) A.Th_prev[a] = A.P[TH][a];
  });
  for (int s = 0; s < n; s++) {
    launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::ac_damp(v, A, i, j, k); });
    launch_cells(c, st, nz, [=] __device__(int i, int j, int k) { gen::ac_horiz(v, A, dtau, i, j, k); });
    launch_cells(c, st, nz + 1, [=] __device__(int i, int j, int k) { gen::ac_slope(v, A, i, j, k); });
    launch_columns(c, st, [=] __device__(int i, int j) { gen::ac_column(v, A, dtau, i, j); });
  }
}

}  // namespace erfb
