// k_scalar.cu -- one transported scalar rho*phi (Eq. 4).
//
// "Equations 4-6 do not directly participate in the substepping; these variables are advanced as if there is no
// substepping, with the exception that the normal momenta used to define the advective fluxes is the time average
// over the RK stage of the intermediate (rho u . n) values used to advance rho each substep" (L138).  So per stage:
//     Q_stage = Q^n + dt_s [ -div(Mbar phi^t) + div(K grad phi^t) ],   phi^t = Q^t / rho^t,
// Mbar = stage momenta + (1/n) sum over the substeps of (U''new, V''new, beta2 Omega''new + beta1 Omega''old) -- the
// fluxes of the substepped continuity equation (Appendix A, L585 row 5 with L591), accumulated by the substep kernels
// (general_cells.cuh: ac_horiz, ac_column).  With them a constant phi stays constant to round-off.  phi is interpolated
// like theta (Eq. 17-21, order reduction at the lids [R:G13]); it diffuses with theta's K, conservative form [R:G25].
//
// The scalar stage itself runs on the terrain-general data path (thread per cell, mass fluxes and vertical quotients
// formed on the fly).  The momenta come from the substep kernels of whichever path runs the step: the general passes, or
// the fused flat-grid kernel k_acoustic_flat<.., ACC = true>.  On the fused path the last substep of a stage overwrites
// the stage state, so there the sums are started at n times the stage momenta ("folded") and phi^t is formed before the
// substeps (scalar_prepare_fused); the stage then needs nothing of S^t.
#include "fused.cuh"
#include "slow_flat.cuh"

namespace erfb {

namespace {

struct Sc {
  const double *rho, *U, *V, *W;     // stage state S^t
  const double *Us, *Vs, *Oms;       // sums over the substeps (null without substepping)
  double rn;                         // 1 / number of substeps
  bool folded;                       // the sums already hold n times the stage momenta (U, V, W are null)
  bool diffuse;
  const double *Qt, *Qn, *K;
  double *phi, *Gx, *Gy, *R, *Qout;
  double dts;
};

template <class VT>
__device__ __forceinline__ double mx(const VT &v, const Sc &s, int i, int j, int k) {  // averaged mass flux, x-face i
  const size_t a = IX(v, i, j, k);
  if (s.folded) return v.hx[a] * (s.rn * s.Us[a]);
  return v.hx[a] * (s.U[a] + (s.Us ? s.rn * s.Us[a] : 0.0));
}
template <class VT>
__device__ __forceinline__ double my(const VT &v, const Sc &s, int i, int j, int k) {
  const size_t a = IX(v, i, j, k);
  if (s.folded) return v.hy[a] * (s.rn * s.Vs[a]);
  return v.hy[a] * (s.V[a] + (s.Vs ? s.rn * s.Vs[a] : 0.0));
}
template <class VT>
__device__ __forceinline__ double mz(const VT &v, const Sc &s, int i, int j, int k) {  // averaged Omega, w-face k
  if (k < 1 || k > v.nz - 1) return 0.0;
  if (s.folded) return s.rn * s.Oms[IX(v, i, j, k)];  // flat grid: Omega = W
  return gen::omega_at(v, s.U, s.V, s.W, i, j, k) + (s.Oms ? s.rn * s.Oms[IX(v, i, j, k)] : 0.0);
}

// mean vertical difference quotient of phi around level k at the two columns (ia, ja), (ib, jb): faces k and k+1
// where they are interior (the chain-rule term of a horizontal derivative [R:G14])
template <class VT>
__device__ __forceinline__ double dz_mean(const VT &v, const Sc &s, int ia, int ja, int ib, int jb, int k) {
  double sum = 0.0;
  int n = 0;
  for (int kk = k; kk <= k + 1; kk++)
    if (kk >= 1 && kk <= v.nz - 1) {
      const size_t a = IX(v, ia, ja, kk), b = IX(v, ib, jb, kk);
      sum += (s.phi[a] - s.phi[IX(v, ia, ja, kk - 1)]) / v.hw[a] + (s.phi[b] - s.phi[IX(v, ib, jb, kk - 1)]) / v.hw[b];
      n += 2;
    }
  return n ? sum / n : 0.0;
}

struct FPhi {
  Sc s;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    const size_t a = IX(v, i, j, k);
    s.phi[a] = s.Qt[a] / s.rho[a];
  }
};

struct FAdvect {
  Sc s;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    const size_t a = IX(v, i, j, k);
    const double fxm = mx(v, s, i, j, k), fxp = mx(v, s, i + 1, j, k), fym = my(v, s, i, j, k), fyp = my(v, s, i, j + 1, k);
    const double omm = mz(v, s, i, j, k), omp = mz(v, s, i, j, k + 1);
    const double ax = fxp * gen::interp_x(v, s.phi, i + 1, j, k, v.osh, fxp) - fxm * gen::interp_x(v, s.phi, i, j, k, v.osh, fxm);
    const double ay = fyp * gen::interp_y(v, s.phi, i, j + 1, k, v.osh, fyp) - fym * gen::interp_y(v, s.phi, i, j, k, v.osh, fym);
    const double zt = (k + 1 <= v.nz - 1) ? omp * gen::interp_z(v, s.phi, i, j, k + 1, 0, v.nz - 1, v.osv, omp) : 0.0;
    const double zb = (k >= 1) ? omm * gen::interp_z(v, s.phi, i, j, k, 0, v.nz - 1, v.osv, omm) : 0.0;
    const double R = -(ax / v.dx + ay / v.dy + (zt - zb)) / v.hc[a];
    if (s.diffuse) s.R[a] = R;
    else s.Qout[a] = s.Qn[a] + s.dts * R;
  }
};

// The same advective tendency with a compile-time horizontal order, the lateral offsets wrapped / clamped once per
// thread and flux = M q_even - |M| q_odd (as tslow::k_adv_terrain does for theta); Eq. 17-21 only.
template <int OH>
__global__ void __launch_bounds__(256) k_scalar_adv(View v, Sc s) {
  const int i = blockIdx.y * 32 + threadIdx.x, j = blockIdx.z * 8 + threadIdx.y, k = blockIdx.x;
  const int nx = v.nx, ny = v.ny, nz = v.nz;
  if (i >= nx || j >= ny) return;
  const size_t plane = (size_t)nx * ny, kb = (size_t)k * plane;
  int xo[7];
  size_t yo[7];
#pragma unroll
  for (int n = 0; n < 7; n++) {
    xo[n] = lati(i + n - 3, nx, v.perx);
    yo[n] = (size_t)lati(j + n - 3, ny, v.pery) * nx;
  }
  const size_t oc = yo[3] + xo[3], a = kb + oc;
  const double fxm = mx(v, s, i, j, k), fxp = mx(v, s, i + 1, j, k), fym = my(v, s, i, j, k), fyp = my(v, s, i, j + 1, k);
  const double omm = mz(v, s, i, j, k), omp = mz(v, s, i, j, k + 1);
  double q[7];
#pragma unroll
  for (int n = 0; n < 7; n++) q[n] = s.phi[kb + yo[3] + xo[n]];
  double acc = (flux_c<OH>(fxp, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(fxm, q[0], q[1], q[2], q[3], q[4], q[5])) / v.dx;
#pragma unroll
  for (int n = 0; n < 7; n++) q[n] = s.phi[kb + yo[n] + xo[3]];
  acc += (flux_c<OH>(fyp, q[1], q[2], q[3], q[4], q[5], q[6]) - flux_c<OH>(fym, q[0], q[1], q[2], q[3], q[4], q[5])) / v.dy;
#pragma unroll
  for (int n = 0; n < 7; n++) q[n] = s.phi[(size_t)min(max(k + n - 3, 0), nz - 1) * plane + oc];
  const double zt = (k + 1 <= nz - 1) ? flux_rt(vorder(v.ov, min(k + 1, nz - k - 1)), omp, q + 1) : 0.0;
  const double zb = (k >= 1) ? flux_rt(vorder(v.ov, min(k, nz - k)), omm, q) : 0.0;
  const double R = -(acc + (zt - zb)) / v.hc[a];
  if (s.diffuse) s.R[a] = R;
  else s.Qout[a] = s.Qn[a] + s.dts * R;
}

struct FHFlux {  // diffusive fluxes through the x- and y-faces
  Sc s;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    const size_t a = IX(v, i, j, k), mxi = IX(v, i - 1, j, k), myi = IX(v, i, j - 1, k);
    // (on a flat grid the slopes vanish identically: the chain-rule terms are skipped, not multiplied by zero)
    const double dxp = (s.phi[a] - s.phi[mxi]) / v.dx - (v.flat ? 0.0 : v.sxu[a] * dz_mean(v, s, i - 1, j, i, j, k));
    const double dyp = (s.phi[a] - s.phi[myi]) / v.dy - (v.flat ? 0.0 : v.syv[a] * dz_mean(v, s, i, j - 1, i, j, k));
    s.Gx[a] = -0.5 * (s.K[mxi] + s.K[a]) * dxp;
    s.Gy[a] = -0.5 * (s.K[myi] + s.K[a]) * dyp;
  }
};

struct FDiffuse {
  Sc s;
  template <class VT> __device__ void operator()(const VT &v, int i, int j, int k) const {
    const size_t a = IX(v, i, j, k), ip = IX(v, i + 1, j, k), jp = IX(v, i, j + 1, k);
    // contravariant vertical flux through w-face kk (zero on the lids)
    auto gz = [&](int kk) -> double {
      if (kk < 1 || kk > v.nz - 1) return 0.0;
      const size_t f = IX(v, i, j, kk), b = IX(v, i, j, kk - 1);
      const double fz = -0.5 * (s.K[b] + s.K[f]) * ((s.phi[f] - s.phi[b]) / v.hw[f]);
      if (v.flat) return fz;
      const double gxb = 0.25 * (s.Gx[b] + s.Gx[IX(v, i + 1, j, kk - 1)] + s.Gx[f] + s.Gx[IX(v, i + 1, j, kk)]);
      const double gyb = 0.25 * (s.Gy[b] + s.Gy[IX(v, i, j + 1, kk - 1)] + s.Gy[f] + s.Gy[IX(v, i, j + 1, kk)]);
      return fz - v.sxw[f] * gxb - v.syw[f] * gyb;
    };
    const double div = ((v.hx[ip] * s.Gx[ip] - v.hx[a] * s.Gx[a]) / v.dx + (v.hy[jp] * s.Gy[jp] - v.hy[a] * s.Gy[a]) / v.dy +
                        (gz(k + 1) - gz(k))) / v.hc[a];
    s.Qout[a] = s.Qn[a] + s.dts * (s.R[a] - div);
  }
};

}  // namespace

// Q_stage from Q^t (stage value) and Q^n; nsub = 0: no substepping (the stage momenta advect)
void scalar_stage(erf_ctx *c, const F5 &St, const double *Qt, const double *Qn, double *Qout, int nsub, double dts,
                  cudaStream_t st, bool folded) {
  Sc s;
  s.folded = folded;
  s.rho = St.f[RHO]; s.U = St.f[UU]; s.V = St.f[VV]; s.W = St.f[WW];
  s.Us = nsub ? c->sc_sum[0] : nullptr; s.Vs = nsub ? c->sc_sum[1] : nullptr; s.Oms = nsub ? c->sc_sum[2] : nullptr;
  s.rn = nsub ? 1.0 / nsub : 0.0;
  s.Qt = Qt; s.Qn = Qn; s.K = c->p.diffusion != 0 ? (folded ? c->fz->Kd : c->diff.K) : nullptr;
  s.phi = c->sc_phi; s.R = c->sc_R; s.Qout = Qout;
  s.Gx = folded ? c->sc_G[0] : c->diff.Fx; s.Gy = folded ? c->sc_G[1] : c->diff.Fy;
  s.dts = dts;
  s.diffuse = c->p.diffusion != 0;
  const int nz = c->nz;
  if (!folded) launch_cells_v(c, st, nz, FPhi{s});
  if (c->v.osh == c->v.oh && c->v.osv == c->v.ov) {
    dim3 block(32, 8), grid(nz, (c->nx + 31) / 32, (c->ny + 7) / 8);
    switch (c->v.oh) {
      case 2: k_scalar_adv<2><<<grid, block, 0, st>>>(c->v, s); break;
      case 3: k_scalar_adv<3><<<grid, block, 0, st>>>(c->v, s); break;
      case 4: k_scalar_adv<4><<<grid, block, 0, st>>>(c->v, s); break;
      case 5: k_scalar_adv<5><<<grid, block, 0, st>>>(c->v, s); break;
      default: k_scalar_adv<6><<<grid, block, 0, st>>>(c->v, s); break;
    }
    c->launches++;
  } else {
    launch_cells_v(c, st, nz, FAdvect{s});  // WENO (L213)
  }
  if (!s.diffuse) return;
  launch_cells_v(c, st, nz, FHFlux{s});
  launch_cells_v(c, st, nz, FDiffuse{s});
}

// fused flat path, before the substeps of a stage: phi^t = Q^t / rho^t and the sums started at n times the stage momenta
void scalar_prepare_fused(erf_ctx *c, const F5 &St, const double *Qt, int nsub, cudaStream_t st) {
  const View v = c->v;
  const double *rho = St.f[RHO], *U = St.f[UU], *V = St.f[VV], *W = St.f[WW];
  double *phi = c->sc_phi, *sU = c->sc_sum[0], *sV = c->sc_sum[1], *sO = c->sc_sum[2];
  const double n = (double)nsub;
  launch_cells(c, st, c->nz + 1, [=] __device__(int i, int j, int k) {
    const size_t a = IX(v, i, j, k);
    if (k < v.nz) {
      phi[a] = Qt[a] / rho[a];
      sU[a] = n * U[a];
      sV[a] = n * V[a];
    }
    sO[a] = n * W[a];
  });
}

// first use: the scalar, its two stage buffers, the three momentum sums and two work arrays
bool ensure_scalar(erf_ctx *c) {
  if (c->sc_Q) return true;
  double **arr[] = {&c->sc_Q, &c->sc_Qt, &c->sc_Qnew, &c->sc_sum[0], &c->sc_sum[1], &c->sc_sum[2], &c->sc_phi, &c->sc_R,
                    &c->sc_G[0], &c->sc_G[1]};
  for (auto p : arr) {
    *p = c->alloc(c->NW);
    if (!*p) return false;
  }
  return true;
}

}  // namespace erfb
