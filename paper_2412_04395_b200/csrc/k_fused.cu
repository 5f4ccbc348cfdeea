// k_fused.cu -- set-up and RK3 driver of the fused flat-grid path.
#include <cstdlib>
#include <cstring>

#include "fused.cuh"

namespace erfb {

// per-level tables from column (0,0) of the 3-D geometry / base-state fields
__global__ void k_level_tables(View v, double *dz, double *rdz, double *rhw, double *tabB, double *rho0,
                               double *Th0, double *rTh0, double *p0, double *pi0, double *csd2) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > v.nz) return;
  size_t a = (size_t)k * v.ny * v.nx;
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
  FusedState *z = new FusedState();
  memset(z, 0, sizeof(*z));
  c->fz = z;
  z->ok = c->v.flat && m->base_is_1d && c->p.substep_mode == 1;
  if (const char *e = getenv("ERF_B200_VARIANT")) z->variant = atoi(e);  // developer tuning knob
  if (!z->ok) return ERF_OK;
  const int nl = c->nz + 1;
  double *t[10];
  for (auto &p : t) {
    p = c->alloc(nl);
    if (!p) return c->status;
  }
  k_level_tables<<<(nl + 127) / 128, 128, 0, st>>>(c->v, t[0], t[1], t[2], t[3], t[4], t[5], t[6], t[7],
                                                       t[8], t[9]);
  c->launches++;
  z->tab = LevelTables{t[0], t[1], t[2], t[3], t[4], t[5], t[6], t[7], t[8], t[9]};
  double **arr[] = {&z->iT, &z->U2, &z->V2, &z->Thd[0], &z->Thd[1], &z->cp_scr};
  for (auto p : arr) {
    *p = c->alloc(c->NW);
    if (!*p) return c->status;
  }
  if (c->p.diffusion != 0) {
    z->mu = c->alloc(c->NW);
    z->Kd = c->alloc(c->NW);
    if (!z->mu || !z->Kd) return c->status;
  }
  return ERF_OK;
}

void fused_release(erf_ctx *c) {
  delete c->fz;
  c->fz = nullptr;
}

bool fused_available(const erf_ctx *c) { return c->fz && c->fz->ok; }

// S'' = S^n - S^t (L581) [R:G7]; Theta''_d = Theta'' (Theta''_prev = Theta'' at the start of a stage)
__global__ void k_stage_init_flat(size_t nc, size_t nw, F5 S, F5 St, F5 P, double *thd) {
  size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= nw) return;
  P.f[WW][a] = S.f[WW][a] - St.f[WW][a];
  if (a < nc) {
    P.f[RHO][a] = S.f[RHO][a] - St.f[RHO][a];
    P.f[UU][a] = S.f[UU][a] - St.f[UU][a];
    P.f[VV][a] = S.f[VV][a] - St.f[VV][a];
    double t = S.f[TH][a] - St.f[TH][a];
    P.f[TH][a] = t;
    thd[a] = t;
  }
}

// S = S^t + S'' (L593); flat lids: W = 0 at k = 0 and k = nz
__global__ void k_stage_finish_flat(size_t nc, size_t nw, size_t plane, F5 St, F5 P) {
  size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= nw) return;
  St.f[WW][a] = (a < plane || a >= nc) ? 0.0 : St.f[WW][a] + P.f[WW][a];
  if (a < nc) {
    St.f[RHO][a] += P.f[RHO][a];
    St.f[UU][a] += P.f[UU][a];
    St.f[VV][a] += P.f[VV][a];
    St.f[TH][a] += P.f[TH][a];
  }
}

void fused_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st) { launch_slow_flat(c, S, st); }

void fused_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st) {
  if (acoustic_zc_available(c)) {
    launch_acoustic_zc(c, dtau, n, 0, st);
    return;
  }
  // entry for erf_acoustic: Theta''_prev = Theta'' => Theta''_d = Theta''
  cudaMemcpyAsync(c->fz->Thd[0], c->P.f[TH], c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  launch_acoustic_flat(c, St, dtau, n, st);
}

void fused_rk3_step(erf_ctx *c, double dt, int ns, cudaStream_t st) {
  const size_t plane = (size_t)c->nx * c->ny, nc = plane * c->nz, nw = c->NW;
  const unsigned blocks = (unsigned)((nw + 255) / 256);
  const bool zc = acoustic_zc_available(c);
  if (!zc)
    for (int f = 0; f < 5; f++)  // S^t = S^n
      cudaMemcpyAsync(c->St.f[f], c->S.f[f], nw * sizeof(double), cudaMemcpyDeviceToDevice, st);
  for (int stage = 1; stage <= 3; stage++) {
    int nsub = stage == 1 ? 1 : (stage == 2 ? ns / 2 : ns);  // L170
    double dtau = stage == 1 ? dt / 3.0 : dt / ns;
    if (zc) {
      // f(S^t) every stage (L140), S^t = S^n in stage 1; the substep kernels form S'' = S^n - S^t at their first
      // launch and write S^t + S'' at their last (L581, L593)
      launch_slow_flat(c, stage == 1 ? c->S : c->St, st);
      launch_acoustic_zc(c, dtau, nsub, stage, st);
      continue;
    }
    launch_slow_flat(c, c->St, st);  // also theta^t, pi^t, 1/Theta^t
    {
      Timed t(c, T_OTHER, st);
      k_stage_init_flat<<<blocks, 256, 0, st>>>(nc, nw, c->S, c->St, c->P, c->fz->Thd[0]);
      c->launches++;
    }
    launch_acoustic_flat(c, c->St, dtau, nsub, st);
    {
      Timed t(c, T_OTHER, st);
      k_stage_finish_flat<<<blocks, 256, 0, st>>>(nc, nw, plane, c->St, c->P);
      c->launches++;
    }
  }
  for (int f = 0; f < 5; f++) {
    double *t = c->S.f[f];
    c->S.f[f] = c->St.f[f];
    c->St.f[f] = t;
  }
}

}  // namespace erfb
