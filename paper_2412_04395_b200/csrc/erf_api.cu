// erf_api.cu -- the C-ABI of liberf_b200.so (include/erf_b200.h): context, state copies,
// the RK3 driver (Eq. 11-13; substep schedule L170).
#include <cstdlib>
#include <cstring>
#include <new>
#include <utility>

#include "erf_ctx.cuh"
#include "fused.cuh"

using namespace erfb;

double *erf_ctx::alloc(size_t n) {
  void *p = nullptr;
  if (cudaMalloc(&p, n * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    status = ERF_ENOMEM;
    return nullptr;
  }
  if (cudaMemset(p, 0, n * sizeof(double)) != cudaSuccess) {
    status = ERF_ECUDA;
    cudaFree(p);
    return nullptr;
  }
  allocs.push_back(p);
  bytes += (long long)(n * sizeof(double));
  return (double *)p;
}

// a copy with its own return code checked: a bad caller pointer is reported by the call that was given it
static void copy(erf_ctx *c, void *dst, const void *src, size_t bytes, cudaMemcpyKind kind, cudaStream_t st) {
  if (cudaMemcpyAsync(dst, src, bytes, kind, st) != cudaSuccess) {
    cudaGetLastError();
    c->status = ERF_ECUDA;
  }
}

static int check(erf_ctx *c) {
  if (c->status != ERF_OK) return c->status;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) c->status = ERF_ECUDA;
  return c->status;
}

extern "C" const char *erf_strerror(int code) {
  switch (code) {
    case ERF_OK: return "ok";
    case ERF_EINVAL: return "invalid argument";
    case ERF_EUNSUPPORTED: return "unsupported configuration (the anelastic mode needs a flat, laterally periodic grid and no transported scalar)";
    case ERF_ENOMEM: return "out of memory";
    case ERF_ECUDA: return "CUDA error";
    case ERF_ETOOLARGE: return "nx*ny*nz exceeds ERF_NOALLOC_MAX_VALUES, the fixed work space of erf_poisson_modes_noalloc";
    default: return "unknown error";
  }
}

extern "C" void erf_destroy(erf_ctx *c) {
  if (!c) return;
  cudaDeviceSynchronize();
  fused_release(c);
  for (auto &g : c->graphs) cudaGraphExecDestroy(g.exec);
  for (auto &s : c->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  for (auto e : c->event_pool) cudaEventDestroy(e);
  for (void *p : c->allocs) cudaFree(p);
  delete c;
}

extern "C" int erf_create(const erf_grid *g, const erf_metrics *m, const erf_params *p, void *stream,
                          erf_ctx **out) {
  if (!g || !m || !p || !out) return ERF_EINVAL;
  *out = nullptr;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1 || !(g->dx > 0) || !(g->dy > 0)) return ERF_EINVAL;
  if (!m->rho0 || !m->rhotheta0 || (!m->z_nodes && !m->z_levels)) return ERF_EINVAL;
  if (g->periodic_x < 0 || g->periodic_x > 2 || g->periodic_y < 0 || g->periodic_y > 2) return ERF_EINVAL;
  if (p->adv_order_h < 2 || p->adv_order_h > 6 || p->adv_order_v < 2 || p->adv_order_v > 6) return ERF_EINVAL;
  if (p->diffusion < 0 || p->diffusion > 2 || (p->substep_mode != 0 && p->substep_mode != 1)) return ERF_EINVAL;
  if (!(p->cp > p->Rd) || !(p->Rd > 0) || !(p->p00 > 0)) return ERF_EINVAL;
  if (p->diffusion == 2 && !(p->Pr_t > 0)) return ERF_EINVAL;
  if (p->scalar_adv != 0 && p->scalar_adv != 13 && p->scalar_adv != 15 && p->scalar_adv != 23 && p->scalar_adv != 25)
    return ERF_EINVAL;
  if (p->ray_depth < 0.0 || p->ray_coef < 0.0 || p->ray_fields < 0 || p->ray_fields > 15) return ERF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    cudaGetLastError();
    return ERF_ECUDA;
  }
  cudaStream_t st = (cudaStream_t)stream;
  erf_ctx *c = new (std::nothrow) erf_ctx();
  if (!c) return ERF_ENOMEM;
  c->nx = g->nx; c->ny = g->ny; c->nz = g->nz;
  c->NW = (size_t)g->nx * g->ny * (g->nz + 1);
  c->p = *p;
  c->path = ERF_PATH_AUTO;
  c->status = ERF_OK;
  c->launches = 0;
  c->bytes = 0;
  c->diff_alloc = false;
  c->zl_dev = nullptr;
  c->timing = false;
  c->fz = nullptr;
  c->terr_U2 = c->terr_V2 = c->terr_rdzc = nullptr;
  for (int i = 0; i < ERF_TIMING_CLASSES; i++) { c->t_calls[i] = 0; c->t_ms[i] = 0.0; }
  memset(&c->diff, 0, sizeof(c->diff));
  memset(&c->ac, 0, sizeof(c->ac));

  View &v = c->v;
  memset(&v, 0, sizeof(v));
  v.nx = g->nx; v.ny = g->ny; v.nz = g->nz;
  v.oh = p->adv_order_h; v.ov = p->adv_order_v; v.diffusion = p->diffusion;
  v.osh = p->scalar_adv ? p->scalar_adv : p->adv_order_h;
  v.osv = p->scalar_adv ? p->scalar_adv : p->adv_order_v;
  v.flat = m->z_nodes ? 0 : 1;
  v.perx = g->periodic_x == 1; v.pery = g->periodic_y == 1;
  c->inx = g->periodic_x == 2; c->iny = g->periodic_y == 2;
  c->in_x = c->in_y = nullptr;
  v.ray_fields = p->ray_depth > 0.0 && p->ray_coef > 0.0 ? p->ray_fields : 0;
  v.ray_depth = p->ray_depth; v.ray_coef = p->ray_coef; v.ray_uref = p->ray_uref; v.ray_vref = p->ray_vref;
  v.dx = g->dx; v.dy = g->dy;
  v.Rd = p->Rd; v.cp = p->cp; v.g = p->g; v.p00 = p->p00;
  v.gam = p->cp / (p->cp - p->Rd);    // L82
  v.rdocv = p->Rd / (p->cp - p->Rd);  // Rd/cv
  v.nu = p->diffusion >= 1 ? p->nu : 0.0;
  v.alpha = p->diffusion >= 1 ? p->alpha_theta : 0.0;
  v.Cs = p->Cs; v.Prt = p->Pr_t; v.beta_s = p->beta_s; v.beta_d = p->beta_d;

  c->gen_ready = false;
  c->graph_on = false;
  c->graph_warm = false;
  c->graph_tick = 0;
  c->sc_Q = c->sc_Qt = c->sc_Qnew = c->sc_phi = c->sc_R = nullptr;
  c->sc_sum[0] = c->sc_sum[1] = c->sc_sum[2] = c->sc_G[0] = c->sc_G[1] = nullptr;
  c->an_pp = c->an_tw = c->an_lev = nullptr;
  c->an_w[0] = c->an_w[1] = c->an_w[2] = c->an_w[3] = nullptr;
  c->base1d_r0 = c->base1d_T0 = nullptr;
  c->zxf = c->zyf = c->zw = c->hx = c->hy = c->hc = c->zc = c->hw = c->hu = c->hv = nullptr;
  c->sxw = c->syw = c->sxu = c->syv = c->rho0 = c->Th0 = c->p0 = c->pi0 = c->Om_slow = nullptr;
  memset(&c->prim, 0, sizeof(c->prim));
  c->theta_t = c->alloc(c->NW);
  c->pi_t = c->alloc(c->NW);
  for (int f = 0; f < 5; f++) {
    c->S.f[f] = c->alloc(c->NW);
    c->St.f[f] = c->alloc(c->NW);
    c->R.f[f] = c->alloc(c->NW);
    c->P.f[f] = c->alloc(c->NW);
  }
  if (c->status != ERF_OK) {
    int rc = c->status;
    erf_destroy(c);
    return rc;
  }
  const bool fused_candidate = !m->z_nodes && m->base_is_1d;
  if (fused_candidate) {
    // flat grid, 1-D base state: keep the small inputs; the 3-D general arrays are built only if that path is used
    c->zl_dev = c->alloc(g->nz + 1);
    c->base1d_r0 = c->alloc(g->nz);
    c->base1d_T0 = c->alloc(g->nz);
    if (!c->zl_dev || !c->base1d_r0 || !c->base1d_T0) { int rc = c->status; erf_destroy(c); return rc; }
    copy(c, c->zl_dev, m->z_levels, (g->nz + 1) * sizeof(double), cudaMemcpyHostToDevice, st);
    copy(c, c->base1d_r0, m->rho0, g->nz * sizeof(double), cudaMemcpyDeviceToDevice, st);
    copy(c, c->base1d_T0, m->rhotheta0, g->nz * sizeof(double), cudaMemcpyDeviceToDevice, st);
  } else {
    gen::NodeH Z;
    Z.zn = m->z_nodes; Z.zl = nullptr; Z.nx = g->nx; Z.ny = g->ny;
    if (!m->z_nodes) {
      c->zl_dev = c->alloc(g->nz + 1);
      if (!c->zl_dev) { int rc = c->status; erf_destroy(c); return rc; }
      copy(c, c->zl_dev, m->z_levels, (g->nz + 1) * sizeof(double), cudaMemcpyHostToDevice, st);
      Z.zl = c->zl_dev;
    }
    int rc = build_general(c, Z, m->rho0, m->rhotheta0, m->base_is_1d, st);
    if (rc != ERF_OK) { erf_destroy(c); return rc; }
  }
  int rc = fused_setup(c, m, st);
  if (rc == ERF_OK && !fused_available(c)) rc = ensure_general(c, st);  // e.g. substep_mode 0 on a flat grid
  if (rc == ERF_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = ERF_ECUDA;
  if (rc == ERF_OK) rc = check(c);
  if (rc != ERF_OK) {
    erf_destroy(c);
    return rc;
  }
  *out = c;
  return ERF_OK;
}

extern "C" int erf_set_state(erf_ctx *c, const double *rho, const double *rhou, const double *rhov,
                             const double *rhow, const double *rhotheta, void *stream) {
  if (!c || !rho || !rhou || !rhov || !rhow || !rhotheta) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  size_t nc = (size_t)c->nx * c->ny * c->nz * sizeof(double);
  copy(c, c->S.f[RHO], rho, nc, cudaMemcpyDeviceToDevice, st);
  copy(c, c->S.f[UU], rhou, nc, cudaMemcpyDeviceToDevice, st);
  copy(c, c->S.f[VV], rhov, nc, cudaMemcpyDeviceToDevice, st);
  copy(c, c->S.f[WW], rhow, c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  copy(c, c->S.f[TH], rhotheta, nc, cudaMemcpyDeviceToDevice, st);
  impose_lids(c, c->S, st);
  inflow_store(c, st);
  return check(c);
}

extern "C" int erf_get_state(erf_ctx *c, double *rho, double *rhou, double *rhov, double *rhow,
                             double *rhotheta, void *stream) {
  if (!c) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  size_t nc = (size_t)c->nx * c->ny * c->nz * sizeof(double);
  if (rho) copy(c, rho, c->S.f[RHO], nc, cudaMemcpyDeviceToDevice, st);
  if (rhou) copy(c, rhou, c->S.f[UU], nc, cudaMemcpyDeviceToDevice, st);
  if (rhov) copy(c, rhov, c->S.f[VV], nc, cudaMemcpyDeviceToDevice, st);
  if (rhow) copy(c, rhow, c->S.f[WW], c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  if (rhotheta) copy(c, rhotheta, c->S.f[TH], nc, cudaMemcpyDeviceToDevice, st);
  return check(c);
}

extern "C" int erf_set_path(erf_ctx *c, int path) {
  if (!c || (path != ERF_PATH_AUTO && path != ERF_PATH_GENERAL)) return ERF_EINVAL;
  c->path = path;
  return ERF_OK;
}

static void drain_timing(erf_ctx *c) {
  for (auto &s : c->spans) {
    cudaEventSynchronize(s.b);
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s.a, s.b) == cudaSuccess) {
      c->t_ms[s.id] += ms;
      c->t_calls[s.id]++;
    }
    c->event_pool.push_back(s.a);
    c->event_pool.push_back(s.b);
  }
  c->spans.clear();
}

extern "C" int erf_set_option(erf_ctx *c, int key, long long value) {
  if (!c) return ERF_EINVAL;
  if (key == ERF_OPT_VARIANT) {
    const long long known = ERF_VARIANT_ADV_SPLIT_MASK | ERF_VARIANT_DIFF_SPLIT | ERF_VARIANT_FORCE_COLUMN |
                            ERF_VARIANT_SPLIT_SLOW_RHS | ERF_VARIANT_FORCE_TILE;
    if (value < 0 || (value & ~known)) return ERF_EINVAL;
    if (!c->fz) return ERF_OK;
    if ((value & ERF_VARIANT_SPLIT_SLOW_RHS) && fused_available(c) && !ensure_prim(c, false)) return c->status;
    c->fz->variant = (int)value;
    for (auto &g : c->graphs) cudaGraphExecDestroy(g.exec);  // captured with the previous kernel choice
    c->graphs.clear();
    c->graph_warm = false;
    return ERF_OK;
  }
  if (key == ERF_OPT_GRAPH) {
    if (value != 0 && value != 1) return ERF_EINVAL;
    c->graph_on = value == 1;
    return ERF_OK;
  }
  return ERF_EINVAL;
}

extern "C" int erf_set_timing(erf_ctx *c, int on) {
  if (!c) return ERF_EINVAL;
  c->timing = on != 0;
  return ERF_OK;
}

extern "C" int erf_reset_timing(erf_ctx *c) {
  if (!c) return ERF_EINVAL;
  drain_timing(c);
  for (int i = 0; i < ERF_TIMING_CLASSES; i++) { c->t_calls[i] = 0; c->t_ms[i] = 0.0; }
  return ERF_OK;
}

extern "C" int erf_get_timing(erf_ctx *c, int id, long long *launches, double *total_ms) {
  if (!c || id < 0 || id >= ERF_TIMING_CLASSES) return ERF_EINVAL;
  drain_timing(c);
  if (launches) *launches = c->t_calls[id];
  if (total_ms) *total_ms = c->t_ms[id];
  return check(c);
}

extern "C" const char *erf_timing_name(int id) {
  static const char *names[ERF_TIMING_CLASSES] = {"slow_rhs_general", "acoustic_general", "stage_general",
                                                  "slow_rhs_fused", "viscosity_fused", "acoustic_fused",
                                                  "other", "unused"};
  return (id >= 0 && id < ERF_TIMING_CLASSES) ? names[id] : "?";
}

extern "C" long long erf_launch_count(const erf_ctx *c) { return c ? c->launches : 0; }
extern "C" long long erf_device_bytes(const erf_ctx *c) { return c ? c->bytes : 0; }

// (with a transported scalar the fused substep kernel accumulates the averaged momenta: k_acoustic_flat<.., ACC>)
static bool use_fused(const erf_ctx *c) { return c->path == ERF_PATH_AUTO && fused_available(c); }

extern "C" int erf_set_scalar(erf_ctx *c, const double *rhophi, void *stream) {
  if (!c || !rhophi) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  if (ensure_general(c, st) != ERF_OK || !ensure_scalar(c)) return c->status;
  copy(c, c->sc_Q, rhophi, (size_t)c->nx * c->ny * c->nz * sizeof(double), cudaMemcpyDeviceToDevice, st);
  return check(c);
}

extern "C" int erf_get_scalar(erf_ctx *c, double *rhophi, void *stream) {
  if (!c || !rhophi || !c->sc_Q) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  copy(c, rhophi, c->sc_Q, (size_t)c->nx * c->ny * c->nz * sizeof(double), cudaMemcpyDeviceToDevice,
                  (cudaStream_t)stream);
  return check(c);
}

extern "C" int erf_anelastic_step(erf_ctx *c, double dt, void *stream) {
  if (!c || !(dt > 0.0)) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  if (c->sc_Q) return ERF_EUNSUPPORTED;  // the RK2 step has no scalar stage: refuse rather than leave rho*phi frozen
  int rc = anelastic_step(c, dt, (cudaStream_t)stream);
  return rc != ERF_OK ? rc : check(c);
}

extern "C" int erf_project(erf_ctx *c, double dt, void *stream) {
  if (!c || !(dt > 0.0)) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  int rc = anelastic_project(c, c->S, dt, (cudaStream_t)stream);
  return rc != ERF_OK ? rc : check(c);
}

extern "C" int erf_get_pprime(erf_ctx *c, double *pprime, void *stream) {
  if (!c || !pprime || !c->an_pp) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  copy(c, pprime, c->an_pp, (size_t)c->nx * c->ny * c->nz * sizeof(double), cudaMemcpyDeviceToDevice,
                  (cudaStream_t)stream);
  return check(c);
}

// substep schedule of RK stage s (L170): one substep of dt/3 in stage 1, then ns/2 and ns of dt/ns
static void schedule(int stage, double dt, int ns, int *nsub, double *dtau, double *dts) {
  if (stage == 1) { *nsub = 1; *dtau = dt / 3.0; *dts = dt / 3.0; }
  else if (stage == 2) { *nsub = ns / 2; *dtau = dt / ns; *dts = dt / 2.0; }
  else { *nsub = ns; *dtau = dt / ns; *dts = dt; }
}

// ERF_OPT_GRAPH: the fused step as a CUDA graph.  A step permutes the roles of the context's buffers (S^n <-> S^t,
// the U''/V'' and Theta'' rotations), so one graph is captured per buffer configuration met (a handful) and the
// permutation it causes is replayed on the host pointers after each launch.
static std::vector<const void *> buffer_roles(const erf_ctx *c) {
  std::vector<const void *> r;
  for (int f = 0; f < 5; f++) { r.push_back(c->S.f[f]); r.push_back(c->St.f[f]); r.push_back(c->P.f[f]); }
  fused_buffer_roles(c, r);
  return r;
}
static void set_buffer_roles(erf_ctx *c, const std::vector<const void *> &r) {
  size_t n = 0;
  for (int f = 0; f < 5; f++) {
    c->S.f[f] = (double *)r[n++]; c->St.f[f] = (double *)r[n++]; c->P.f[f] = (double *)r[n++];
  }
  fused_set_buffer_roles(c, r, n);
}

// Graphs are kept for at most GRAPH_KEYS distinct (dt, n_acoustic) pairs; a caller whose dt changes from step to step
// (a CFL-controlled step) would otherwise instantiate graphs without bound.  When a new pair arrives with the cache
// full, every graph of the least recently used pair is destroyed (a graph still executing is released when it ends).
constexpr int GRAPH_KEYS = 4;
static void evict_graphs_for(erf_ctx *c, double dt, int ns) {
  for (;;) {
    std::vector<std::pair<double, int>> keys;
    std::vector<long long> used;
    for (auto &g : c->graphs) {
      size_t n = 0;
      while (n < keys.size() && !(keys[n].first == g.dt && keys[n].second == g.ns)) n++;
      if (n == keys.size()) { keys.push_back({g.dt, g.ns}); used.push_back(g.last_use); }
      else if (g.last_use > used[n]) used[n] = g.last_use;
    }
    bool present = false;
    for (auto &k : keys) present |= k.first == dt && k.second == ns;
    if (present || (int)keys.size() < GRAPH_KEYS) return;
    size_t lru = 0;
    for (size_t n = 1; n < keys.size(); n++)
      if (used[n] < used[lru]) lru = n;
    for (size_t n = c->graphs.size(); n-- > 0;)
      if (c->graphs[n].dt == keys[lru].first && c->graphs[n].ns == keys[lru].second) {
        cudaGraphExecDestroy(c->graphs[n].exec);
        c->graphs.erase(c->graphs.begin() + n);
      }
  }
}

static int graph_step(erf_ctx *c, double dt, int ns, cudaStream_t st) {
  const std::vector<const void *> now = buffer_roles(c);
  for (auto &g : c->graphs)
    if (g.dt == dt && g.ns == ns && g.before == now) {
      g.last_use = ++c->graph_tick;
      if (cudaGraphLaunch(g.exec, st) != cudaSuccess) c->status = ERF_ECUDA;
      set_buffer_roles(c, g.after);
      c->launches += g.launches;
      return check(c);
    }
  if (!c->graph_warm) {
    c->graph_warm = true;
    fused_rk3_step(c, dt, ns, st);
    return check(c);
  }
  evict_graphs_for(c, dt, ns);
  erf_ctx::StepGraph g;
  g.before = now; g.dt = dt; g.ns = ns;
  g.last_use = ++c->graph_tick;
  const long long l0 = c->launches;
  cudaGraph_t graph = nullptr;
  if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();  // the stream cannot be captured (legacy default stream): plain launches
    fused_rk3_step(c, dt, ns, st);
    return check(c);
  }
  fused_rk3_step(c, dt, ns, st);
  if (cudaStreamEndCapture(st, &graph) != cudaSuccess || !graph) { c->status = ERF_ECUDA; return check(c); }
  if (cudaGraphInstantiate(&g.exec, graph, 0) != cudaSuccess) { cudaGraphDestroy(graph); c->status = ERF_ECUDA; return check(c); }
  cudaGraphDestroy(graph);
  g.after = buffer_roles(c);
  g.launches = c->launches - l0;
  c->graphs.push_back(g);
  if (cudaGraphLaunch(g.exec, st) != cudaSuccess) c->status = ERF_ECUDA;
  return check(c);
}

extern "C" int erf_rk3_step(erf_ctx *c, double dt, int n_acoustic, void *stream) {
  if (!c || !(dt > 0.0)) return ERF_EINVAL;
  if (c->p.substep_mode == 1 && (n_acoustic < 2 || (n_acoustic & 1))) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  if (use_fused(c)) {
    if (c->graph_on && !c->timing && !c->sc_Q) return graph_step(c, dt, n_acoustic, st);
    fused_rk3_step(c, dt, n_acoustic, st);
    return check(c);
  }
  if (ensure_general(c, st) != ERF_OK) return c->status;
  for (int f = 0; f < 5; f++)  // S^t = S^n
    copy(c, c->St.f[f], c->S.f[f], c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  if (c->sc_Q) copy(c, c->sc_Qt, c->sc_Q, c->NW * sizeof(double), cudaMemcpyDeviceToDevice, st);
  for (int stage = 1; stage <= 3; stage++) {
    int nsub; double dtau, dts;
    schedule(stage, dt, n_acoustic, &nsub, &dtau, &dts);
    {
      Timed t(c, T_SLOW_GENERAL, st);
      general_slow_rhs(c, c->St, st);  // f(S^t), every stage (L140)
    }
    if (c->p.substep_mode == 0) {
      if (c->sc_Q) {  // Eq. 4 with the stage momenta (L140)
        scalar_stage(c, c->St, c->sc_Qt, c->sc_Q, c->sc_Qnew, 0, dts, st);
        double *t = c->sc_Qt; c->sc_Qt = c->sc_Qnew; c->sc_Qnew = t;
      }
      F5 S = c->S, St = c->St, R = c->R;
      View v = c->v;
      launch_cells(c, st, c->nz + 1, [=] __device__(int i, int j, int k) {
        size_t a = IX(v, i, j, k);
        for (int f = 0; f < 5; f++)
          if (f == WW || k < v.nz) St.f[f][a] = S.f[f][a] + dts * R.f[f][a];
      });
      inflow_impose(c, c->St, st);
      impose_lids(c, c->St, st);
    } else {
      {
        Timed t(c, T_STAGE_GENERAL, st);
        general_stage_init(c, st);  // S'' = S^n - S^t (L581) [R:G7]
      }
      {
        Timed t(c, T_ACOUSTIC_GENERAL, st);
        if (c->path == ERF_PATH_AUTO && terrain_acoustic_available(c) && !c->sc_Q) terrain_acoustic(c, c->St, dtau, nsub, st);
        else general_acoustic(c, c->St, dtau, nsub, st);
      }
      if (c->sc_Q) {  // Eq. 4 after the substeps of the stage (L138), before S^t becomes the stage result
        scalar_stage(c, c->St, c->sc_Qt, c->sc_Q, c->sc_Qnew, nsub, dts, st);
        double *t = c->sc_Qt; c->sc_Qt = c->sc_Qnew; c->sc_Qnew = t;
      }
      {
        Timed t(c, T_STAGE_GENERAL, st);
        general_stage_finish(c, st);  // S = S^t + S'' (L593), lids
      }
    }
  }
  for (int f = 0; f < 5; f++) {
    double *t = c->S.f[f];
    c->S.f[f] = c->St.f[f];
    c->St.f[f] = t;
  }
  if (c->sc_Q) { double *t = c->sc_Q; c->sc_Q = c->sc_Qt; c->sc_Qt = t; }
  return check(c);
}

extern "C" int erf_slow_rhs(erf_ctx *c, double *R_rho, double *R_U, double *R_V, double *R_W, double *R_Theta,
                            void *stream) {
  if (!c) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  if (use_fused(c)) fused_slow_rhs(c, c->S, st);
  else {
    if (ensure_general(c, st) != ERF_OK) return c->status;
    general_slow_rhs(c, c->S, st);
  }
  size_t nc = (size_t)c->nx * c->ny * c->nz * sizeof(double);
  double *out[5] = {R_rho, R_U, R_V, R_W, R_Theta};
  for (int f = 0; f < 5; f++)
    if (out[f])
      copy(c, out[f], c->R.f[f], f == WW ? c->NW * sizeof(double) : nc, cudaMemcpyDeviceToDevice, st);
  return check(c);
}

extern "C" int erf_acoustic(erf_ctx *c, double dtau, int n, const double *R_rho, const double *R_U,
                            const double *R_V, const double *R_W, const double *R_Theta, double *rho_pp,
                            double *U_pp, double *V_pp, double *W_pp, double *Theta_pp, void *stream) {
  if (!c || !R_rho || !R_U || !R_V || !R_W || !R_Theta || !rho_pp || !U_pp || !V_pp || !W_pp || !Theta_pp)
    return ERF_EINVAL;
  if (!(dtau > 0.0) || n < 0) return ERF_EINVAL;
  if (c->status != ERF_OK) return c->status;
  cudaStream_t st = (cudaStream_t)stream;
  size_t nc = (size_t)c->nx * c->ny * c->nz * sizeof(double), nw = c->NW * sizeof(double);
  // stage constants theta^t, pi^t from the current state (the slow-RHS kernels produce them)
  if (use_fused(c)) fused_slow_rhs(c, c->S, st);
  else {
    if (ensure_general(c, st) != ERF_OK) return c->status;
    general_slow_rhs(c, c->S, st);
  }
  const double *Rin[5] = {R_rho, R_U, R_V, R_W, R_Theta};
  double *Pio[5] = {rho_pp, U_pp, V_pp, W_pp, Theta_pp};
  for (int f = 0; f < 5; f++) {
    copy(c, c->R.f[f], Rin[f], f == WW ? nw : nc, cudaMemcpyDeviceToDevice, st);
    copy(c, c->P.f[f], Pio[f], f == WW ? nw : nc, cudaMemcpyDeviceToDevice, st);
  }
  if (use_fused(c)) fused_acoustic(c, c->S, dtau, n, st);
  else if (c->path == ERF_PATH_AUTO && terrain_acoustic_available(c)) terrain_acoustic(c, c->S, dtau, n, st);
  else general_acoustic(c, c->S, dtau, n, st);
  for (int f = 0; f < 5; f++)
    copy(c, Pio[f], c->P.f[f], f == WW ? nw : nc, cudaMemcpyDeviceToDevice, st);
  return check(c);
}
