// fused.cuh -- the fused flat-grid kernels (k_fused_*.cu) and their per-context state.
//
// "Flat" = z_nodes == NULL (level heights depend on k only) with a 1-D base state: every
// metric term is a per-level constant (hx = hy = hc = dz(k), slopes = 0, Omega = W), so
// the column operators read short per-level tables instead of 3-D metric fields.
#pragma once
#include <cuda.h>

#include <map>
#include <vector>

#include "erf_ctx.cuh"

namespace erfb {

// per-level tables (device, length nz+1 each)
struct LevelTables {
  const double *dz;     // [k] cell thickness hc(k), k < nz
  const double *rdz;    // [k] 1/hc(k)
  const double *rhw;    // [k] 1/hw(k), k = 1..nz-1 (centre-to-centre spacing)
  const double *tabB;   // [k] rho0f(k) * (Rd/cv) / pi0f(k) at w-face k = 1..nz-1
  const double *rho0;   // [k] base-state density
  const double *Th0;    // [k] base-state rho*theta
  const double *rTh0;   // [k] 1/Th0
  const double *p0;     // [k] base-state pressure (Eq. 7)
  const double *pi0;    // [k] base-state Exner function
  const double *csd2;   // [k] (Cs Delta)^2, Delta = (dx dy dz_k)^(1/3)  [R:G9]
  const double *tauc;   // [k] Rayleigh damping rate at cell centres (L622) [R:G28]
  const double *tauw;   // [k] ... and at w-faces
};

struct FusedState {
  bool ok;            // fused kernels cover this context
  LevelTables tab;
  double *iT;         // 1/Theta^t (stage constant)
  double *U2, *V2;    // second buffers of U'', V'' (ping-pong across substeps)
  double *Thd[2];     // with P.Theta the three rotating Theta'' buffers (current, previous, next)
  double *cp_scr;     // Thomas c' of the thread-per-column substep kernel (stage constant)
  double *mu, *Kd;    // dynamic viscosity and scalar diffusivity at cell centres (diffusion != 0)
  std::map<const void *, CUtensorMap> tmaps;  // TMA tensor maps of the state buffers (k_slow_adv.cu)
  int ray_k0;         // first level with a non-zero Rayleigh rate (nz: none)
  int variant;        // ERF_VARIANT_* mask (erf_set_option, diagnostics block of erf_b200.h); 0 = defaults
};

int fused_setup(erf_ctx *c, const erf_metrics *m, cudaStream_t st);
void fused_release(erf_ctx *c);
bool fused_available(const erf_ctx *c);
void fused_rk3_step(erf_ctx *c, double dt, int n_acoustic, cudaStream_t st);
void fused_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st);
void fused_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st);
// the fused path's own rotating buffers, appended to / restored from the list erf_api.cu keeps per CUDA graph
void fused_buffer_roles(const erf_ctx *c, std::vector<const void *> &r);
void fused_set_buffer_roles(erf_ctx *c, const std::vector<const void *> &r, size_t n);

// k_fused_slow.cu
void launch_slow_flat(erf_ctx *c, const F5 &S, cudaStream_t st);

}  // namespace erfb
