// slow_flat.cuh -- parameter block and the Eq. 17-21 flux functions shared by the flat-grid slow-RHS kernels.
#pragma once
#include "fused.cuh"

namespace erfb {

struct SlowFlat {
  int nx, ny, nz, ov;
  double rdx, rdy, g;
  const double *rho, *U, *V, *W, *Th;
  double *theta, *u, *v, *w, *pp, *pi, *iT;
  double *Rrho, *RU, *RV, *RW, *RTh;
  double *mu, *K;
  const double *dz, *rdz, *rhw, *rho0, *Th0, *rTh0, *p0, *pi0, *csd2;
  double gam, rdocv, nu, alpha, rPrt;
  int diffusion;
  int use_tma;  // k_slow_adv: tensor maps are valid
};

// ------------------------------------------------------------------ Eq. 17-21
// q0..q5 = q_{m-3} .. q_{m+2}, flux point m-1/2; returns M * q_interp with the upwind sign of M:
// flux = M q_even - |M| q_odd  (Eq. 20-21 with sgn = sign(M); Eq. 21 repaired [R:G1])
template <int ORD>
__device__ __forceinline__ double flux_c(double M, double q0, double q1, double q2, double q3, double q4, double q5) {
  const double s2 = q3 + q2;
  if (ORD == 2) return M * (0.5 * s2);
  const double s4 = q4 + q1;
  const double q4th = (7.0 / 12.0) * s2 - (1.0 / 12.0) * s4;
  if (ORD == 4) return M * q4th;
  if (ORD == 3) return M * q4th + fabs(M) * ((1.0 / 12.0) * ((q4 - q1) - 3.0 * (q3 - q2)));
  const double q6th = (37.0 / 60.0) * s2 - (2.0 / 15.0) * s4 + (1.0 / 60.0) * (q5 + q0);
  if (ORD == 6) return M * q6th;
  return M * q6th - fabs(M) * ((1.0 / 60.0) * ((q5 - q0) - 5.0 * (q4 - q1) + 10.0 * (q3 - q2)));
}

__device__ __forceinline__ double flux_rt(int ord, double M, const double *q) {
  switch (ord) {
    case 2: return flux_c<2>(M, q[0], q[1], q[2], q[3], q[4], q[5]);
    case 3: return flux_c<3>(M, q[0], q[1], q[2], q[3], q[4], q[5]);
    case 4: return flux_c<4>(M, q[0], q[1], q[2], q[3], q[4], q[5]);
    case 5: return flux_c<5>(M, q[0], q[1], q[2], q[3], q[4], q[5]);
    default: return flux_c<6>(M, q[0], q[1], q[2], q[3], q[4], q[5]);
  }
}

// order next to the lids [R:G13]; r = min(#valid points below, above)
__device__ __forceinline__ int vorder(int req, int r) {
  const int need = (req + 1) >> 1;
  if (r >= need) return req;
  if (r >= 2 && req >= 3) return (req & 1) ? 3 : 4;
  return 2;
}

// k_slow_adv.cu: primitives + advection + pressure gradient + buoyancy in one kernel (needs nx even)
bool slow_adv_available(const erf_ctx *c);
void launch_slow_adv(erf_ctx *c, const SlowFlat &p, cudaStream_t st);

// k_slow_tiled.cu
void launch_adv_diff_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st);
void launch_diff_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st);
void launch_visc_tiled(erf_ctx *c, const SlowFlat &p, cudaStream_t st);

}  // namespace erfb
