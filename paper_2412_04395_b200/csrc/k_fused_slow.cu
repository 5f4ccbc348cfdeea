// k_fused_slow.cu -- slow right-hand side f(S) on flat grids (Eq. 1-3).
#include "fused.cuh"

namespace erfb {

__global__ void k_inv_theta(size_t n, const double *Th, double *iT) {
  size_t a = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (a < n) iT[a] = 1.0 / Th[a];
}

void launch_slow_flat(erf_ctx *c, const F5 &S, cudaStream_t st) {
  Timed t(c, T_SLOW_FUSED, st);
  general_slow_rhs(c, S, st);
  size_t n = (size_t)c->nx * c->ny * c->nz;
  k_inv_theta<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, S.f[TH], c->fz->iT);
  c->launches++;
}

}  // namespace erfb
