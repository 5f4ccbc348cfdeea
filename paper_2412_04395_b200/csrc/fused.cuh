// fused.cuh -- interface of the fused flat-grid kernels (k_fused_*.cu).
#pragma once
#include "erf_ctx.cuh"

namespace erfb {

// allocate / precompute what the fused kernels need; called at the end of erf_create
int fused_setup(erf_ctx *c, const erf_metrics *m, cudaStream_t st);
void fused_release(erf_ctx *c);
// true when the fused kernels cover this context's grid and parameters
bool fused_available(const erf_ctx *c);
void fused_rk3_step(erf_ctx *c, double dt, int n_acoustic, cudaStream_t st);
void fused_slow_rhs(erf_ctx *c, const F5 &S, cudaStream_t st);
void fused_acoustic(erf_ctx *c, const F5 &St, double dtau, int n, cudaStream_t st);

}  // namespace erfb
