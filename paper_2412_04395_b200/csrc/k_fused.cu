// k_fused.cu -- fused flat-grid kernels (placeholder until the first fused kernel lands).
#include "fused.cuh"

namespace erfb {

int fused_setup(erf_ctx *, const erf_metrics *, cudaStream_t) { return ERF_OK; }
void fused_release(erf_ctx *) {}
bool fused_available(const erf_ctx *) { return false; }
void fused_rk3_step(erf_ctx *, double, int, cudaStream_t) {}
void fused_slow_rhs(erf_ctx *, const F5 &, cudaStream_t) {}
void fused_acoustic(erf_ctx *, const F5 &, double, int, cudaStream_t) {}

}  // namespace erfb
