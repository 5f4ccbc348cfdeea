// k_noalloc.cu -- erf_poisson_modes_noalloc: the vertical solve of the anelastic Poisson equation (Sec. 3.2
// Eq. 16; reading G29) for callers that must not allocate device memory.
//
// Who that is.  A library call that ends in cudaMalloc is off limits for code that runs while device memory is not the
// caller's to take: a time loop inside a host application (PyTorch, a weather model with its own arena) that has handed
// the whole card to its own allocator, so that a cudaMalloc from a guest library fails or fragments what is left; a job
// that runs under a fixed per-process memory budget which its own buffers already fill; a latency-bound loop that
// cannot take the device-wide synchronisation cudaMalloc / cudaFree imply.  Such a caller brings every input and output
// buffer itself.  What it cannot bring is the solver's own work space, and this file supplies that from the library
// image instead of from the heap.
//
// The operation is the one k_anelastic.cu's k_modes carries out in the middle of erf_project: after the horizontal
// transforms, one real tridiagonal system in z per horizontal mode (m, n),
//     [lx(m) + ly(n)] P_k + [ (P_{k+1} - P_k)/dzw_{k+1} - (P_k - P_{k-1})/dzw_k ] / dz_k = Dhat_k / dt,
//     lx(m) = -(4/dx^2) sin^2(pi m / nx),  ly(n) = -(4/dy^2) sin^2(pi n / ny),   mode (0, 0): P_0 = 0,
// solved by the Thomas algorithm, real and imaginary part with the same coefficients.  The forward sweep leaves one
// value c' per (mode, level) that the backward sweep reads again: nx*ny*nz doubles of scratch.  In erf_project that
// scratch is a cudaMalloc'ed work array of the context; here it is the file-scope array below.
//
// The array.  ERF_NOALLOC_MAX_VALUES doubles (8 MiB) that are part of liberf_b200.so's device image: every GPU on
// which the process uses the library carries them from the moment the image is loaded there until the process exits,
// whether or not this entry point is ever called.  There is one array per GPU, not per call: all calls on a GPU share
// it, it still holds the previous call's c' when the next call starts, and two calls that can run at the same time on
// one GPU (different streams, different host threads) overwrite each other's c' and return garbage without any error.
// Nothing in it has to start at zero: the forward sweep writes c'(k) of a mode before the backward sweep of that same
// mode reads it, and no thread reads an entry it has not written in the same launch, so stale contents are harmless.
//
// Host-side name versus device address.  In host code `g_cprime` is only a handle for the runtime, not a device
// pointer; the address the kernel needs comes from cudaGetSymbolAddress, asked once per GPU with that GPU current
// (noalloc_scratch below), and is handed to the kernel as an ordinary argument.
#include <cuda_runtime.h>

#include <mutex>

#include "../../include/erf_b200.h"

namespace erfb {
namespace noalloc {

static __device__ __align__(256) double g_cprime[ERF_NOALLOC_MAX_VALUES];

constexpr double PI = 3.14159265358979323846;
constexpr int MAX_DEVICES = 64;
static std::mutex g_mu;
static double *g_addr[MAX_DEVICES];  // device address of g_cprime on GPU d; null until the first call there

// The device address of this GPU's copy of g_cprime (null + *err set on failure).  The first call on a GPU asks the
// runtime; that may also make the runtime load the library's device image onto the GPU, which is why the header asks
// for the first call to happen outside any stream capture.
static double *noalloc_scratch(cudaError_t *err) {
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  if (dev < 0 || dev >= MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    double *p = nullptr;
    *err = cudaGetSymbolAddress((void **)&p, g_cprime);
    if (*err != cudaSuccess) return nullptr;
    g_addr[dev] = p;
  }
  return g_addr[dev];
}

// One thread per horizontal mode; the arithmetic of anel::k_modes (k_anelastic.cu) with the level metrics as two
// arrays and c' in `cp`, the static array's device address.
__global__ void __launch_bounds__(256) k_modes_static(int nx, int ny, int nz, double dx, double dy, double rdt,
                                                      const double *__restrict__ dz, const double *__restrict__ dzw,
                                                      double *br, double *bi, double *cp) {
  const int m = blockIdx.x * 32 + threadIdx.x, n = blockIdx.y * 8 + threadIdx.y;
  if (m >= nx || n >= ny) return;
  const size_t nh = (size_t)nx * ny, o = (size_t)n * nx + m;
  const double sx = sin(PI * m / nx), sy = sin(PI * n / ny);
  const double lam = -4.0 * sx * sx / (dx * dx) - 4.0 * sy * sy / (dy * dy);
  double cpm = 0.0, drm = 0.0, dim = 0.0;
  for (int k = 0; k < nz; k++) {
    double lo = k >= 1 ? 1.0 / (dzw[k] * dz[k]) : 0.0;
    double up = k <= nz - 2 ? 1.0 / (dzw[k + 1] * dz[k]) : 0.0;
    double diag = lam - lo - up;
    double rr = br[k * nh + o] * rdt, ri = bi[k * nh + o] * rdt;
    if (m == 0 && n == 0 && k == 0) { lo = 0.0; up = 0.0; diag = 1.0; rr = 0.0; ri = 0.0; }  // the gauge: P_0(0,0) = 0
    const double den = 1.0 / (diag - lo * cpm);
    cpm = up * den;
    drm = (rr - lo * drm) * den;
    dim = (ri - lo * dim) * den;
    cp[k * nh + o] = cpm;
    br[k * nh + o] = drm;
    bi[k * nh + o] = dim;
  }
  double pr = 0.0, pi = 0.0;
  for (int k = nz - 1; k >= 0; k--) {
    const double c = k <= nz - 2 ? cp[k * nh + o] : 0.0;
    pr = br[k * nh + o] - c * pr;
    pi = bi[k * nh + o] - c * pi;
    br[k * nh + o] = pr;
    bi[k * nh + o] = pi;
  }
}

}  // namespace noalloc
}  // namespace erfb

extern "C" int erf_poisson_modes_noalloc(int nx, int ny, int nz, double dx, double dy, double dt, const double *dz,
                                         const double *dzw, double *hat_re, double *hat_im, void *cuda_stream) {
  using namespace erfb::noalloc;
  if (nx <= 0 || ny <= 0 || nz <= 0 || !(dx > 0.0) || !(dy > 0.0) || !(dt > 0.0)) return ERF_EINVAL;
  if (!dz || !dzw || !hat_re || !hat_im) return ERF_EINVAL;
  // the limit is checked before anything touches CUDA; each factor first, so that the 64-bit product cannot wrap
  constexpr long long MAXV = ERF_NOALLOC_MAX_VALUES;
  if (nx > MAXV || ny > MAXV || nz > MAXV || (long long)nx * ny > MAXV || (long long)nx * ny * nz > MAXV)
    return ERF_ETOOLARGE;
  cudaError_t err = cudaSuccess;
  double *cp = noalloc_scratch(&err);
  if (!cp) {
    cudaGetLastError();
    return ERF_ECUDA;
  }
  const dim3 block(32, 8), grid((nx + 31) / 32, (ny + 7) / 8);
  k_modes_static<<<grid, block, 0, (cudaStream_t)cuda_stream>>>(nx, ny, nz, dx, dy, 1.0 / dt, dz, dzw, hat_re, hat_im, cp);
  return cudaGetLastError() == cudaSuccess ? ERF_OK : ERF_ECUDA;
}
