// k_anelastic.cu -- the anelastic mode (Sec. 2.2 Eq. 8; Sec. 3.2 Eq. 14-16) on flat,
// laterally periodic grids: RK2 without substepping, a projection after each stage.
//
//   S*      = S^n + dt f(S^n)                      (Eq. 14), projected;
//   S^{n+1} = S^n + dt/2 (f(S^n) + f(S*))           (Eq. 15), projected ("an analogous procedure", L162);
//   projection (Eq. 16):  dt div(grad psi) = div(rho0 u**),  rho0 u* = rho0 u** - dt grad psi,  p' += psi.
//
// f is the slow right-hand side of the compressible core (general kernels) with the pressure-gradient / buoyancy pair of
// Sec. 2.2 (gen::anel_pgbuoy_cell); rho is held at the base state (L94).  The Poisson equation is solved with the discrete
// Fourier transform in the two periodic directions ("Fast Fourier Transforms", L164) and one real tridiagonal system in z
// per horizontal mode [R:G29]:
//     [lx(m) + ly(n)] P_k + [ (P_{k+1} - P_k)/hw_{k+1} - (P_k - P_{k-1})/hw_k ] / dz_k = Dhat_k / dt,
//     lx(m) = -(4/dx^2) sin^2(pi m / nx), ly(n) = -(4/dy^2) sin^2(pi n / ny);  mode (0, 0): psi_hat(k = 0) = 0.
//
// Kernels.  Power-of-two lengths: radix-2 transforms in shared memory (x: one row per CTA; y: eight neighbouring columns
// of a level per CTA).  Other lengths: direct sums over the twiddle table, one output per thread (O(n) work per output).
// The column solve is one thread per mode (m, n), Thomas in place, real and imaginary part together.
#include "erf_ctx.cuh"

namespace erfb {
namespace anel {

constexpr double PI = 3.14159265358979323846;

// D = dU/dx + dV/dy + dW/dz at cell centres (flat grid: Omega = W, hx = hy = hc)
__global__ void k_div(View v, const double *U, const double *V, const double *W, const double *lev, double *D) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
  if (i >= v.nx || j >= v.ny) return;
  const size_t a = IX(v, i, j, k);
  D[a] = (U[IX(v, i + 1, j, k)] - U[a]) / v.dx + (V[IX(v, i, j + 1, k)] - V[a]) / v.dy +
         (W[IX(v, i, j, k + 1)] - W[a]) / lev[k];
}

// twiddles: tw[t] = cos(2 pi t / n), tw[n + t] = sin(2 pi t / n)
__global__ void k_twiddle(double *tw, int n) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  tw[t] = cos(2.0 * PI * t / n);
  tw[n + t] = sin(2.0 * PI * t / n);
}

// transform along x of one (j, k) row per CTA.  SIGN = -1 forward, +1 inverse.  in: (ar, ai), ai may be null (real
// input); out: (br, bi), bi may be null (real output wanted), scaled by `scale`.
template <int SIGN>
__global__ void k_dft_x(int nx, const double *__restrict__ ar, const double *__restrict__ ai, double *br, double *bi,
                        const double *__restrict__ tw, double scale) {
  extern __shared__ double sm[];
  double *xr = sm, *xi = sm + nx, *tc = sm + 2 * nx, *ts = sm + 3 * nx;
  const size_t row = (size_t)blockIdx.x * nx;
  for (int t = threadIdx.x; t < nx; t += blockDim.x) {
    xr[t] = ar[row + t];
    xi[t] = ai ? ai[row + t] : 0.0;
    tc[t] = tw[t];
    ts[t] = SIGN * tw[nx + t];
  }
  __syncthreads();
  for (int m = threadIdx.x; m < nx; m += blockDim.x) {
    double sr = 0.0, si = 0.0;
    int idx = 0;
    for (int i = 0; i < nx; i++) {
      const double c = tc[idx], s = ts[idx];
      sr += xr[i] * c - xi[i] * s;
      si += xr[i] * s + xi[i] * c;
      idx += m;
      if (idx >= nx) idx -= nx;
    }
    br[row + m] = sr * scale;
    if (bi) bi[row + m] = si * scale;
  }
}

// transform along y: one output (m, n, k) per thread, m fastest (coalesced reads of A[k][j][m] over j)
template <int SIGN>
__global__ void k_dft_y(int nx, int ny, const double *__restrict__ ar, const double *__restrict__ ai, double *br,
                        double *bi, const double *__restrict__ tw) {
  extern __shared__ double sm[];
  double *tc = sm, *ts = sm + ny;
  for (int t = threadIdx.y * 32 + threadIdx.x; t < ny; t += 256) {
    tc[t] = tw[t];
    ts[t] = SIGN * tw[ny + t];
  }
  __syncthreads();
  const int m = blockIdx.x * 32 + threadIdx.x, n = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
  if (m >= nx || n >= ny) return;
  const size_t kb = (size_t)k * nx * ny;
  double sr = 0.0, si = 0.0;
  int idx = 0;
  for (int j = 0; j < ny; j++) {
    const double c = tc[idx], s = ts[idx];
    const double xr = ar[kb + (size_t)j * nx + m], xi = ai[kb + (size_t)j * nx + m];
    sr += xr * c - xi * s;
    si += xr * s + xi * c;
    idx += n;
    if (idx >= ny) idx -= ny;
  }
  br[kb + (size_t)n * nx + m] = sr;
  bi[kb + (size_t)n * nx + m] = si;
}

// ---- power-of-two lengths: radix-2 transforms in shared memory (decimation in time: bit-reversed load, log2 n butterfly
// stages with the twiddles of the table).  NB sequences of length n per CTA, sequence b at re/im[b * n ...].
template <int SIGN>
__device__ __forceinline__ void fft_stages(double *re, double *im, int n, int logn, int nb, const double *tc,
                                           const double *ts, int tid, int nthr) {
  const int half_n = n >> 1;
  for (int s = 1; s <= logn; s++) {
    const int len = 1 << s, half = len >> 1, tstep = n >> s;
    __syncthreads();
    for (int t = tid; t < nb * half_n; t += nthr) {
      const int b = t / half_n, q = t - b * half_n;
      const int grp = q / half, pos = q - grp * half;
      const int i0 = b * n + grp * len + pos, i1 = i0 + half;
      const double wr = tc[pos * tstep], wi = SIGN * ts[pos * tstep];
      const double xr = re[i1] * wr - im[i1] * wi, xi = re[i1] * wi + im[i1] * wr;
      const double ar = re[i0], ai = im[i0];
      re[i0] = ar + xr; im[i0] = ai + xi;
      re[i1] = ar - xr; im[i1] = ai - xi;
    }
  }
  __syncthreads();
}

// x: one (j, k) row per CTA; ai may be null (real input), bi may be null (real output)
template <int SIGN>
__global__ void k_fft_x(int nx, int logn, const double *__restrict__ ar, const double *__restrict__ ai, double *br,
                        double *bi, const double *__restrict__ tw, double scale) {
  extern __shared__ double sm[];
  double *re = sm, *im = sm + nx, *tc = sm + 2 * nx, *ts = sm + 3 * nx;
  const size_t row = (size_t)blockIdx.x * nx;
  for (int t = threadIdx.x; t < nx; t += blockDim.x) {
    const int r = (int)(__brev((unsigned)t) >> (32 - logn));
    re[r] = ar[row + t];
    im[r] = ai ? ai[row + t] : 0.0;
    tc[t] = tw[t];
    ts[t] = tw[nx + t];
  }
  fft_stages<SIGN>(re, im, nx, logn, 1, tc, ts, threadIdx.x, blockDim.x);
  for (int t = threadIdx.x; t < nx; t += blockDim.x) {
    br[row + t] = re[t] * scale;
    if (bi) bi[row + t] = im[t] * scale;
  }
}

// y: NB = 8 neighbouring columns m of one level per CTA
template <int SIGN>
__global__ void k_fft_y(int nx, int ny, int logn, const double *__restrict__ ar, const double *__restrict__ ai,
                        double *br, double *bi, const double *__restrict__ tw) {
  constexpr int NB = 8;
  extern __shared__ double sm[];
  double *re = sm, *im = sm + NB * ny, *tc = sm + 2 * NB * ny, *ts = tc + ny;
  const int m0 = blockIdx.x * NB, k = blockIdx.y, tid = threadIdx.x, nthr = blockDim.x;
  const size_t kb = (size_t)k * nx * ny;
  for (int t = tid; t < ny; t += nthr) { tc[t] = tw[t]; ts[t] = tw[ny + t]; }
  for (int t = tid; t < NB * ny; t += nthr) {
    const int b = t % NB, j = t / NB;  // b fastest: 64-byte segments of a row
    if (m0 + b < nx) {
      const int r = (int)(__brev((unsigned)j) >> (32 - logn));
      re[b * ny + r] = ar[kb + (size_t)j * nx + m0 + b];
      im[b * ny + r] = ai[kb + (size_t)j * nx + m0 + b];
    } else {
      re[b * ny + j] = 0.0; im[b * ny + j] = 0.0;
    }
  }
  fft_stages<SIGN>(re, im, ny, logn, NB, tc, ts, tid, nthr);
  for (int t = tid; t < NB * ny; t += nthr) {
    const int b = t % NB, n = t / NB;
    if (m0 + b < nx) {
      br[kb + (size_t)n * nx + m0 + b] = re[b * ny + n];
      bi[kb + (size_t)n * nx + m0 + b] = im[b * ny + n];
    }
  }
}

// one tridiagonal system per mode: lev = [dz(0..nz-1) | hw(0..nz), hw(0) unused]; (br, bi) in/out; cp = scratch c'
__global__ void k_modes(int nx, int ny, int nz, double dx, double dy, double rdt, const double *__restrict__ lev,
                        double *br, double *bi, double *cp) {
  const int m = blockIdx.x * 32 + threadIdx.x, n = blockIdx.y * 8 + threadIdx.y;
  if (m >= nx || n >= ny) return;
  const size_t nh = (size_t)nx * ny, o = (size_t)n * nx + m;
  const double sx = sin(PI * m / nx), sy = sin(PI * n / ny);
  const double lam = -4.0 * sx * sx / (dx * dx) - 4.0 * sy * sy / (dy * dy);
  const double *dz = lev, *hw = lev + nz;
  double cpm = 0.0, drm = 0.0, dim = 0.0;
  for (int k = 0; k < nz; k++) {
    double lo = k >= 1 ? 1.0 / (hw[k] * dz[k]) : 0.0;
    double up = k <= nz - 2 ? 1.0 / (hw[k + 1] * dz[k]) : 0.0;
    double diag = lam - lo - up;
    double rr = br[k * nh + o] * rdt, ri = bi[k * nh + o] * rdt;
    if (m == 0 && n == 0 && k == 0) { lo = 0.0; up = 0.0; diag = 1.0; rr = 0.0; ri = 0.0; }
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

// rho0 u* = rho0 u** - dt grad psi, p' += psi (L158-L160); nothing on the rigid lids
__global__ void k_correct(View v, const double *psi, const double *lev, double dt, double *U, double *V, double *W,
                          double *pp) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
  if (i >= v.nx || j >= v.ny) return;
  const size_t a = IX(v, i, j, k);
  const double ps = psi[a];
  U[a] -= dt * (ps - psi[IX(v, i - 1, j, k)]) / v.dx;
  V[a] -= dt * (ps - psi[IX(v, i, j - 1, k)]) / v.dy;
  if (k >= 1) W[a] -= dt * (ps - psi[IX(v, i, j, k - 1)]) / lev[v.nz + k];
  pp[a] += ps;
}

// level tables from column (0, 0) of the 3-D metric arrays
__global__ void k_levels(View v, double *lev) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > v.nz) return;
  const size_t a = (size_t)k * v.nx * v.ny;
  if (k < v.nz) lev[k] = v.hc[a];
  lev[v.nz + k] = (k >= 1 && k < v.nz) ? v.hw[a] : 0.0;
}

// out = S + a1 R1, or S + a1 (R1 + R2) with `two`, for U, V, W, Theta; rho = rho0; flat lids W = 0
__global__ void k_rk2(View v, F5 S, F5 R1, F5 R2, double a1, bool two, F5 out) {
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
  if (i >= v.nx || j >= v.ny) return;
  const size_t a = IX(v, i, j, k);
  if (k < v.nz) {
    out.f[RHO][a] = v.rho0[a];
    for (int f = UU; f <= TH; f++) {
      if (f == WW) continue;
      out.f[f][a] = S.f[f][a] + a1 * (two ? R1.f[f][a] + R2.f[f][a] : R1.f[f][a]);
    }
  }
  out.f[WW][a] = (k == 0 || k == v.nz) ? 0.0 : S.f[WW][a] + a1 * (two ? R1.f[WW][a] + R2.f[WW][a] : R1.f[WW][a]);
}

}  // namespace anel

static int ensure_anelastic(erf_ctx *c, cudaStream_t st) {
  if (!c->v.flat || !c->v.perx || !c->v.pery) return ERF_EUNSUPPORTED;
  if (ensure_general(c, st) != ERF_OK) return c->status;
  if (c->an_pp) return c->status;
  const size_t nc = (size_t)c->nx * c->ny * c->nz;
  c->an_pp = c->alloc(c->NW);
  for (auto &w : c->an_w) w = c->alloc(nc);
  c->an_tw = c->alloc(2 * (size_t)(c->nx + c->ny));
  c->an_lev = c->alloc(2 * (size_t)c->nz + 2);
  if (c->status != ERF_OK) return c->status;
  anel::k_twiddle<<<(c->nx + 127) / 128, 128, 0, st>>>(c->an_tw, c->nx);
  anel::k_twiddle<<<(c->ny + 127) / 128, 128, 0, st>>>(c->an_tw + 2 * c->nx, c->ny);
  anel::k_levels<<<(c->nz + 128) / 128, 128, 0, st>>>(c->v, c->an_lev);
  c->launches += 3;
  return c->status;
}

// Eq. 16 applied to the momenta of S
int anelastic_project(erf_ctx *c, const F5 &S, double dt, cudaStream_t st) {
  int rc = ensure_anelastic(c, st);
  if (rc != ERF_OK) return rc;
  const int nx = c->nx, ny = c->ny, nz = c->nz;
  double *Ar = c->an_w[0], *Ai = c->an_w[1], *Br = c->an_w[2], *Bi = c->an_w[3];
  const double *twx = c->an_tw, *twy = c->an_tw + 2 * nx;
  dim3 block(32, 8), grid((nx + 31) / 32, (ny + 7) / 8, nz), gmodes((nx + 31) / 32, (ny + 7) / 8);
  const int tx = nx < 256 ? ((nx + 31) / 32) * 32 : 256;
  const size_t smx = 4 * (size_t)nx * sizeof(double), smy = 2 * (size_t)ny * sizeof(double);
  if (smx > 200 * 1024 || smy > 200 * 1024) return ERF_EUNSUPPORTED;
  auto log2i = [](int n) { int l = 0; while ((1 << l) < n) l++; return ((1 << l) == n && n >= 2) ? l : -1; };
  const int lx = log2i(nx), ly = log2i(ny);  // -1: not a power of two, the direct sums run
  const size_t smfy = (size_t)(2 * 8 + 2) * ny * sizeof(double);
  const int tfx = nx / 2 < 256 ? (nx / 2 < 32 ? 32 : nx / 2) : 256;
  static OncePerDevice attr;
  attr.run([] {
    cudaFuncSetAttribute(anel::k_fft_x<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_fft_x<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_fft_y<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_fft_y<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_dft_x<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_dft_x<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_dft_y<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(anel::k_dft_y<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  });
  anel::k_div<<<grid, block, 0, st>>>(c->v, S.f[UU], S.f[VV], S.f[WW], c->an_lev, Br);
  const bool fy = ly > 0 && smfy <= 200 * 1024;
  dim3 gfy((nx + 7) / 8, nz);
  if (lx > 0) anel::k_fft_x<-1><<<ny * nz, tfx, smx, st>>>(nx, lx, Br, nullptr, Ar, Ai, twx, 1.0);
  else anel::k_dft_x<-1><<<ny * nz, tx, smx, st>>>(nx, Br, nullptr, Ar, Ai, twx, 1.0);
  if (fy) anel::k_fft_y<-1><<<gfy, 256, smfy, st>>>(nx, ny, ly, Ar, Ai, Br, Bi, twy);
  else anel::k_dft_y<-1><<<grid, block, smy, st>>>(nx, ny, Ar, Ai, Br, Bi, twy);
  anel::k_modes<<<gmodes, block, 0, st>>>(nx, ny, nz, c->v.dx, c->v.dy, 1.0 / dt, c->an_lev, Br, Bi, Ar);
  if (fy) anel::k_fft_y<1><<<gfy, 256, smfy, st>>>(nx, ny, ly, Br, Bi, Ar, Ai, twy);
  else anel::k_dft_y<1><<<grid, block, smy, st>>>(nx, ny, Br, Bi, Ar, Ai, twy);
  if (lx > 0) anel::k_fft_x<1><<<ny * nz, tfx, smx, st>>>(nx, lx, Ar, Ai, Br, nullptr, twx, 1.0 / ((double)nx * ny));
  else anel::k_dft_x<1><<<ny * nz, tx, smx, st>>>(nx, Ar, Ai, Br, nullptr, twx, 1.0 / ((double)nx * ny));
  anel::k_correct<<<grid, block, 0, st>>>(c->v, Br, c->an_lev, dt, S.f[UU], S.f[VV], S.f[WW], c->an_pp);
  c->launches += 7;
  return c->status;
}

// one RK2 step (Eq. 14-15) with a projection after each stage; c->P holds f(S^n) between the stages
int anelastic_step(erf_ctx *c, double dt, cudaStream_t st) {
  int rc = ensure_anelastic(c, st);
  if (rc != ERF_OK) return rc;
  Timed t(c, T_OTHER, st);
  dim3 block(32, 8), grid((c->nx + 31) / 32, (c->ny + 7) / 8, c->nz + 1);
  const size_t nc = (size_t)c->nx * c->ny * c->nz * sizeof(double);
  cudaMemcpyAsync(c->S.f[RHO], c->rho0, nc, cudaMemcpyDeviceToDevice, st);  // rho = rho0 (L94)
  general_slow_rhs(c, c->S, st, c->an_pp);
  { F5 tmp = c->R; c->R = c->P; c->P = tmp; }  // f(S^n) kept in c->P
  anel::k_rk2<<<grid, block, 0, st>>>(c->v, c->S, c->P, c->P, dt, false, c->St);
  c->launches++;
  if ((rc = anelastic_project(c, c->St, dt, st)) != ERF_OK) return rc;
  general_slow_rhs(c, c->St, st, c->an_pp);
  anel::k_rk2<<<grid, block, 0, st>>>(c->v, c->S, c->P, c->R, 0.5 * dt, true, c->St);
  c->launches++;
  if ((rc = anelastic_project(c, c->St, dt, st)) != ERF_OK) return rc;
  for (int f = 0; f < 5; f++) { double *tmp = c->S.f[f]; c->S.f[f] = c->St.f[f]; c->St.f[f] = tmp; }
  return c->status;
}

}  // namespace erfb
