// erf_view.cuh -- plain-data view of a context that kernels take by value, and the
// index helpers every kernel uses.  Internal to liberf_b200.so.
//
// HBM layout: every 3-D field is dense, x fastest, [nlev][ny][nx] with nlev = nz (cell
// and horizontal-face fields) or nz+1 (w-face fields); all are allocated with nz+1
// levels.  There are no ghost cells: the lateral boundary is an index wrap (periodic) or an index
// clamp (open) at load time, so no halo-fill pass ever touches HBM.
#pragma once
#include <cstddef>

#define ERF_HD __device__ __forceinline__  // every cell function runs on the device only

namespace erfb {

enum { RHO = 0, UU = 1, VV = 2, WW = 3, TH = 4 };

struct View {
  int nx, ny, nz;
  int oh, ov, diffusion;
  int flat;
  int perx, pery;  // lateral boundary per direction: 1 periodic (index wrap), 0 open (index clamp) [R:G27]
  int ray_fields;  // Rayleigh layer: bit 1 u, 2 v, 4 w, 8 theta (0 = off)
  double ray_depth, ray_coef, ray_uref, ray_vref;
  int osh, osv;  // interpolation of the cell-centred scalars theta, phi: oh / ov, or a WENO code (13, 15, 23, 25)
  double dx, dy;
  double Rd, cp, g, p00, gam, rdocv;
  double nu, alpha, Cs, Prt, beta_s, beta_d;
  // geometry (S0), 3-D, levels as noted
  const double *zw;        // 0..nz   w-face centre height
  const double *hx, *hy;   // 0..nz-1 x-/y-face heights
  const double *hc, *zc;   // 0..nz-1 cell thickness, centre height
  const double *hw;        // 1..nz-1 centre-to-centre spacing
  const double *hu, *hv;   // 0..nz-1 U/V control-volume thickness
  const double *sxw, *syw; // 0..nz   slopes of the w-faces
  const double *sxu, *syv; // 0..nz-1 slopes of the centre surface at u-/v-points
  // base state, 3-D
  const double *rho0, *Th0, *p0, *pi0;
};

// periodic wrap; offsets are at most a few cells, so one add or subtract almost always does (the modulo only
// runs on grids narrower than the stencil)
ERF_HD int wrapi(int a, int n) {
  if (a < 0) {
    a += n;
    if (a < 0) a = (a % n + n) % n;
  } else if (a >= n) {
    a -= n;
    if (a >= n) a %= n;
  }
  return a;
}

// open boundary: the ghost value is the nearest interior value, i.e. the index is clamped
ERF_HD int clampi(int a, int n) { return a < 0 ? 0 : (a >= n ? n - 1 : a); }
ERF_HD int lati(int a, int n, int periodic) { return periodic ? wrapi(a, n) : clampi(a, n); }

// index into a dense [.][ny][nx] field with the lateral boundary condition folded in
ERF_HD size_t IX(const View &c, int i, int j, int k) {
  return ((size_t)k * c.ny + lati(j, c.ny, c.pery)) * c.nx + lati(i, c.nx, c.perx);
}

// The same view for threads whose stencils cannot leave the domain (CTAs at least a stencil width away from the lateral
// boundary): no wrap, no clamp.  The per-cell bodies of general_cells.cuh are templates over the view type, so an
// interior CTA runs index arithmetic that the compiler folds into constant offsets.
struct ViewNW : View {
  ERF_HD explicit ViewNW(const View &v) : View(v) {}
};
ERF_HD size_t IX(const ViewNW &c, int i, int j, int k) { return ((size_t)k * c.ny + j) * c.nx + i; }

}  // namespace erfb
