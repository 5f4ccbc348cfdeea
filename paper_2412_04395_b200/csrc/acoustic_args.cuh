// acoustic_args.cuh -- the argument block shared by the flat-grid acoustic-substep kernels (k_acoustic_tile.cu:
// column tiles with on-chip scratch; k_fused_acoustic.cu: thread per column) and their common driver.
#pragma once
#include "fused.cuh"

namespace erfb {

// stage-combine bits of a substep launch
enum { MODE_FIRST = 1, MODE_LAST = 2, MODE_ZERO = 4 };

struct AcArgs {
  int nx, ny, nz;
  int write_cp;  // thread-per-column kernel: store c' (stage constant, so only the first substep of a stage does)
  double dtau, rdx, rdy, b1, b2, beta_d, g, gR;
  const double *Pu, *Pv, *Pw, *Pr, *Pt, *Ptp;  // S'' in: U'', V'', W'', rho'', Theta'' and Theta''_prev
  const double *Sn[5], *St[5];                 // FIRST: S'' = Sn - St;  LAST: St is added to the result
  double *oU, *oV, *oW, *oR, *oT, *oTp;        // out: S'' (or the stage result); oTp: initial Theta'' (FIRST)
  double *sumU, *sumV, *sumOm;                 // null, or the sums over the substeps of the momenta that advance rho'' (L138)
  double *kW, *kR, *kT, *cp_scr;               // column scratch between the sweeps (thread-per-column kernel)
  const double *RU, *RV, *RW, *Rrho, *RTh;
  const double *theta, *pi, *iT;
  const double *rdz, *rhw, *tabB;
};

void launch_acoustic_flat_one(const AcArgs &p, int mode, cudaStream_t st);  // k_fused_acoustic.cu
bool acoustic_tile_selected(const erf_ctx *c);                              // k_acoustic_tile.cu
void launch_acoustic_tile_one(const AcArgs &p, int mode, cudaStream_t st);

}  // namespace erfb
