// tiles.cuh -- shared-memory plane tiles with periodic halos, filled by asynchronous copies.
//
// A CTA of TX x TY threads owns a TX x TY patch of (i,j) columns and marches upward in k.
// For each level it needs a horizontal plane of several fields with a halo (3 cells for the
// 5th/6th-order stencils of PAPER.md Eq. 19/21, 1 cell for everything else).  The plane of
// level k+1 is copied global -> shared with cp.async (LDGSTS, 16 B per copy where the row is
// 16-byte aligned, 8 B otherwise) while level k is being computed; the periodic lateral
// boundary is an index wrap in the copy's source address, so the dense
// unpadded HBM layout needs no ghost cells and no halo-fill pass.
#pragma once
#include <cuda_runtime.h>

namespace erfb {

constexpr int TX = 32, TY = 8, NTHR = TX * TY;

__device__ __forceinline__ int pmod(int a, int n) {
  a %= n;
  return a < 0 ? a + n : a;
}

__device__ __forceinline__ void cp_async16(double *smem, const double *g) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async8(double *smem, const double *g) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

// Tile geometry: x halo HXP (even, so that every 2-double chunk starts on an even column), y halo HY.
template <int HXP, int HY>
struct TileG {
  static constexpr int W = TX + 2 * HXP, H = TY + 2 * HY, CW = W / 2, NCH = CW * H, SZ = W * H;
  static constexpr int PER = (NCH + NTHR - 1) / NTHR;  // chunks per thread
  static_assert(HXP % 2 == 0, "x halo must be even");
  // index of the thread's own column in the tile
  __device__ static __forceinline__ int centre(int tx, int ty) { return (ty + HY) * W + tx + HXP; }
};

// One thread's share of a tile copy (the same for every field with this geometry and every level).
template <int HXP, int HY>
struct ChunkSet {
  using G = TileG<HXP, HY>;
  int g0[G::PER];  // offset of the chunk's first double within a plane, or -1 if the thread has no such chunk
  int g1[G::PER];  // offset of the second double, or -1 when both are moved by one 16-byte copy
  int s[G::PER];   // offset within the tile
  __device__ __forceinline__ void init(int tid, int x0, int y0, int nx, int ny) {
#pragma unroll
    for (int n = 0; n < G::PER; n++) {
      const int c = tid + n * NTHR;
      if (c < G::NCH) {
        const int ry = c / G::CW, cx = c - ry * G::CW;
        const int gy = pmod(y0 - HY + ry, ny);
        const int gxa = pmod(x0 - HXP + 2 * cx, nx), gxb = pmod(x0 - HXP + 2 * cx + 1, nx);
        g0[n] = gy * nx + gxa;
        const bool vec = !(nx & 1) && !(gxa & 1) && gxb == gxa + 1;
        g1[n] = vec ? -1 : gy * nx + gxb;
        s[n] = ry * G::W + 2 * cx;
      } else {
        g0[n] = -1;
        g1[n] = -1;
        s[n] = 0;
      }
    }
  }
  // copy this thread's chunks of one field plane (gplane = field + k * plane) into a tile
  __device__ __forceinline__ void issue(double *tile, const double *__restrict__ gplane) const {
#pragma unroll
    for (int n = 0; n < G::PER; n++) {
      if (g0[n] >= 0) {
        if (g1[n] < 0) {
          cp_async16(tile + s[n], gplane + g0[n]);
        } else {
          cp_async8(tile + s[n], gplane + g0[n]);
          cp_async8(tile + s[n] + 1, gplane + g1[n]);
        }
      }
    }
  }
};

}  // namespace erfb
