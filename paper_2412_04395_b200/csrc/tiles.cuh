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
__device__ __forceinline__ void cp_async_wait_but_one() { asm volatile("cp.async.wait_group 1;\n" ::: "memory"); }

// Tile geometry: x halo HXP (even, so that every 2-double chunk starts on an even column), y halo HY.
template <int HXP, int HY>
struct TileG {
  static constexpr int W = TX + 2 * HXP, H = TY + 2 * HY, CW = W / 2, NCH = CW * H, SZ = W * H;
  static constexpr int PER = (NCH + NTHR - 1) / NTHR;  // chunks per thread
  static_assert(HXP % 2 == 0, "x halo must be even");
  // index of the thread's own column in the tile
  __device__ static __forceinline__ int centre(int tx, int ty) { return (ty + HY) * W + tx + HXP; }
};

// One thread's share of a tile copy (the same for every field with this geometry and every level).  The
// source/destination offsets live in shared memory ([3*PER][NTHR] ints at `tab`, each thread reads only its
// own column), not in registers: the column kernels need every register for their stencil windows.
template <int HXP, int HY, bool REGS = false>
struct ChunkSet {
  using G = TileG<HXP, HY>;
  static constexpr int TAB = 3 * G::PER * NTHR;  // ints of shared memory
  const int *t;  // tab + tid
  // REGS: when every chunk is one aligned 16-byte copy (nx even), its two offsets are kept in registers instead
  // (kernels with registers to spare: saves three shared-memory loads and a branch per copy)
  int rg0[REGS ? G::PER : 1], rso[REGS ? G::PER : 1];
  bool fast;
  // g0 = offset of the chunk's first double within a plane (-1: the thread has no such chunk); g1 = offset of
  // the second double (-1: both are moved by one 16-byte copy); s = offset within the tile
  __device__ __forceinline__ void init(int *tab, int tid, int x0, int y0, int nx, int ny) {
    fast = REGS && !(nx & 1);
#pragma unroll
    for (int n = 0; n < G::PER; n++) {
      // a thread without an n-th chunk repeats the copy of chunk n of thread 0 (harmless, keeps issue() branch-free)
      const int c = tid + n * NTHR < G::NCH ? tid + n * NTHR : n * NTHR;
      const bool have = tid + n * NTHR < G::NCH;
      const int ry = c / G::CW, cx = c - ry * G::CW;
      const int gy = pmod(y0 - HY + ry, ny);
      const int gxa = pmod(x0 - HXP + 2 * cx, nx), gxb = pmod(x0 - HXP + 2 * cx + 1, nx);
      const int g0 = gy * nx + gxa;
      const bool vec = !(nx & 1) && !(gxa & 1) && gxb == gxa + 1;
      const int g1 = vec ? -1 : gy * nx + gxb;
      const int so = ry * G::W + 2 * cx;
      if (REGS) { rg0[n] = g0; rso[n] = so; }
      tab[(3 * n) * NTHR + tid] = have ? g0 : -1;
      tab[(3 * n + 1) * NTHR + tid] = g1;
      tab[(3 * n + 2) * NTHR + tid] = so;
    }
    t = tab + tid;
  }
  // copy this thread's chunks of one field plane (gplane = field + k * plane) into a tile
  __device__ __forceinline__ void issue(double *tile, const double *__restrict__ gplane) const {
    if (REGS && fast) {
#pragma unroll
      for (int n = 0; n < G::PER; n++) cp_async16(tile + rso[n], gplane + rg0[n]);
      return;
    }
#pragma unroll
    for (int n = 0; n < G::PER; n++) {
      const int g0 = t[(3 * n) * NTHR], g1 = t[(3 * n + 1) * NTHR], so = t[(3 * n + 2) * NTHR];
      if (g0 >= 0) {
        if (g1 < 0) {
          cp_async16(tile + so, gplane + g0);
        } else {
          cp_async8(tile + so, gplane + g0);
          cp_async8(tile + so + 1, gplane + g1);
        }
      }
    }
  }
};

}  // namespace erfb
