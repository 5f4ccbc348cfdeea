// bulk.cuh -- shared-memory plane tiles filled by the bulk-copy engine with mbarrier completion (SASS SYNCS):
// TMA tensor copies (cp.async.bulk.tensor.3d, SASS UTMALDG) -- one instruction per field and level -- for the CTAs
// whose halo tile lies inside the domain, row-wise bulk copies (cp.async.bulk, SASS UBLKCP) with the periodic wrap
// in the source address for the CTAs on the periodic seam (the tensor unit fills out-of-range boxes with zeros, it
// cannot wrap).
//
// A tile is H rows of W doubles of one horizontal plane of a dense [.][ny][nx] field, starting at column
// xs (even) and row ys, both taken modulo the domain: the periodic lateral boundary is a wrap of
// the copy's SOURCE address, so HBM holds no ghost cells and nothing ever fills a halo.  One row is one bulk copy
// of 8 W bytes (two or more where the row crosses the periodic seam); a handful of threads issue a whole
// multi-field stage, every thread then waits on the stage's mbarrier.  Requirements of cp.async.bulk: 16-byte
// aligned source, destination and size -- hence nx even, xs even, W even (checked by the launchers).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

namespace erfb {

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
// make the initialised barriers visible to the async proxy (the bulk-copy engine)
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }

// one arrival that also announces `bytes` of bulk-copy traffic for the current phase
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

// plain arrival (no transaction bytes): one of the `count` arrivals that complete the current phase
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// global -> shared bulk copy of `bytes` (multiple of 16), completion counted on `bar`
__device__ __forceinline__ void bulk_g2s(double *dst, const double *src, unsigned bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// whole-tile TMA copy: box (bw x bh x 1) of the 3-D tensor described by `map` with its corner at (x, y, z)
__device__ __forceinline__ void tma_tile_g2s(double *dst, const CUtensorMap *map, int x, int y, int z, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
      : "memory");
}

// host: tensor map of a dense [nlev][ny][nx] fp64 field with a (bw x bh x 1) box; false if the driver refuses
bool make_tile_map(CUtensorMap *out, const double *base, int nx, int ny, int nlev, int bw, int bh);

__device__ __forceinline__ int pmodi(int a, int n) {
  a %= n;
  return a < 0 ? a + n : a;
}

// one tile row: W doubles of row gy (already wrapped) of `plane`, starting at column gxs (wrapped, even),
// continuing across the periodic seam as often as needed (grids narrower than the tile)
__device__ __forceinline__ void bulk_row(double *dst, const double *__restrict__ plane, int gy, int gxs, int W, int nx,
                                         uint64_t *bar) {
  const double *row = plane + (size_t)gy * nx;
  int pos = gxs, rem = W;
  while (rem > 0) {
    const int len = min(rem, nx - pos);
    bulk_g2s(dst, row + pos, (unsigned)len * 8u, bar);
    dst += len;
    rem -= len;
    pos = 0;
  }
}

}  // namespace erfb
