// TMA / mbarrier / cp.async primitives and the tile geometry shared by the z-marching kernels
// (rhs_march_kernel in streams_march.cu, sensor_march_kernel in streams_canon.cu).  sm_100a only.
#pragma once
#include <cuda.h>
#include "streams_dev.cuh"

#ifndef STREAMS_MARCH_TY
#define STREAMS_MARCH_TY 8
#endif

#ifndef STREAMS_SENSOR_TY
#define STREAMS_SENSOR_TY 8
#endif

namespace streams {

// ------------------------------------------------------------------ async-copy / mbarrier / TMA primitives
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// copies 8 bytes when `take`, writes zeros (and reads nothing) otherwise
__device__ __forceinline__ void cp_async8_zfill(void* smem_dst, const void* gsrc, bool take) {
  const unsigned n = take ? 8u : 0u;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(n) : "memory");
}
// 8 bytes, global -> shared
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
// 16 bytes (L2 only) when `take`, zeros otherwise; both addresses 16-byte aligned
__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gsrc, bool take) {
  const unsigned n = take ? 16u : 0u;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// waits until at most N of this thread's most recent commit groups are still pending
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// this thread's arrival on `bar` (counted in the barrier's init count), performed when all its earlier cp.async have
// landed; earlier shared-memory stores of the thread are ordered before it too
__device__ __forceinline__ void cp_async_mbar_arrive(unsigned long long* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// a load the compiler may not sink to its first use
__device__ __forceinline__ unsigned ld_u8_now(const unsigned char* p) {
  unsigned v;
  asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// one box of a 4-D tensor (x, y, z, field) into shared memory, completion counted on `bar`
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, unsigned long long* bar, int c0, int c1,
                                            int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::
          "r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// the same box brought into L2 only (no shared-memory destination, no completion tracking)
__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap* map, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];" ::"l"(map), "r"(c0), "r"(c1), "r"(c2),
               "r"(c3)
               : "memory");
}

constexpr int MTX = 32;

// Tile geometry of the z-marching kernels: a block owns MTX x TY nodes of a plane; NG = ghost width of the layout
// (DevP::ng: 3, or 4 when an order of the scheme needs four layers) = halo rows / ring depth of the tile.
template <int TY, int NG>
struct MarchGeom {
  static constexpr int ROW = MTX + 8;            // row pitch: 4 halo columns each side (NG used), rows stay 32 B aligned
  static constexpr int ROWS = TY + 2 * NG;
  static constexpr int PLANE = ROW * ROWS;       // doubles per field per buffer
  static constexpr int NT = MTX * TY;
  static_assert(NG >= 1 && NG <= 4, "the halo columns of a row hold at most four ghost nodes");
};

// z chunks per tile: enough blocks to fill every SM slot in whole waves, long enough that the ring fill
// (6 planes of loads, no arithmetic) stays a small part of a chunk.
static inline int pick_chunks(int tiles, int nz, int slots) {
  int best_c = 1;
  double best = 1e300;
  for (int c = 1; c <= (nz + 3) / 4; ++c) {
    const int kz = (nz + c - 1) / c, ce = (nz + kz - 1) / kz;
    const long long waves = ((long long)tiles * ce + slots - 1) / slots;
    const double cost = (double)waves * (kz + 1.0);
    if (cost < best - 1e-9) { best = cost; best_c = ce; }
  }
  return best_c;
}

}  // namespace streams
