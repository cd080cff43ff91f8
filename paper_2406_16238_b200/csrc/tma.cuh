// tma.cuh - TMA (cp.async.bulk.tensor) + mbarrier building blocks for the warp-specialised
// DMMA kernels, and the swizzled fragment addressing that goes with them.
//
// Shared-memory tiles are rows of 16 doubles (128 bytes) written by TMA with SWIZZLE_128B:
// the 16-byte chunk c (0..7) of row r lives at chunk c ^ (r & 7) (tile base 1024-aligned).
//
// DMMA fragments out of such tiles, conflict free, with a permuted k order inside each
// group of 8 k (the same permutation on both operands, so the sum is unchanged):
//   k-step "even" of a pair uses k = 8 kp + 2 t, k-step "odd" uses k = 8 kp + 2 t + 1.
//   * k-major operand (row = m or n index, k contiguous): ONE 16-byte load per lane and k
//     pair, chunk (4 kp + t) of row 8 b + rperm(g): .x feeds the even step, .y the odd one.
//     A quarter warp (g in {2q, 2q+1}, t = 0..3) touches rows whose bit 2 differs, i.e. the
//     two complementary 64-byte halves of the bank space.
//   * n-major operand (row = k, n contiguous, 16 n per box): an 8-byte load per lane and k
//     step from row 8 kp + 2 t + parity; a half warp touches 4 rows with distinct (r >> 1) & 3.
// Fragment row g of an 8-row block maps to tile row rperm(g) = (g >> 1) + 4 (g & 1); the
// accumulator columns 2t, 2t+1 therefore map to tile columns t and t + 4 of the block.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace afq {

struct alignas(64) TensorMap { unsigned char bytes[128]; };   // CUtensorMap, opaque here

// Host: encode a tiled FP64 tensor map with SWIZZLE_128B (tmap.cu).  dims/box innermost first;
// strides_bytes[i] is the byte stride of dimension i + 1 (rank - 1 entries, multiples of 16).
// Returns 0 on success, nonzero (CUresult or -1) on failure.
int make_tensor_map_f64(TensorMap* out, const void* base, int rank, const uint64_t* dims,
                        const uint64_t* strides_bytes, const uint32_t* box);

// the same for bfloat16 elements; swizzle_bytes = 64 or 128 = the byte extent of the box's inner dimension
int make_tensor_map_bf16(TensorMap* out, const void* base, int rank, const uint64_t* dims,
                         const uint64_t* strides_bytes, const uint32_t* box, int swizzle_bytes);

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
// the same on shared-memory addresses (saves the 64-bit generic pointers in register-tight loops)
__device__ __forceinline__ void mbar_arrive_u32(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_u32(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
// Consumer release of a ring stage, LAGGED BY ONE ITERATION.  Releasing stage `it` right after its
// fragment loads lets ptxas place the mbarrier.arrive directly behind the last LDS, ahead of the
// DMMAs that consume it; that LDS can then still be in flight when the producer's TMA refills the
// stage (seen on B200 as one warp's last-loaded B fragment of one stage going stale, about once per
// 1e6 stages).  Called right after the full-barrier wait of iteration `it`, it releases the stage of
// iteration it - 1: every DMMA of that iteration sits before the wait loop, and a DMMA cannot
// issue before the LDS feeding it has returned.  Costs one stage of prefetch depth.
__device__ __forceinline__ void consumer_release_prev(uint64_t* empty, uint32_t it, int stages, int lane) {
  if (it > 0 && lane == 0) mbar_arrive(&empty[(it - 1) % stages]);
}
// named barrier among `count` threads (count a multiple of 32), id 1..15
__device__ __forceinline__ void named_bar_sync(int id, int count) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(count) : "memory");
}

__device__ __forceinline__ void tma_load_2d(void* smem, const TensorMap* tm, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];\n"
      ::"r"(smem_u32(smem)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* smem, const TensorMap* tm, uint64_t* bar, int c0, int c1,
                                            int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];\n"
      ::"r"(smem_u32(smem)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* smem, const TensorMap* tm, uint64_t* bar, int c0, int c1,
                                            int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];\n"
      ::"r"(smem_u32(smem)), "l"(tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}
__device__ __forceinline__ void prefetch_tensormap(const TensorMap* tm) {
  asm volatile("prefetch.tensormap [%0];\n" ::"l"(tm) : "memory");
}

template <int N>
__device__ __forceinline__ void reg_alloc() {
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void reg_dealloc() {
  asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(N));
}

__device__ __forceinline__ int rperm(int g) { return (g >> 1) + 4 * (g & 1); }

__device__ __forceinline__ double2 lds128(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts64(uint32_t addr, double v) {
  asm volatile("st.shared.f64 [%0], %1;\n" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ double lds64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
  return v;
}

}  // namespace afq
