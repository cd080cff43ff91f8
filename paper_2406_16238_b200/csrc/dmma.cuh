// dmma.cuh - FP64 tensor-core building blocks for sm_100a.
//
// tcgen05.mma has no f64 kind (ptxas rejects .kind::f64), so the FP64 tensor path on B200
// is the warp-level mma.sync, which ptxas lowers to DMMA.8x8x4 for every PTX shape.  The
// operands reach it through registers: shared-memory tiles are laid out so that the 8x4 /
// 4x8 fragment reads are bank-conflict free, and the tiles are fed by cp.async (LDGSTS)
// multi-stage pipelines.
//
// Fragment layout of mma.sync.m8n8k4.f64 (lane l, g = l / 4, t = l % 4):
//   A (8x4, row)  : a  = A[g][t]
//   B (4x8, col)  : b  = B[t][g]
//   C/D (8x8)     : c0 = C[g][2t], c1 = C[g][2t+1]
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace afq {

constexpr int kThreads = 256;  // 8 warps per CTA everywhere in the GEMM-like kernels
constexpr int BK = 16;         // k extent of one pipeline stage (4 DMMA k-steps)
constexpr int LDK = BK + 4;    // row stride (doubles) of k-major tiles: 20 mod 16 = 4 -> conflict free

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile(
      "mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c0), "+d"(c1)
      : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async8(void* smem, const void* gmem, int src_bytes) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// Load a [ROWS][BK] tile whose rows are k-contiguous in global memory into smem [ROWS][LDK].
// rowptr(r) returns the global pointer of element k = 0 of tile row r, or nullptr for a row
// that must read as zeros.  kvalid = number of valid k in this stage (<= BK), the rest is
// zero-filled.  vec16: rows and k0 are 16-byte aligned (two doubles per cp.async).
template <int ROWS, class RowPtr>
__device__ __forceinline__ void load_kmajor_tile(double* s, RowPtr rowptr, int k0, int kvalid,
                                                 bool vec16, const double* safe) {
  const int tid = threadIdx.x;
  if (vec16) {
    constexpr int CH = BK / 2;  // 16-byte chunks per row
#pragma unroll
    for (int c = tid; c < ROWS * CH; c += kThreads) {
      int r = c / CH, ch = c % CH;
      const double* gp = rowptr(r);
      int nb = (kvalid - 2 * ch) * 8;
      nb = nb < 0 ? 0 : (nb > 16 ? 16 : nb);
      if (gp == nullptr) nb = 0;
      const double* src = nb ? gp + k0 + 2 * ch : safe;
      cp_async16(s + r * LDK + 2 * ch, src, nb);
    }
  } else {
#pragma unroll
    for (int c = tid; c < ROWS * BK; c += kThreads) {
      int r = c / BK, k = c % BK;
      const double* gp = rowptr(r);
      int nb = (k < kvalid && gp != nullptr) ? 8 : 0;
      const double* src = nb ? gp + k0 + k : safe;
      cp_async8(s + r * LDK + k, src, nb);
    }
  }
}

// Load a [BK][COLS] tile whose rows (k) hold n-contiguous data into smem [BK][COLS + 4].
// base points at element (k = 0 of the whole matrix, n = n0 of this tile); row stride ld.
// nvalid = valid columns in this tile, kvalid = valid k rows in this stage.
template <int COLS>
__device__ __forceinline__ void load_nmajor_tile(double* s, const double* base, long ld, int k0,
                                                 int kvalid, int nvalid, bool vec16,
                                                 const double* safe) {
  constexpr int LDS_ = COLS + 4;
  const int tid = threadIdx.x;
  if (vec16) {
    constexpr int CH = COLS / 2;
#pragma unroll
    for (int c = tid; c < BK * CH; c += kThreads) {
      int k = c / CH, ch = c % CH;
      int nb = (nvalid - 2 * ch) * 8;
      nb = nb < 0 ? 0 : (nb > 16 ? 16 : nb);
      if (k >= kvalid) nb = 0;
      const double* src = nb ? base + (long)(k0 + k) * ld + 2 * ch : safe;
      cp_async16(s + k * LDS_ + 2 * ch, src, nb);
    }
  } else {
#pragma unroll
    for (int c = tid; c < BK * COLS; c += kThreads) {
      int k = c / COLS, n = c % COLS;
      int nb = (k < kvalid && n < nvalid) ? 8 : 0;
      const double* src = nb ? base + (long)(k0 + k) * ld + n : safe;
      cp_async8(s + k * LDS_ + n, src, nb);
    }
  }
}

// One pipeline stage (BK = 16 -> 4 k-steps) of a warp tile of MI x NI 8x8 blocks.
//   A tile: k-major  As[(m)*LDK + k]            (A_KM = false)
//           m-major  As[k*LDA_M + m]            (A_KM = true,  LDA_M = BM + 4)
//   B tile: k-major  Bs[(n)*LDK + k]            (B_NK = true)
//           n-major  Bs[k*LDB_N + n]            (B_NK = false, LDB_N = BN + 4)
template <int MI, int NI, bool A_KM, bool B_NK, int LDA_M, int LDB_N>
__device__ __forceinline__ void mma_stage(const double* __restrict__ As,
                                          const double* __restrict__ Bs, int wm0, int wn0, int g,
                                          int t, double (&acc)[MI][NI][2]) {
#pragma unroll
  for (int s = 0; s < BK / 4; ++s) {
    double af[MI], bf[NI];
#pragma unroll
    for (int i = 0; i < MI; ++i)
      af[i] = A_KM ? As[(4 * s + t) * LDA_M + wm0 + 8 * i + g] : As[(wm0 + 8 * i + g) * LDK + 4 * s + t];
#pragma unroll
    for (int j = 0; j < NI; ++j)
      bf[j] = B_NK ? Bs[(wn0 + 8 * j + g) * LDK + 4 * s + t] : Bs[(4 * s + t) * LDB_N + wn0 + 8 * j + g];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
  }
}

}  // namespace afq
