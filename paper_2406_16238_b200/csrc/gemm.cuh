// gemm.cuh - batched real FP64 GEMM on DMMA with a cp.async multi-stage pipeline.
//
//   C[b][m][n] = alpha * sum_k A[b](m,k) * B[b](k,n)
//
// Used for every dense contraction of the walker step except the exchange energy:
//   a3 force bias, a5 V_HS build, a6/a8 one-body propagator, a7 Taylor propagation (CPLX),
//   and the setup contractions (half rotation, sum_g L_g^2, expm).
//
// Complex operands never change the kernel: a complex matrix in the N dimension is its
// row-major complex128 storage viewed as doubles (re, im interleaved = two real columns),
// a complex matrix in the M dimension is two real row blocks (planar).  With CPLX = true the
// A operand is complex planar (A, A2) and B/C are interleaved complex: two accumulator sets
// P = A B, Q = A2 B are combined in the lane that owns both (re, im) columns.
#pragma once
#include "dmma.cuh"

namespace afq {

struct GemmArgs {
  const double* A;   // A_KM ? [K][lda] (m contiguous) : [M][lda] (k contiguous)
  const double* A2;  // imaginary plane of A (CPLX only), same geometry
  const double* B;   // B_NK ? [N][ldb] (k contiguous) : [K][ldb] (n contiguous)
  double* C;         // [M][ldc]
  double* C2;        // optional second output (mode 1: C2 += C, mode 2: C2 = C)
  long lda, ldb, ldc;
  long sA, sB, sC;   // batch strides in doubles (0 = shared operand)
  int M, N, K, batch;
  int splitK;        // >1: K is cut in splitK ranges, slice s written to C + s * sCsplit
  long sCsplit;
  double alpha;
  int mode;          // 0 plain, 1 Taylor (C = alpha*acc, C2 += C), 2 dual write
  int vecA, vecB, vecC;  // 16-byte alignment of the operand rows holds
};

template <int BM, int BN, int WM, int WN, bool A_KM, bool B_NK, bool CPLX, int STAGES>
struct GemmCfg {
  static constexpr int MI = BM / WM / 8, NI = BN / WN / 8;
  static constexpr int LDA_M = BM + 4, LDB_N = BN + 4;
  static constexpr int A_TILE = A_KM ? BK * LDA_M : BM * LDK;
  static constexpr int B_TILE = B_NK ? BN * LDK : BK * LDB_N;
  static constexpr int STAGE = A_TILE * (CPLX ? 2 : 1) + B_TILE;
  static constexpr size_t SMEM = (size_t)STAGES * STAGE * sizeof(double);
  static_assert(WM * WN == 8, "8 warps");
  static_assert(BM % (WM * 8) == 0 && BN % (WN * 8) == 0, "warp tiling");
};

template <int BM, int BN, int WM, int WN, bool A_KM, bool B_NK, bool CPLX, int STAGES>
__global__ void __launch_bounds__(kThreads, 1) gemm_dmma_kernel(GemmArgs p) {
  using Cfg = GemmCfg<BM, BN, WM, WN, A_KM, B_NK, CPLX, STAGES>;
  constexpr int MI = Cfg::MI, NI = Cfg::NI;
  extern __shared__ __align__(16) double smem[];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;
  const int wm0 = (warp / WN) * (MI * 8), wn0 = (warp % WN) * (NI * 8);
  const int n0 = blockIdx.x * BN, m0 = blockIdx.y * BM;
  const int b = blockIdx.z / p.splitK, ks = blockIdx.z % p.splitK;

  int kchunk = (p.K + p.splitK - 1) / p.splitK;
  kchunk = (kchunk + BK - 1) / BK * BK;
  const int kbeg = ks * kchunk;
  const int kend = min(p.K, kbeg + kchunk);
  const int KT = kend > kbeg ? (kend - kbeg + BK - 1) / BK : 0;

  const double* A = p.A + (long)b * p.sA;
  const double* A2 = CPLX ? p.A2 + (long)b * p.sA : nullptr;
  const double* B = p.B + (long)b * p.sB;
  const int mvalid = min(BM, p.M - m0), nvalid = min(BN, p.N - n0);

  auto load_stage = [&](int slot, int kt) {
    double* sa = smem + slot * Cfg::STAGE;
    double* sb = sa + Cfg::A_TILE * (CPLX ? 2 : 1);
    const int k0 = kbeg + kt * BK;
    const int kvalid = min(BK, kend - k0);
    if (A_KM) {
      load_nmajor_tile<BM>(sa, A + m0, p.lda, k0, kvalid, mvalid, p.vecA, p.A);
    } else {
      load_kmajor_tile<BM>(sa, [&](int r) { return r < mvalid ? A + (long)(m0 + r) * p.lda : nullptr; },
                           k0, kvalid, p.vecA, p.A);
      if (CPLX)
        load_kmajor_tile<BM>(sa + Cfg::A_TILE,
                             [&](int r) { return r < mvalid ? A2 + (long)(m0 + r) * p.lda : nullptr; },
                             k0, kvalid, p.vecA, p.A);
    }
    if (B_NK)
      load_kmajor_tile<BN>(sb, [&](int r) { return r < nvalid ? B + (long)(n0 + r) * p.ldb : nullptr; },
                           k0, kvalid, p.vecB, p.B);
    else
      load_nmajor_tile<BN>(sb, B + n0, p.ldb, k0, kvalid, nvalid, p.vecB, p.B);
  };

  double acc[MI][NI][2];
  double acq[CPLX ? MI : 1][CPLX ? NI : 1][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) {
      acc[i][j][0] = acc[i][j][1] = 0.0;
      if (CPLX) acq[CPLX ? i : 0][CPLX ? j : 0][0] = acq[CPLX ? i : 0][CPLX ? j : 0][1] = 0.0;
    }

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < KT) load_stage(s, s);
    cp_async_commit();
  }
  for (int kt = 0; kt < KT; ++kt) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    if (kt + STAGES - 1 < KT) load_stage((kt + STAGES - 1) % STAGES, kt + STAGES - 1);
    cp_async_commit();
    const double* sa = smem + (kt % STAGES) * Cfg::STAGE;
    const double* sb = sa + Cfg::A_TILE * (CPLX ? 2 : 1);
    mma_stage<MI, NI, A_KM, B_NK, Cfg::LDA_M, Cfg::LDB_N>(sa, sb, wm0, wn0, g, t, acc);
    if constexpr (CPLX)
      mma_stage<MI, NI, A_KM, B_NK, Cfg::LDA_M, Cfg::LDB_N>(sa + Cfg::A_TILE, sb, wm0, wn0, g, t, acq);
  }
  cp_async_wait<0>();

  // epilogue: each lane owns C[m][n], C[m][n+1] with n even
  double* C = p.C + (long)b * p.sC + (long)ks * p.sCsplit;
  double* C2 = p.C2 ? p.C2 + (long)b * p.sC : nullptr;
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int m = m0 + wm0 + 8 * i + g;
    if (m >= p.M) continue;
#pragma unroll
    for (int j = 0; j < NI; ++j) {
      const int n = n0 + wn0 + 8 * j + 2 * t;
      if (n >= p.N) continue;
      double v0, v1;
      if constexpr (CPLX) {
        v0 = p.alpha * (acc[i][j][0] - acq[i][j][1]);
        v1 = p.alpha * (acc[i][j][1] + acq[i][j][0]);
      } else {
        v0 = p.alpha * acc[i][j][0];
        v1 = p.alpha * acc[i][j][1];
      }
      const long off = (long)m * p.ldc + n;
      const bool two = (n + 1 < p.N);
      if (two && p.vecC) {
        *reinterpret_cast<double2*>(C + off) = make_double2(v0, v1);
        if (C2) {
          if (p.mode == 1) {
            double2 o = *reinterpret_cast<double2*>(C2 + off);
            *reinterpret_cast<double2*>(C2 + off) = make_double2(o.x + v0, o.y + v1);
          } else {
            *reinterpret_cast<double2*>(C2 + off) = make_double2(v0, v1);
          }
        }
      } else {
        C[off] = v0;
        if (two) C[off + 1] = v1;
        if (C2) {
          if (p.mode == 1) {
            C2[off] += v0;
            if (two) C2[off + 1] += v1;
          } else {
            C2[off] = v0;
            if (two) C2[off + 1] = v1;
          }
        }
      }
    }
  }
}

}  // namespace afq
