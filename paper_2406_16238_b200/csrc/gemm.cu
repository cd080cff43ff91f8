// gemm.cu - tile-configuration dispatch for the DMMA GEMM (gemm.cuh).
#include "internal.h"

namespace afq {

template <int BM, int BN, int WM, int WN, bool A_KM, bool B_NK, bool CPLX, int STAGES>
static int launch_cfg(const GemmArgs& a, cudaStream_t st) {
  using Cfg = GemmCfg<BM, BN, WM, WN, A_KM, B_NK, CPLX, STAGES>;
  auto kern = gemm_dmma_kernel<BM, BN, WM, WN, A_KM, B_NK, CPLX, STAGES>;
  static uint64_t attr_done = 0;
  if (auto once_ = first_use_on_device(&attr_done)) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
  }
  dim3 grid((a.N + BN - 1) / BN, (a.M + BM - 1) / BM, a.batch * a.splitK);
  kern<<<grid, kThreads, Cfg::SMEM, st>>>(a);
  return 1;
}

static bool al16(const void* p) { return ((uintptr_t)p & 15) == 0; }

template <bool CPLX>
static int launch_narrow(const GemmArgs& a, cudaStream_t st) {
  // N fits one or a few n-tiles: pick the tile width with the least padding.
  constexpr int BMn = CPLX ? 64 : 128;
  const int cands[5] = {32, 64, 96, 112, 128};
  int best = 128;
  long bestcost = 1L << 60;
  for (int c : cands) {
    long cost = (long)((a.N + c - 1) / c) * c;
    if (cost < bestcost) { bestcost = cost; best = c; }
  }
  switch (best) {
    case 32: return launch_cfg<BMn, 32, 4, 2, false, false, CPLX, 4>(a, st);
    case 64: return launch_cfg<BMn, 64, 4, 2, false, false, CPLX, 4>(a, st);
    case 96: return launch_cfg<BMn, 96, 4, 2, false, false, CPLX, 4>(a, st);
    case 112: return launch_cfg<BMn, 112, 4, 2, false, false, CPLX, 4>(a, st);
    default: return launch_cfg<BMn, 128, 4, 2, false, false, CPLX, 4>(a, st);
  }
}

int run_gemm(GemmKind kind, GemmArgs a, cudaStream_t st) {
  if (a.M <= 0 || a.N <= 0 || a.batch <= 0) return 0;
  if (a.splitK < 1) a.splitK = 1;
  const bool stridesA = (a.lda % 2 == 0) && (a.sA % 2 == 0);
  const bool stridesB = (a.ldb % 2 == 0) && (a.sB % 2 == 0);
  a.vecA = stridesA && al16(a.A) && (a.A2 == nullptr || al16(a.A2));
  a.vecB = stridesB && al16(a.B);
  a.vecC = (a.ldc % 2 == 0) && (a.sC % 2 == 0) && (a.sCsplit % 2 == 0) && al16(a.C) &&
           (a.C2 == nullptr || al16(a.C2));
  switch (kind) {
    case GEMM_KN:
      if (a.N <= 128) return launch_narrow<false>(a, st);
      if (a.M <= 64) return launch_cfg<64, 128, 4, 2, false, false, false, 4>(a, st);
      return launch_cfg<128, 128, 2, 4, false, false, false, 4>(a, st);
    case GEMM_NK:
      return launch_cfg<128, 128, 2, 4, false, true, false, 4>(a, st);
    case GEMM_KMKN:
      return launch_cfg<128, 128, 2, 4, true, false, false, 4>(a, st);
    case GEMM_CPLX_KN:
      return launch_narrow<true>(a, st);
  }
  return 0;
}

}  // namespace afq
