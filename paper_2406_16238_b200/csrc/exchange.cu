// exchange.cu - the exchange contraction of the local energy (Eq. 11,
// PAPER.md:94; D7): for every Cholesky vector g and walker w
//     T^g_w = Lrot^g [ns x M] * Theta_w [M x ns]      (real x complex, on DMMA)
//     expart += tr(T T) = sum_ij T_ij T_ji,   X_g = tr(T)
// fused: the T blocks never leave the SM.  One CTA owns G whole (g, w) blocks: rows are
// (g, i), columns are (re/im plane, j) of one walker; after the K = M loop the accumulators
// are staged through shared memory (aliasing the pipeline buffers) for the transposed product.
//
// Both operands are k-contiguous: Lrot rows [M], and ThT[w][plane][j][M] (the transposed,
// planar Theta written by the overlap kernel), so both tiles use the conflict-free LDK stride.
#include "internal.h"

namespace afq {

namespace {

// NP8: 8-column tiles per plane (Np = 8 NP8 >= ns).  Variant A (SPLIT = 1): every warp owns
// GW whole planes stacked in M (MI = GW * NP8), CTA tile = 4 GW gammas.  Variant B (SPLIT = 2,
// NP8 = 7, 8): rows per gamma padded to 64, two warps share a plane (MI = 4), CTA = 2 gammas.
template <int NP8, int GW, int SPLIT>
struct ExCfg {
  static constexpr int Np = 8 * NP8;
  static constexpr int RP = SPLIT == 1 ? Np : 64;            // padded rows per gamma
  static constexpr int G = SPLIT == 1 ? 4 * GW : 2;          // gammas per CTA
  static constexpr int MI = SPLIT == 1 ? GW * NP8 : 4;
  static constexpr int NI = NP8;
  static constexpr int BM = G * RP, BN = 2 * Np;
  static constexpr int STAGES = 3;
  static constexpr int STAGE = (BM + BN) * LDK;
  static constexpr int LDT = Np + 1;
  static constexpr size_t PIPE = (size_t)STAGES * STAGE * 8;
  static constexpr size_t STG = (size_t)G * 2 * RP * LDT * 8;
  static constexpr size_t SMEM = PIPE > STG ? PIPE : STG;
};

template <int NP8, int GW, int SPLIT>
__global__ void __launch_bounds__(kThreads, 1) exchange_kernel(ExArgs a) {
  using Cfg = ExCfg<NP8, GW, SPLIT>;
  constexpr int MI = Cfg::MI, NI = Cfg::NI, Np = Cfg::Np, RP = Cfg::RP, G = Cfg::G;
  constexpr int BM = Cfg::BM, BN = Cfg::BN, STAGES = Cfg::STAGES, LDT = Cfg::LDT;
  extern __shared__ __align__(16) double smem[];
  __shared__ double red[8 * 2];

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;
  const int w = blockIdx.x, grp = blockIdx.y;
  const int g0 = grp * G;
  const int M = a.M, ns = a.ns;

  // warp -> (first gamma-local row, plane)
  int wm0, wn0;
  if (SPLIT == 1) {
    wm0 = (warp >> 1) * (MI * 8);
    wn0 = (warp & 1) * Np;
  } else {
    wm0 = (warp >> 2) * RP + (warp & 1) * 32;
    wn0 = ((warp >> 1) & 1) * Np;
  }

  const bool vec = (M % 2 == 0);
  const double* LrotB = a.Lrot + (size_t)a.off * M;                    // + g * Nt * M + i * M
  const double* ThB = a.ThT + ((size_t)w * 2 * a.Nt + a.off) * M;      // + plane * Nt * M + j * M
  const size_t lrot_g = (size_t)a.Nt * M, th_pl = (size_t)a.Nt * M;
  auto rowA = [&](int r) -> const double* {
    const int gl = r / RP, i = r % RP;
    return (i < ns && g0 + gl < a.n_chol) ? LrotB + (size_t)(g0 + gl) * lrot_g + (size_t)i * M : nullptr;
  };
  auto rowB = [&](int r) -> const double* {
    const int pl = r / Np, j = r % Np;
    return (j < ns) ? ThB + (size_t)pl * th_pl + (size_t)j * M : nullptr;
  };
  const int KT = (M + BK - 1) / BK;
  auto load_stage = [&](int slot, int kt) {
    double* sa = smem + slot * Cfg::STAGE;
    double* sb = sa + BM * LDK;
    const int k0 = kt * BK, kvalid = min(BK, M - k0);
    load_kmajor_tile<BM>(sa, rowA, k0, kvalid, vec, a.Lrot);
    load_kmajor_tile<BN>(sb, rowB, k0, kvalid, vec, a.Lrot);
  };

  double acc[MI][NI][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

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
    const double* sb = sa + BM * LDK;
    mma_stage<MI, NI, false, true, 0, 0>(sa, sb, wm0, wn0, g, t, acc);
  }
  cp_async_wait<0>();
  __syncthreads();   // every warp is done reading the pipeline buffers: alias them

  // stage T: stT[(gl * 2 + plane) * RP + i][j], row stride LDT
  double* stT = smem;
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int r = wm0 + 8 * i + g;           // CTA row = gl * RP + i_in_plane
    const int gl = r / RP, ii = r % RP;
    const int pl = wn0 / Np;
#pragma unroll
    for (int j = 0; j < NI; ++j) {
      const int jj = 8 * j + 2 * t;
      double* dst = stT + ((size_t)(gl * 2 + pl) * RP + ii) * LDT + jj;
      dst[0] = acc[i][j][0];
      dst[1] = acc[i][j][1];
    }
  }
  __syncthreads();

  // tr(T T) over the CTA's gammas; padded entries are exact zeros
  double v[2] = {0.0, 0.0};
  for (int idx = tid; idx < G * ns * ns; idx += kThreads) {
    const int gl = idx / (ns * ns), rem = idx % (ns * ns);
    const int i = rem / ns, j = rem % ns;
    const double* pr = stT + (size_t)(gl * 2 + 0) * RP * LDT;
    const double* pi = stT + (size_t)(gl * 2 + 1) * RP * LDT;
    const double ar = pr[i * LDT + j], ai = pi[i * LDT + j];
    const double br = pr[j * LDT + i], bi = pi[j * LDT + i];
    v[0] += ar * br - ai * bi;
    v[1] += ar * bi + ai * br;
  }
  // X_g = tr(T_g): warp gl sums the diagonal of its gamma
  for (int gl = warp; gl < G; gl += 8) {
    double xr = 0.0, xi = 0.0;
    for (int i = lane; i < ns; i += 32) {
      xr += stT[((size_t)(gl * 2 + 0) * RP + i) * LDT + i];
      xi += stT[((size_t)(gl * 2 + 1) * RP + i) * LDT + i];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      xr += __shfl_down_sync(0xffffffffu, xr, o);
      xi += __shfl_down_sync(0xffffffffu, xi, o);
    }
    if (lane == 0 && g0 + gl < a.n_chol) {
      double* xo = a.X + ((size_t)(g0 + gl) * a.nw + w) * 2;
      if (a.accumulate) { xo[0] += xr; xo[1] += xi; } else { xo[0] = xr; xo[1] = xi; }
    }
  }
#pragma unroll
  for (int k = 0; k < 2; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  if (lane == 0) { red[warp * 2] = v[0]; red[warp * 2 + 1] = v[1]; }
  __syncthreads();
  if (tid == 0) {
    double sr = 0.0, si = 0.0;
    for (int k = 0; k < 8; ++k) { sr += red[2 * k]; si += red[2 * k + 1]; }
    double* eo = a.expart + ((size_t)grp * a.nw + w) * 2;
    eo[0] = sr;
    eo[1] = si;
  }
}

template <int NP8, int GW, int SPLIT>
int launch_ex(const ExArgs& a, cudaStream_t st) {
  using Cfg = ExCfg<NP8, GW, SPLIT>;
  auto kern = exchange_kernel<NP8, GW, SPLIT>;
  static uint64_t done = 0;
  if (auto once_ = first_use_on_device(&done)) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::SMEM);
  }
  dim3 grid(a.nw, (a.n_chol + Cfg::G - 1) / Cfg::G);
  kern<<<grid, kThreads, Cfg::SMEM, st>>>(a);
  return 1;
}

__global__ void __launch_bounds__(256) energy_reduce_kernel(EnergyArgs a, const double* expart2, int ngroups2) {
  __shared__ double red[8 * 4];
  const int w = blockIdx.x;
  double v[4] = {0.0, 0.0, 0.0, 0.0};   // sum X^2 (re, im), sum tr(TT) (re, im)
  for (int gq = threadIdx.x; gq < a.n_chol; gq += blockDim.x) {
    const double xr = a.spin_factor * a.X[((size_t)gq * a.nw + w) * 2];
    const double xi = a.spin_factor * a.X[((size_t)gq * a.nw + w) * 2 + 1];
    v[0] += xr * xr - xi * xi;
    v[1] += 2.0 * xr * xi;
  }
  for (int q = threadIdx.x; q < a.ngroups; q += blockDim.x) {
    v[2] += a.expart[((size_t)q * a.nw + w) * 2];
    v[3] += a.expart[((size_t)q * a.nw + w) * 2 + 1];
  }
  if (expart2)
    for (int q = threadIdx.x; q < ngroups2; q += blockDim.x) {
      v[2] += expart2[((size_t)q * a.nw + w) * 2];
      v[3] += expart2[((size_t)q * a.nw + w) * 2 + 1];
    }
  // block sum
#pragma unroll
  for (int k = 0; k < 4; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0)
    for (int k = 0; k < 4; ++k) red[warp * 4 + k] = v[k];
  __syncthreads();
  if (threadIdx.x == 0) {
    double s[4] = {0, 0, 0, 0};
    for (int q = 0; q < 8; ++q)
      for (int k = 0; k < 4; ++k) s[k] += red[q * 4 + k];
    double e1r = 0.0, e1i = 0.0;
    for (int b = 0; b < a.nblk; ++b) {
      e1r += a.e1[((size_t)w * a.nblk + b) * 2];
      e1i += a.e1[((size_t)w * a.nblk + b) * 2 + 1];
    }
    e1r *= a.spin_factor;
    e1i *= a.spin_factor;
    const double e2r = 0.5 * s[0] - 0.5 * a.spin_factor * s[2];
    const double e2i = 0.5 * s[1] - 0.5 * a.spin_factor * s[3];
    double* o = a.E_out + (size_t)w * 6;
    o[0] = e1r + e2r; o[1] = e1i + e2i;
    o[2] = e1r;       o[3] = e1i;
    o[4] = e2r;       o[5] = e2i;
  }
}

}  // namespace

static int np8_of(int ns) { return (ns + 7) / 8; }

int exchange_group_size(int ns) {
  switch (np8_of(ns)) {
    case 1: return ExCfg<1, 8, 1>::G;
    case 2: return ExCfg<2, 4, 1>::G;
    case 3: return ExCfg<3, 2, 1>::G;
    case 4: return ExCfg<4, 2, 1>::G;
    case 5: return ExCfg<5, 1, 1>::G;
    case 6: return ExCfg<6, 1, 1>::G;
    default: return 2;
  }
}

int run_exchange(const ExArgs& a, cudaStream_t st) {
  switch (np8_of(a.ns)) {
    case 1: return launch_ex<1, 8, 1>(a, st);
    case 2: return launch_ex<2, 4, 1>(a, st);
    case 3: return launch_ex<3, 2, 1>(a, st);
    case 4: return launch_ex<4, 2, 1>(a, st);
    case 5: return launch_ex<5, 1, 1>(a, st);
    case 6: return launch_ex<6, 1, 1>(a, st);
    case 7: return launch_ex<7, 1, 2>(a, st);
    case 8: return launch_ex<8, 1, 2>(a, st);
  }
  return 0;
}

// two (expart, ngroups) pairs: UHF blocks use different tile shapes
int run_energy_reduce2(const EnergyArgs& a, const double* expart2, int ngroups2, cudaStream_t st) {
  energy_reduce_kernel<<<a.nw, 256, 0, st>>>(a, expart2, ngroups2);
  return 1;
}
int run_energy_reduce(const EnergyArgs& a, cudaStream_t st) { return run_energy_reduce2(a, nullptr, 0, st); }

}  // namespace afq
