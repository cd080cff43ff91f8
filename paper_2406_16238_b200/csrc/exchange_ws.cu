// exchange_ws.cu - exchange contraction of the local energy (Eq. 11,
// PAPER.md:94; D7), warp-specialised TMA version:
//     T^g_w = Lrot^g [ns x M] * Theta_w [M x ns],   expart += tr(T T),   X_g = tr(T)
//
// One persistent CTA per SM.  A producer warp feeds a ring of shared-memory stages with TMA
// (cp.async.bulk.tensor, SWIZZLE_128B, mbarrier full/empty pairs); WM x WN consumer warps
// issue nothing but 16-byte fragment loads and DMMA.  A tile is G whole Cholesky vectors
// (rows (g, i), taken UNPADDED out of Lrot[n_chol][Nt][M] by a 3-D box) times Wn whole
// walkers (columns (w, plane, j) out of ThT[nw][2][Nt][M] by a 4-D box), so the only padding
// is the round-up of G*ns and Wn*2*ns to the warp grid.  After the K = M loop the tile is
// staged through shared memory Wp walkers at a time for tr(T T) and tr(T); T never reaches HBM.
#include "internal.h"
#include "tma.cuh"

namespace afq {

namespace {

constexpr int kProducerThreads = 128;     // one warpgroup (setmaxnreg is warpgroup-wide)
constexpr int kSmemMax = 232448;          // 227 KB opt-in limit per CTA

struct XwsArgs {
  double* expart;      // [ngroups][nw] complex
  double* X;           // [n_chol][nw] complex
  int M, ns, off, n_chol, nw;
  int G, Wn, Wp;       // gammas / walkers per tile, walkers per epilogue pass
  int ldt;             // staging row stride (doubles), odd
  int stages;
  int ntile_w, ntiles;
  int accumulate;
  int split;           // epilogue work items per (gamma, walker)
};

template <int WM, int WN, int MI, int NI>
struct XwsCfg {
  static constexpr int NCW = WM * WN;
  static constexpr int NCT = NCW * 32;
  static constexpr int THREADS = NCT + kProducerThreads;
  static constexpr int TA = 8 * WM * MI, TB = 8 * WN * NI;
  static constexpr int STAGE_BYTES = (TA + TB) * 128;
  static constexpr int CREGS = ((65536 - kProducerThreads * 24) / NCT) / 8 * 8 > 240
                                   ? 240 : ((65536 - kProducerThreads * 24) / NCT) / 8 * 8;
  static constexpr int MAXITEMS = 256;    // comb slots
};

template <int WM, int WN, int MI, int NI>
__global__ void __launch_bounds__(XwsCfg<WM, WN, MI, NI>::THREADS, 1)
exchange_ws_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB,
                   const XwsArgs a) {
  using Cfg = XwsCfg<WM, WN, MI, NI>;
  constexpr int NCW = Cfg::NCW, NCT = Cfg::NCT, TA = Cfg::TA;
  extern __shared__ unsigned char smem_raw[];
  // SWIZZLE_128B tiles need a 1024-byte aligned base (the launch adds the slack)
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int S = a.stages;
  unsigned char* tiles = smem;
  double* stg = reinterpret_cast<double*>(smem + (size_t)S * Cfg::STAGE_BYTES);
  const int RAp = (a.G * a.ns + 7) & ~7;
  double* comb = stg + (size_t)RAp * a.ldt;                       // [MAXITEMS][4]
  uint64_t* full = reinterpret_cast<uint64_t*>(comb + Cfg::MAXITEMS * 4);
  uint64_t* empty = full + S;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KT = (a.M + 15) >> 4;

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
    fence_barrier_init();
  }
  // rows of the A / B tiles that TMA never writes (round-up of G*ns, Wn*2*ns) must read as
  // finite numbers: zero all stages once
  {
    uint4* z = reinterpret_cast<uint4*>(tiles);
    const int n16 = S * Cfg::STAGE_BYTES / 16;
    for (int i = tid; i < n16; i += Cfg::THREADS) z[i] = make_uint4(0, 0, 0, 0);
  }
  fence_proxy_async();
  __syncthreads();

  if (warp >= NCW) {
    // ------------------------------------------------------------------ producer warpgroup
    reg_dealloc<24>();
    if (warp == NCW && lane == 0) {
      prefetch_tensormap(&tmA);
      prefetch_tensormap(&tmB);
      const uint32_t bytes = (uint32_t)(a.G * a.ns + a.Wn * 2 * a.ns) * 128u;
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
        const int g0 = (tile / a.ntile_w) * a.G, w0 = (tile % a.ntile_w) * a.Wn;
        for (int kt = 0; kt < KT; ++kt, ++it) {
          const int s = it % S;
          const uint32_t ph = (it / S) & 1;
          mbar_wait(&empty[s], ph ^ 1);
          mbar_expect_tx(&full[s], bytes);
          unsigned char* sa = tiles + (size_t)s * Cfg::STAGE_BYTES;
          tma_load_3d(sa, &tmA, &full[s], kt * 16, a.off, g0);
          tma_load_4d(sa + TA * 128, &tmB, &full[s], kt * 16, a.off, 0, w0);
        }
      }
    }
    return;
  }

  // -------------------------------------------------------------------- consumer warps
  reg_alloc<Cfg::CREGS>();
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp % WM, wn = warp / WM;
  const int p = rperm(g);
  const uint32_t lane0 = (uint32_t)(p * 128 + ((t ^ p) << 4));
  const uint32_t lane1 = (uint32_t)(p * 128 + (((t ^ p) ^ 4) << 4));
  const uint32_t tiles_u32 = smem_u32(tiles);
  const uint32_t aoff = (uint32_t)(wm * MI) * 1024u;
  const uint32_t boff = (uint32_t)(TA * 128) + (uint32_t)(wn * NI) * 1024u;
  const int ns = a.ns, RA = a.G * ns;

  uint32_t it = 0;
  for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
    const int tg = tile / a.ntile_w;
    const int g0 = tg * a.G, w0 = (tile % a.ntile_w) * a.Wn;

    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kt = 0; kt < KT; ++kt, ++it) {
      const int s = it % S;
      mbar_wait(&full[s], (it / S) & 1);
      consumer_release_prev(empty, it, S, lane);
      const uint32_t sa = tiles_u32 + (uint32_t)s * Cfg::STAGE_BYTES + aoff;
      const uint32_t sb = tiles_u32 + (uint32_t)s * Cfg::STAGE_BYTES + boff;
#pragma unroll
      for (int kp = 0; kp < 2; ++kp) {
        const uint32_t lo = kp ? lane1 : lane0;
        double2 af[MI];
#pragma unroll
        for (int i = 0; i < MI; ++i) af[i] = lds128(sa + i * 1024 + lo);
#pragma unroll
        for (int j = 0; j < NI; ++j) {
          const double2 bf = lds128(sb + j * 1024 + lo);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], af[i].x, bf.x);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], af[i].y, bf.y);
        }
      }
    }

    // ------------------------------------------------------------------ epilogue
    const int ldt = a.ldt;
    const int nsns = ns * ns;
    for (int wp0 = 0; wp0 < a.Wn; wp0 += a.Wp) {
      const int Wp = min(a.Wp, a.Wn - wp0);
      const int clo = wp0 * 2 * ns, chi = (wp0 + Wp) * 2 * ns;
      // (1) stage the columns of walkers [wp0, wp0 + Wp)
#pragma unroll
      for (int i = 0; i < MI; ++i) {
        const int r = 8 * (wm * MI + i) + p;
        if (r < RA) {
#pragma unroll
          for (int j = 0; j < NI; ++j) {
            const int c = 8 * (wn * NI + j) + t;
            if (c >= clo && c < chi) stg[(size_t)r * ldt + (c - clo)] = acc[i][j][0];
            if (c + 4 >= clo && c + 4 < chi) stg[(size_t)r * ldt + (c + 4 - clo)] = acc[i][j][1];
          }
        }
      }
      named_bar_sync(1, NCT);
      // (2) work items (gamma_local, walker_local, slice of the (i, j) range)
      const int nitems = a.G * Wp * a.split;
      const int chunk = (nsns + a.split - 1) / a.split;
      for (int item = warp; item < nitems; item += NCW) {
        const int sl = item % a.split, gw = item / a.split;
        const int wl = gw % Wp, gl = gw / Wp;
        const double* pr = stg + (size_t)(gl * ns) * ldt + wl * 2 * ns;
        const double* pi = pr + ns;
        double vr = 0.0, vi = 0.0, xr = 0.0, xi = 0.0;
        const int e1 = min(nsns, (sl + 1) * chunk);
        for (int idx = sl * chunk + lane; idx < e1; idx += 32) {
          const int i = idx / ns, j = idx - i * ns;
          const double ar = pr[i * ldt + j], ai = pi[i * ldt + j];
          const double br = pr[j * ldt + i], bi = pi[j * ldt + i];
          vr += ar * br - ai * bi;
          vi += ar * bi + ai * br;
          if (i == j) { xr += ar; xi += ai; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          vr += __shfl_down_sync(0xffffffffu, vr, o);
          vi += __shfl_down_sync(0xffffffffu, vi, o);
          xr += __shfl_down_sync(0xffffffffu, xr, o);
          xi += __shfl_down_sync(0xffffffffu, xi, o);
        }
        if (lane == 0) {
          comb[item * 4 + 0] = vr; comb[item * 4 + 1] = vi;
          comb[item * 4 + 2] = xr; comb[item * 4 + 3] = xi;
        }
      }
      named_bar_sync(1, NCT);
      // (3) fixed-order final sums
      for (int wl = tid; wl < Wp; wl += NCT) {
        const int w = w0 + wp0 + wl;
        if (w < a.nw) {
          double sr = 0.0, si = 0.0;
          for (int gl = 0; gl < a.G; ++gl)
            for (int sl = 0; sl < a.split; ++sl) {
              const int item = (gl * Wp + wl) * a.split + sl;
              sr += comb[item * 4 + 0];
              si += comb[item * 4 + 1];
            }
          double* eo = a.expart + ((size_t)tg * a.nw + w) * 2;
          eo[0] = sr; eo[1] = si;
        }
      }
      for (int gw = NCT - 1 - tid; gw < a.G * Wp; gw += NCT) {
        const int wl = gw % Wp, gl = gw / Wp;
        const int w = w0 + wp0 + wl, gg = g0 + gl;
        if (w < a.nw && gg < a.n_chol) {
          double xr = 0.0, xi = 0.0;
          for (int sl = 0; sl < a.split; ++sl) {
            xr += comb[(gw * a.split + sl) * 4 + 2];
            xi += comb[(gw * a.split + sl) * 4 + 3];
          }
          double* xo = a.X + ((size_t)gg * a.nw + w) * 2;
          if (a.accumulate) { xo[0] += xr; xo[1] += xi; } else { xo[0] = xr; xo[1] = xi; }
        }
      }
      // the next pass (or tile) overwrites stg / comb only after its own first barrier;
      // that barrier is reached by every thread after it has finished (3)
      named_bar_sync(1, NCT);
    }
  }
}

struct Plan {
  int cfg = -1;       // index into the instantiation table
  int G = 0, Wn = 0, Wp = 0, ldt = 0, stages = 0, split = 1;
  size_t smem = 0;
  double eff = 0.0;
};

struct Inst { int WM, WN, MI, NI; };
constexpr Inst kInst[] = {{4, 3, 4, 7}, {4, 2, 5, 5}, {4, 2, 5, 7}, {4, 2, 6, 6}};
constexpr int kNumInst = sizeof(kInst) / sizeof(kInst[0]);

Plan make_plan(int ns) {
  Plan best;
  for (int c = 0; c < kNumInst; ++c) {
    const Inst& I = kInst[c];
    const int TA = 8 * I.WM * I.MI, TB = 8 * I.WN * I.NI, ncw = I.WM * I.WN;
    Plan p;
    p.cfg = c;
    p.G = TA / ns;
    p.Wn = TB / (2 * ns);
    if (p.G < 1 || p.Wn < 1) continue;
    if (p.G > 256) p.G = 256;
    if (p.Wn > 256) p.Wn = 256;
    p.eff = (double)(p.G * ns) * (p.Wn * 2 * ns) / ((double)TA * TB);
    const int RAp = (p.G * ns + 7) & ~7;
    const size_t fixed = 256 * 4 * 8 + 2 * 8 * 8 + 1024;   // comb + barriers + alignment slack
    // The staging shape with the FEWEST epilogue passes first (Wp walkers of the tile at a time), then the deepest
    // ring that still fits beside it.  Measured on B200: the operands come out of L2 and two stages already keep
    // the DMMA pipe fed, while every extra epilogue pass costs three CTA-wide barriers (c2: 5 passes with 4 stages
    // 4.26 ms, 2 passes with 2 stages 3.4 ms; c5 and c4 keep 3 stages and 2 passes).
    bool ok = false;
    int best_passes = 1 << 30;
    for (int S = 4; S >= 2; --S) {
      const size_t pipe = (size_t)S * (TA + TB) * 128;
      for (int Wp = p.Wn; Wp >= 1; --Wp) {
        const int ldt = (Wp * 2 * ns) | 1;
        const size_t tot = pipe + (size_t)RAp * ldt * 8 + fixed;
        if (tot > (size_t)kSmemMax) continue;
        int split = 1, wp = Wp;
        while (p.G * wp * split < ncw && split < 8) split *= 2;
        while (p.G * wp * split > 256 && wp > 1) wp -= 1;      // items per pass must fit the comb table
        if (p.G * wp * split > 256) continue;
        const int passes = (p.Wn + wp - 1) / wp;
        if (passes < best_passes) {             // strictly fewer: the deeper ring wins ties (S descends)
          best_passes = passes;
          p.stages = S; p.Wp = wp; p.ldt = (wp * 2 * ns) | 1; p.split = split;
          p.smem = pipe + (size_t)RAp * p.ldt * 8 + fixed;
          ok = true;
        }
        break;                                  // smaller Wp only means more passes at this S
      }
    }
    if (!ok) continue;
    if (p.eff > best.eff + 1e-9) best = p;
  }
  return best;
}

template <int WM, int WN, int MI, int NI>
int launch_xws(const ExArgs& e, const Plan& p, cudaStream_t st) {
  using Cfg = XwsCfg<WM, WN, MI, NI>;
  auto kern = exchange_ws_kernel<WM, WN, MI, NI>;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  }
  const int nsm = sm_count_current();
  TensorMap tmA, tmB;
  {
    const uint64_t dims[3] = {(uint64_t)e.M, (uint64_t)e.Nt, (uint64_t)e.n_chol};
    const uint64_t str[2] = {(uint64_t)e.M * 8, (uint64_t)e.Nt * e.M * 8};
    const uint32_t box[3] = {16, (uint32_t)e.ns, (uint32_t)p.G};
    if (make_tensor_map_f64(&tmA, e.Lrot, 3, dims, str, box) != 0) return -1;
  }
  {
    const uint64_t dims[4] = {(uint64_t)e.M, (uint64_t)e.Nt, 2, (uint64_t)e.nw};
    const uint64_t str[3] = {(uint64_t)e.M * 8, (uint64_t)e.Nt * e.M * 8, (uint64_t)2 * e.Nt * e.M * 8};
    const uint32_t box[4] = {16, (uint32_t)e.ns, 2, (uint32_t)p.Wn};
    if (make_tensor_map_f64(&tmB, e.ThT, 4, dims, str, box) != 0) return -1;
  }
  XwsArgs a;
  a.expart = e.expart; a.X = e.X;
  a.M = e.M; a.ns = e.ns; a.off = e.off; a.n_chol = e.n_chol; a.nw = e.nw;
  a.G = p.G; a.Wn = p.Wn; a.Wp = p.Wp; a.ldt = p.ldt; a.stages = p.stages; a.split = p.split;
  a.ntile_w = (e.nw + p.Wn - 1) / p.Wn;
  a.ntiles = a.ntile_w * ((e.n_chol + p.G - 1) / p.G);
  a.accumulate = e.accumulate;
  const int grid = a.ntiles < nsm ? a.ntiles : nsm;
  kern<<<grid, Cfg::THREADS, p.smem, st>>>(tmA, tmB, a);
  return 1;
}

}  // namespace

bool exchange_ws_usable(int M, const void* Lrot, const void* ThT) {
  return (M % 2 == 0) && (((uintptr_t)Lrot | (uintptr_t)ThT) & 15) == 0;
}

int exchange_ws_group_size(int ns) { return make_plan(ns).G; }

double exchange_ws_efficiency(int ns) { return make_plan(ns).eff; }

// returns launches issued, or -1 if the tensor maps could not be encoded
int run_exchange_ws(const ExArgs& e, cudaStream_t st) {
  const Plan p = make_plan(e.ns);
  if (p.cfg < 0) return -1;
  switch (p.cfg) {
    case 0: return launch_xws<4, 3, 4, 7>(e, p, st);
    case 1: return launch_xws<4, 2, 5, 5>(e, p, st);
    case 2: return launch_xws<4, 2, 5, 7>(e, p, st);
    case 3: return launch_xws<4, 2, 6, 6>(e, p, st);
  }
  return -1;
}

}  // namespace afq
