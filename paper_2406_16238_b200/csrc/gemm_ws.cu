// gemm_ws.cu - warp-specialised TMA + DMMA GEMMs for the medium-sized contractions of the step:
//
//   KN (batched):  C[b][m][n] = alpha * sum_k A[b](m,k) B[b](k,n)
//       A k-major (one or two planes: CPLX = planar complex A), B n-major with N = 2 Nt
//       (interleaved complex columns), one CTA tile = 64*MI rows x all N columns.
//       a6/a8 one-body propagator (A = E1 shared by the batch), a7 Taylor terms (CPLX,
//       C = alpha * A T, C2 += C).                       (Eqs. 7, 9, 12)
//   NK (split-K):  C[s][m][n] = sum_{k in slice s} A(m,k) B(n,k), both k-major.
//       a3 force bias X = ThT * Lrot^T.                  (Eq. 14)
//
// Same pipeline as exchange_ws.cu: one producer lane issues cp.async.bulk.tensor boxes of 16 k
// (SWIZZLE_128B) into an mbarrier ring, the consumer warps only load fragments and issue DMMA.
#include "internal.h"
#include "tma.cuh"

namespace afq {

namespace {

constexpr int kProdT = 128;
constexpr int kSmemCap = 232448;

int sm_count() { return sm_count_current(); }

// ------------------------------------------------------------------------------------ KN
struct KnArgs {
  double* C;
  double* C2;
  long ldc, sC;
  double alpha;
  int mode;            // 0 plain, 1 Taylor (C = v, C2 += v), 2 dual write
  int M, N, K, batch;
  int mtiles, ntiles_n;
  int a_shared;        // A is the same matrix for every batch entry
  int stages;
  int nb16;            // 16-column boxes of B per n tile
  // stream-K (sk_w > 0): CTA c works on the k iterations [c sk_w, (c + 1) sk_w) of the tile-major iteration space, so
  // every SM gets the same amount of work whatever the tile count; a tile cut by a chunk boundary is finished by
  // the CTA holding its LAST part, which adds the first part's accumulators out of sk_part[c - 1]
  int sk_w;
  double* sk_part;     // [grid][PL * MI * NI * 2][256]
  int* sk_flag;        // [grid], zero between launches
};

// Work of one CTA as a short list of segments (tile, k range, mode): 0 whole tile, 1 first part of a tile whose rest
// belongs to CTA c + 1 (accumulators go to sk_part[c]), 2 last part of a tile started by CTA c - 1.  The first part
// comes FIRST so that the neighbour never waits long.
// Forward progress of the spin wait (CTA c polls the flag CTA c - 1 sets): parking depends on nothing - a CTA parks
// before it ever waits - so a CTA that has been dispatched always reaches its atomicExch.  CTA c therefore only needs
// CTA c - 1 to have been DISPATCHED, not to be co-resident with it: the grid is at most one CTA per SM and the
// hardware hands out CTAs of a grid in increasing blockIdx order, so this holds alone on the device and also when
// other kernels (another handle's stream, torch, MPS clients) occupy some SMs - a CTA that is running had all its
// predecessors started before it.  What it does NOT survive is a scheduler that starts CTA c while withholding
// CTA c - 1 for good; no CUDA device does that today, and a cooperative launch would make it a guarantee at the
// price of refusing to run beside other work.
struct KnSeg { int tile, kb, ke, mode; };
__device__ __forceinline__ bool kn_segment(const KnArgs& a, int KT, int ntiles, int idx, KnSeg& s) {
  if (a.sk_w <= 0) {
    s.tile = blockIdx.x + idx * gridDim.x; s.kb = 0; s.ke = KT; s.mode = 0;
    return s.tile < ntiles;
  }
  const long total = (long)ntiles * KT;
  const long begin = (long)blockIdx.x * a.sk_w, end = min(begin + a.sk_w, total);
  if (begin >= end) return false;
  const int ft = (int)(begin / KT), kb = (int)(begin % KT);
  const int lt = (int)((end - 1) / KT), ke = (int)((end - 1) % KT) + 1;
  const bool head = ke < KT, tail = kb > 0;
  if (head) {
    if (idx == 0) { s.tile = lt; s.kb = 0; s.ke = ke; s.mode = 1; return true; }
    idx -= 1;
  }
  const int f0 = ft + (tail ? 1 : 0), l0 = lt - (head ? 1 : 0);
  if (idx <= l0 - f0) { s.tile = f0 + idx; s.kb = 0; s.ke = KT; s.mode = 0; return true; }
  idx -= (l0 - f0 + 1);
  if (tail && idx == 0) { s.tile = ft; s.kb = kb; s.ke = KT; s.mode = 2; return true; }
  return false;
}

template <int MI, int NI, bool CPLX>
struct KnCfg {
  static constexpr int NCW = 8, NCT = 256, THREADS = NCT + kProdT;
  static constexpr int BM = 64 * MI;
  static constexpr int PL = CPLX ? 2 : 1;
  static constexpr int A_BYTES = PL * BM * 128;
  static constexpr int NB16 = (NI + 1) / 2;
  static constexpr int B_BYTES = NB16 * 2048;
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
};

template <int MI, int NI, bool CPLX>
__global__ void __launch_bounds__(KnCfg<MI, NI, CPLX>::THREADS, 1)
gemm_ws_kn_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB, const KnArgs a) {
  using Cfg = KnCfg<MI, NI, CPLX>;
  constexpr int NCW = Cfg::NCW, BM = Cfg::BM, PL = Cfg::PL, NB16 = Cfg::NB16;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int S = a.stages;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)S * Cfg::STAGE_BYTES);
  uint64_t* empty = full + S;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KT = (a.K + 15) >> 4;
  const int per_b = a.mtiles * a.ntiles_n;
  const int ntiles = per_b * a.batch;

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
    fence_barrier_init();
  }
  __syncthreads();

  if (warp >= NCW) {
    reg_dealloc<24>();
    if (warp == NCW && lane == 0) {
      prefetch_tensormap(&tmA);
      prefetch_tensormap(&tmB);
      uint32_t it = 0;
      KnSeg sg;
      for (int si = 0; kn_segment(a, KT, ntiles, si, sg); ++si) {
        const int tile = sg.tile;
        const int b = tile / per_b, rem = tile % per_b;
        const int mt = rem / a.ntiles_n, nt = rem % a.ntiles_n;
        for (int kt = sg.kb; kt < sg.ke; ++kt, ++it) {
          const int s = it % S;
          mbar_wait(&empty[s], ((it / S) & 1) ^ 1);
          mbar_expect_tx(&full[s], Cfg::STAGE_BYTES);
          unsigned char* sa = smem + (size_t)s * Cfg::STAGE_BYTES;
          tma_load_4d(sa, &tmA, &full[s], kt * 16, mt * BM, 0, a.a_shared ? 0 : b);
#pragma unroll
          for (int q = 0; q < NB16; ++q)
            tma_load_3d(sa + Cfg::A_BYTES + q * 2048, &tmB, &full[s], (nt * NB16 + q) * 16, kt * 16, b);
        }
      }
    }
    return;
  }

  reg_alloc<240>();
  const int g = lane >> 2, t = lane & 3;
  const int p = rperm(g);
  const uint32_t la0 = (uint32_t)(p * 128 + ((t ^ p) << 4));
  const uint32_t la1 = (uint32_t)(p * 128 + (((t ^ p) ^ 4) << 4));
  uint32_t lb[2][2];   // [kp][par], half h = 0; h = 1 is the same offset ^ 64
#pragma unroll
  for (int kp = 0; kp < 2; ++kp)
#pragma unroll
    for (int par = 0; par < 2; ++par) {
      const int k = 8 * kp + 2 * t + par;
      lb[kp][par] = (uint32_t)(k * 128 + (((g >> 1) ^ (k & 7)) << 4) + (g & 1) * 8);
    }
  // Paired blocks: ONE 16-byte load per k row gives a lane the columns (2 g, 2 g + 1) of a 16-column box, i.e. the B
  // fragments of TWO blocks whose columns are interleaved (block 2 j2 takes the even columns of box j2, block
  // 2 j2 + 1 the odd ones; the epilogue undoes the interleave).  Half the fragment-load instructions of the 8-byte
  // loads; an unpaired last block (odd NI) keeps them.
  uint32_t lbp[2][2];
#pragma unroll
  for (int kp = 0; kp < 2; ++kp)
#pragma unroll
    for (int par = 0; par < 2; ++par) {
      const int k = 8 * kp + 2 * t + par;
      lbp[kp][par] = (uint32_t)(k * 128 + ((g ^ (k & 7)) << 4));
    }
  // measured on B200: pairing gains 2.5 % (NI = 11, c5), 5 % (13, c3), 9 % (8, c2) on the Taylor GEMM and loses 4 % for
  // the planar-complex kernel at NI = 10 (c4), which therefore keeps the 8-byte loads
  constexpr int NP = (CPLX && NI == 10) ? 0 : NI / 2;           // paired boxes
  const uint32_t smem_u = smem_u32(smem);
  const uint32_t aoff = (uint32_t)(warp * MI) * 1024u;

  uint32_t it = 0;
  KnSeg sg;
  for (int si = 0; kn_segment(a, KT, ntiles, si, sg); ++si) {
    const int tile = sg.tile;
    const int b = tile / per_b, rem = tile % per_b;
    const int mt = rem / a.ntiles_n, nt = rem % a.ntiles_n;

    double acc[PL][MI][NI][2];
#pragma unroll
    for (int pl = 0; pl < PL; ++pl)
#pragma unroll
      for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NI; ++j) acc[pl][i][j][0] = acc[pl][i][j][1] = 0.0;

    for (int kt = sg.kb; kt < sg.ke; ++kt, ++it) {
      const int s = it % S;
      mbar_wait(&full[s], (it / S) & 1);
      consumer_release_prev(empty, it, S, lane);
      const uint32_t sa = smem_u + (uint32_t)s * Cfg::STAGE_BYTES + aoff;
      const uint32_t sb = smem_u + (uint32_t)s * Cfg::STAGE_BYTES + Cfg::A_BYTES;
#pragma unroll
      for (int kp = 0; kp < 2; ++kp) {
        double2 af[PL][MI];
#pragma unroll
        for (int pl = 0; pl < PL; ++pl)
#pragma unroll
          for (int i = 0; i < MI; ++i) af[pl][i] = lds128(sa + pl * (BM * 128) + i * 1024 + (kp ? la1 : la0));
#pragma unroll
        for (int j2 = 0; j2 < NP; ++j2) {
          const uint32_t bo = sb + j2 * 2048;
          const double2 q0 = lds128(bo + lbp[kp][0]);       // k even: columns 2 g, 2 g + 1
          const double2 q1 = lds128(bo + lbp[kp][1]);       // k odd
#pragma unroll
          for (int pl = 0; pl < PL; ++pl)
#pragma unroll
            for (int i = 0; i < MI; ++i) {
              dmma884(acc[pl][i][2 * j2][0], acc[pl][i][2 * j2][1], af[pl][i].x, q0.x);
              dmma884(acc[pl][i][2 * j2 + 1][0], acc[pl][i][2 * j2 + 1][1], af[pl][i].x, q0.y);
            }
#pragma unroll
          for (int pl = 0; pl < PL; ++pl)
#pragma unroll
            for (int i = 0; i < MI; ++i) {
              dmma884(acc[pl][i][2 * j2][0], acc[pl][i][2 * j2][1], af[pl][i].y, q1.x);
              dmma884(acc[pl][i][2 * j2 + 1][0], acc[pl][i][2 * j2 + 1][1], af[pl][i].y, q1.y);
            }
        }
#pragma unroll
        for (int j = 2 * NP; j < NI; ++j) {                  // unpaired blocks (an odd last one): 8-byte loads
          const uint32_t bo = sb + (j >> 1) * 2048;
          const double b0 = lds64(bo + (lb[kp][0] ^ ((j & 1) * 64)));
          const double b1 = lds64(bo + (lb[kp][1] ^ ((j & 1) * 64)));
#pragma unroll
          for (int pl = 0; pl < PL; ++pl)
#pragma unroll
            for (int i = 0; i < MI; ++i) dmma884(acc[pl][i][j][0], acc[pl][i][j][1], af[pl][i].x, b0);
#pragma unroll
          for (int pl = 0; pl < PL; ++pl)
#pragma unroll
            for (int i = 0; i < MI; ++i) dmma884(acc[pl][i][j][0], acc[pl][i][j][1], af[pl][i].y, b1);
        }
      }
    }

    if (sg.mode != 0) {
      constexpr int NACC = PL * MI * NI * 2;
      if (sg.mode == 1) {                      // first part: park the accumulators, tell the neighbour, go on
        double* dst = a.sk_part + (size_t)blockIdx.x * NACC * 256 + tid;
        int q = 0;
#pragma unroll
        for (int pl = 0; pl < PL; ++pl)
#pragma unroll
          for (int i = 0; i < MI; ++i)
#pragma unroll
            for (int j = 0; j < NI; ++j) { dst[(q++) * 256] = acc[pl][i][j][0]; dst[(q++) * 256] = acc[pl][i][j][1]; }
        __threadfence();
        named_bar_sync(1, 256);
        if (tid == 0) atomicExch(a.sk_flag + blockIdx.x, 1);
        continue;
      }
      // last part: wait for the neighbour's first part (written as the very first thing it did), add it
      if (tid == 0) {
        while (atomicAdd(a.sk_flag + blockIdx.x - 1, 0) == 0) {}
        atomicExch(a.sk_flag + blockIdx.x - 1, 0);      // ready for the next launch
        __threadfence();
      }
      named_bar_sync(1, 256);
      const double* src = a.sk_part + (size_t)(blockIdx.x - 1) * NACC * 256 + tid;
      int q = 0;
#pragma unroll
      for (int pl = 0; pl < PL; ++pl)
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
          for (int j = 0; j < NI; ++j) { acc[pl][i][j][0] += __ldcg(src + (q++) * 256); acc[pl][i][j][1] += __ldcg(src + (q++) * 256); }
    }
    double* C = a.C + (size_t)b * a.sC;
    double* C2 = a.C2 ? a.C2 + (size_t)b * a.sC : nullptr;
#pragma unroll
    for (int i = 0; i < MI; ++i) {
      const int r = mt * BM + 8 * (warp * MI + i) + p;
      if (r >= a.M) continue;
      auto put = [&](int n, double v0, double v1) {
        if (n >= a.N) return;
        const size_t off = (size_t)r * a.ldc + n;
        *reinterpret_cast<double2*>(C + off) = make_double2(v0, v1);
        if (C2) {
          if (a.mode == 1) {
            const double2 o = *reinterpret_cast<const double2*>(C2 + off);
            *reinterpret_cast<double2*>(C2 + off) = make_double2(o.x + v0, o.y + v1);
          } else {
            *reinterpret_cast<double2*>(C2 + off) = make_double2(v0, v1);
          }
        }
      };
#pragma unroll
      for (int j2 = 0; j2 < NP; ++j2) {
        // the lane holds columns 4 t .. 4 t + 3 of box j2: (even block c0, odd block c0, even block c1, odd block c1)
        const int n = (nt * NB16 + j2) * 16 + 4 * t;
        const int je = 2 * j2, jo = 2 * j2 + 1;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          double v0, v1;
          if constexpr (CPLX) {      // (re, im) columns: re = P_re - Q_im, im = P_im + Q_re
            v0 = a.alpha * (acc[0][i][je][h] - acc[PL - 1][i][jo][h]);
            v1 = a.alpha * (acc[0][i][jo][h] + acc[PL - 1][i][je][h]);
          } else {
            v0 = a.alpha * acc[0][i][je][h];
            v1 = a.alpha * acc[0][i][jo][h];
          }
          put(n + 2 * h, v0, v1);
        }
      }
#pragma unroll
      for (int j = 2 * NP; j < NI; ++j) {
        const int n = (nt * NB16 * 2 + j) * 8 + 2 * t;
        double v0, v1;
        if constexpr (CPLX) {
          v0 = a.alpha * (acc[0][i][j][0] - acc[PL - 1][i][j][1]);
          v1 = a.alpha * (acc[0][i][j][1] + acc[PL - 1][i][j][0]);
        } else {
          v0 = a.alpha * acc[0][i][j][0];
          v1 = a.alpha * acc[0][i][j][1];
        }
        put(n, v0, v1);
      }
    }
  }
}

template <int MI, int NI, bool CPLX>
int launch_kn(const TensorMap& tmA, const TensorMap& tmB, KnArgs a, const KnStreamK* sk, cudaStream_t st) {
  using Cfg = KnCfg<MI, NI, CPLX>;
  auto kern = gemm_ws_kn_kernel<MI, NI, CPLX>;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemCap);
  }
  int S = (kSmemCap - 1024 - 256) / Cfg::STAGE_BYTES;
  if (S > 8) S = 8;
  if (S < 2) return -1;
  a.stages = S;
  const size_t smem = (size_t)S * Cfg::STAGE_BYTES + 1024 + 256;
  const long nt = (long)a.mtiles * a.ntiles_n * a.batch;
  const int grid = nt < sm_count() ? (int)nt : sm_count();
  a.sk_w = 0; a.sk_part = nullptr; a.sk_flag = nullptr;
  if (sk && sk->part && sk->flag && nt > grid && nt % grid != 0) {
    // stream-K when the tile count leaves a partial last wave (c5 Taylor: 1216 tiles = 8.2 waves on 148 SMs)
    const int KT = (a.K + 15) / 16;
    const long w = (nt * KT + grid - 1) / grid;
    const size_t need = (size_t)grid * Cfg::PL * MI * NI * 2 * 256;
    // parking and fetching a tile's accumulators costs about 8 k iterations per CTA (c2, c3: no gain, measured)
    const long plain = ((nt + grid - 1) / grid) * KT;
    if (w >= KT && (sk->force || (double)(w + 8) < 0.99 * plain) && need <= sk->part_doubles && grid <= sk->flags) {
      a.sk_w = (int)w; a.sk_part = sk->part; a.sk_flag = sk->flag;
      // The kernel leaves every flag at 0 when it completes; a launch that was aborted (sticky error, device reset of
      // a peer context) may not have, and its stale 1 would let a consumer read accumulators that were never parked.
      // Clearing on the stream costs one memset node per stream-K launch (8 per step at c5, ~2 us each).
      cudaMemsetAsync(sk->flag, 0, (size_t)grid * sizeof(int), st);
    }
  }
  kern<<<grid, Cfg::THREADS, smem, st>>>(tmA, tmB, a);
  return 1;
}

template <bool CPLX>
int dispatch_kn(int MI, int NI, const TensorMap& tmA, const TensorMap& tmB, const KnArgs& a, const KnStreamK* sk,
                cudaStream_t st) {
#define KN_CASE(mi, ni) \
  if (MI == mi && NI == ni) return launch_kn<mi, ni, CPLX>(tmA, tmB, a, sk, st);
  KN_CASE(1, 2) KN_CASE(1, 4) KN_CASE(1, 6) KN_CASE(1, 8) KN_CASE(1, 10) KN_CASE(1, 11) KN_CASE(1, 12)
  KN_CASE(1, 13) KN_CASE(1, 14) KN_CASE(1, 16)
  KN_CASE(2, 2) KN_CASE(2, 4) KN_CASE(2, 6) KN_CASE(2, 8) KN_CASE(2, 10) KN_CASE(2, 11) KN_CASE(2, 12)
  if constexpr (!CPLX) {
    KN_CASE(2, 13) KN_CASE(2, 14) KN_CASE(2, 16)
  }
#undef KN_CASE
  return -1;
}

const int kNiAvail[] = {2, 4, 6, 8, 10, 11, 12, 13, 14, 16};

// ------------------------------------------------------------------------------------ NK
struct NkArgs {
  double* C;           // [split][M][ldc]
  long ldc, sCsplit;
  int M, N, K;
  int mtiles, ntiles_n, split, kchunk;   // kchunk: k extent per slice (multiple of 16)
  int stages;
};

constexpr int NK_MI = 8, NK_NI = 4, NK_BM = 128, NK_BN = 128;
constexpr int NK_STAGE = (NK_BM + NK_BN) * 128;

__global__ void __launch_bounds__(256 + kProdT, 1)
gemm_ws_nk_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB, const NkArgs a) {
  constexpr int NCW = 8, MI = NK_MI, NI = NK_NI;
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int S = a.stages;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)S * NK_STAGE);
  uint64_t* empty = full + S;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int per_s = a.mtiles * a.ntiles_n;
  const int ntiles = per_s * a.split;

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
    fence_barrier_init();
  }
  __syncthreads();

  if (warp >= NCW) {
    reg_dealloc<24>();
    if (warp == NCW && lane == 0) {
      prefetch_tensormap(&tmA);
      prefetch_tensormap(&tmB);
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int ks = tile / per_s, rem = tile % per_s;
        const int mt = rem / a.ntiles_n, nt = rem % a.ntiles_n;
        const int kbeg = ks * a.kchunk, kend = min(a.K, kbeg + a.kchunk);
        for (int k0 = kbeg; k0 < kend; k0 += 16, ++it) {
          const int s = it % S;
          mbar_wait(&empty[s], ((it / S) & 1) ^ 1);
          mbar_expect_tx(&full[s], NK_STAGE);
          unsigned char* sa = smem + (size_t)s * NK_STAGE;
          tma_load_2d(sa, &tmA, &full[s], k0, mt * NK_BM);
          tma_load_2d(sa + NK_BM * 128, &tmB, &full[s], k0, nt * NK_BN);
        }
      }
    }
    return;
  }

  reg_alloc<240>();
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp & 1, wn = warp >> 1;
  const int p = rperm(g);
  const uint32_t l0 = (uint32_t)(p * 128 + ((t ^ p) << 4));
  const uint32_t l1 = (uint32_t)(p * 128 + (((t ^ p) ^ 4) << 4));
  const uint32_t smem_u = smem_u32(smem);
  const uint32_t aoff = (uint32_t)(wm * MI) * 1024u;
  const uint32_t boff = (uint32_t)(NK_BM * 128) + (uint32_t)(wn * NI) * 1024u;

  uint32_t it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int ks = tile / per_s, rem = tile % per_s;
    const int mt = rem / a.ntiles_n, nt = rem % a.ntiles_n;
    const int kbeg = ks * a.kchunk, kend = min(a.K, kbeg + a.kchunk);

    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int k0 = kbeg; k0 < kend; k0 += 16, ++it) {
      const int s = it % S;
      mbar_wait(&full[s], (it / S) & 1);
      consumer_release_prev(empty, it, S, lane);
      const uint32_t sa = smem_u + (uint32_t)s * NK_STAGE + aoff;
      const uint32_t sb = smem_u + (uint32_t)s * NK_STAGE + boff;
#pragma unroll
      for (int kp = 0; kp < 2; ++kp) {
        const uint32_t lo = kp ? l1 : l0;
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

    double* C = a.C + (size_t)ks * a.sCsplit;
#pragma unroll
    for (int i = 0; i < MI; ++i) {
      const int r = mt * NK_BM + 8 * (wm * MI + i) + p;
      if (r >= a.M) continue;
#pragma unroll
      for (int j = 0; j < NI; ++j) {
        const int c = nt * NK_BN + 8 * (wn * NI + j) + t;   // accumulator columns map to t, t + 4
        if (c < a.N) C[(size_t)r * a.ldc + c] = acc[i][j][0];
        if (c + 4 < a.N) C[(size_t)r * a.ldc + c + 4] = acc[i][j][1];
      }
    }
  }
}

bool even(long v) { return (v & 1) == 0; }
bool al16(const void* p) { return ((uintptr_t)p & 15) == 0; }

}  // namespace

// KN batched GEMM.  A: [batch or 1][planes][M][lda] (k contiguous; plane stride sPlane),
// B: [batch][K][ldb] (n contiguous), C/C2: [batch][M][ldc].  Returns launches or -1 when the
// shapes cannot be served (caller falls back to the cp.async GEMM).
int run_gemm_ws_kn(const double* A, long lda, long sPlane, long sA, bool cplx, const double* B, long ldb, long sB,
                   double* C, double* C2, long ldc, long sC, int M, int N, int K, int batch, double alpha,
                   int mode, cudaStream_t st, const KnStreamK* sk) {
  if (!(even(lda) && even(sPlane) && even(sA) && even(ldb) && even(sB) && even(ldc) && even(sC) && even(N)))
    return -1;
  if (!(al16(A) && al16(B) && al16(C) && (C2 == nullptr || al16(C2)))) return -1;
  const int blocks = (N + 7) / 8;
  const int ntn = (blocks + 15) / 16;
  const int want = (blocks + ntn - 1) / ntn;
  int NI = 16;
  for (int c : kNiAvail)
    if (c >= want && (ntn == 1 || c % 2 == 0)) { NI = c; break; }   // several n tiles: whole 16-column boxes
  // rows per tile: 64 (MI = 1) or 128 (MI = 2), whichever needs less time on the SM grid
  const int nsm = sm_count();
  int MI = 1;
  {
    const long t1 = (long)((M + 63) / 64) * ntn * batch, t2 = (long)((M + 127) / 128) * ntn * batch;
    const long c1 = (t1 + nsm - 1) / nsm, c2 = 2 * ((t2 + nsm - 1) / nsm);
    const bool mi2_ok = cplx ? (NI <= 12) : true;
    if (mi2_ok && c2 <= c1) MI = 2;
  }
  TensorMap tmA, tmB;
  {
    const int planes = cplx ? 2 : 1;
    const uint64_t dims[4] = {(uint64_t)K, (uint64_t)M, (uint64_t)planes, (uint64_t)(sA == 0 ? 1 : batch)};
    const uint64_t sp = (uint64_t)(planes > 1 ? sPlane : (long)lda * M) * 8;
    const uint64_t sb_ = (uint64_t)(sA == 0 ? (long)lda * M * planes : sA) * 8;
    const uint64_t str[3] = {(uint64_t)lda * 8, sp, sb_};
    const uint32_t box[4] = {16, (uint32_t)(64 * MI), (uint32_t)planes, 1};
    if (make_tensor_map_f64(&tmA, A, 4, dims, str, box) != 0) return -1;
  }
  {
    const uint64_t dims[3] = {(uint64_t)N, (uint64_t)K, (uint64_t)batch};
    const uint64_t str[2] = {(uint64_t)ldb * 8, (uint64_t)(batch > 1 ? sB : (long)ldb * K) * 8};
    const uint32_t box[3] = {16, 16, 1};
    if (make_tensor_map_f64(&tmB, B, 3, dims, str, box) != 0) return -1;
  }
  KnArgs a;
  a.C = C; a.C2 = C2; a.ldc = ldc; a.sC = sC; a.alpha = alpha; a.mode = mode;
  a.M = M; a.N = N; a.K = K; a.batch = batch;
  a.mtiles = (M + 64 * MI - 1) / (64 * MI); a.ntiles_n = ntn;
  a.a_shared = sA == 0; a.stages = 0; a.nb16 = (NI + 1) / 2;
  return cplx ? dispatch_kn<true>(MI, NI, tmA, tmB, a, sk, st) : dispatch_kn<false>(MI, NI, tmA, tmB, a, sk, st);
}

// split-K choice for the NK GEMM: the slice count whose tile count fills the SM grid best
int gemm_ws_nk_split(int M, int N, int K, int max_split) {
  const int nsm = sm_count();
  const long base = (long)((M + NK_BM - 1) / NK_BM) * ((N + NK_BN - 1) / NK_BN);
  int best = 1;
  double best_cost = 1e300;
  for (int s = 1; s <= max_split; ++s) {
    const int kchunk = ((K + s - 1) / s + 15) / 16 * 16;
    if ((long)kchunk * (s - 1) >= K && s > 1) continue;   // empty last slice
    const long tiles = base * s;
    const double cost = (double)((tiles + nsm - 1) / nsm) * (kchunk + 64);   // + pipeline fill per tile
    if (cost < best_cost) { best_cost = cost; best = s; }
  }
  return best;
}

int run_gemm_ws_nk(const double* A, long lda, const double* B, long ldb, double* C, long ldc, long sCsplit,
                   int M, int N, int K, int split, cudaStream_t st) {
  if (!(even(lda) && even(ldb) && al16(A) && al16(B))) return -1;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(gemm_ws_nk_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemCap);
  }
  TensorMap tmA, tmB;
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)M};
    const uint64_t str[1] = {(uint64_t)lda * 8};
    const uint32_t box[2] = {16, NK_BM};
    if (make_tensor_map_f64(&tmA, A, 2, dims, str, box) != 0) return -1;
  }
  {
    const uint64_t dims[2] = {(uint64_t)K, (uint64_t)N};
    const uint64_t str[1] = {(uint64_t)ldb * 8};
    const uint32_t box[2] = {16, NK_BN};
    if (make_tensor_map_f64(&tmB, B, 2, dims, str, box) != 0) return -1;
  }
  NkArgs a;
  a.C = C; a.ldc = ldc; a.sCsplit = sCsplit; a.M = M; a.N = N; a.K = K;
  a.mtiles = (M + NK_BM - 1) / NK_BM; a.ntiles_n = (N + NK_BN - 1) / NK_BN;
  a.split = split < 1 ? 1 : split;
  a.kchunk = ((K + a.split - 1) / a.split + 15) / 16 * 16;
  a.stages = 6;
  const size_t smem = (size_t)a.stages * NK_STAGE + 1024 + 256;
  const long nt = (long)a.mtiles * a.ntiles_n * a.split;
  const int grid = nt < sm_count() ? (int)nt : sm_count();
  gemm_ws_nk_kernel<<<grid, 256 + kProdT, smem, st>>>(tmA, tmB, a);
  return 1;
}

}  // namespace afq
