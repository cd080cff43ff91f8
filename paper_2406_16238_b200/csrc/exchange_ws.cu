// exchange_ws.cu - exchange contraction of the local energy (Eq. 11,
// PAPER.md:94; D7), warp-specialised TMA version:
//     T^g_w = Lrot^g [ns x M] * Theta_w [M x ns],   expart += tr(T T),   X_g = tr(T)
//
// One persistent CTA per SM, three roles:
//   * producer warp: feeds a ring of shared-memory stages with TMA (cp.async.bulk.tensor,
//     SWIZZLE_128B, mbarrier full/empty pairs);
//   * 8 or 12 consumer warps: 16-byte fragment loads and DMMA, nothing else.  A tile is G whole
//     Cholesky vectors (rows (g, i), UNPADDED out of Lrot[n_chol][Nt][M] by a 3-D box) times Wn
//     whole walkers (columns (w, plane, j) out of ThT[nw][2][Nt][M] by a 4-D box).  The tile's 8 x 8
//     blocks are dealt to the warps as RECTANGLES of unequal size (XwsArgs::rect): the block counts
//     19 x 13 of N_occ = 50 do not factor over a warp grid, so the plan balances the four
//     sub-partitions' DMMA load instead of padding every warp to the largest rectangle;
//   * 3 epilogue warps (the rest of the producer's warpgroup): after the K = M loop the consumers
//     only DUMP their accumulators into a shared-memory staging buffer (one pass = Gp vectors x Wp
//     walkers, two buffers when a tile needs several passes) and go on with the next tile; the
//     epilogue warps form tr(T T) and tr(T) from the staging buffer while the DMMA pipe is busy
//     with the next main loop.  T never reaches HBM.
// Pair mode (complex Cholesky vectors / complex trial: Lrot = Lr + i Li as two planes): the tile's rows are
// [plane][g][i], the four real products share the Theta fragments and the epilogue warps put
// T = (Lr Th_r - Li Th_i) + i (Lr Th_i + Li Th_r) together: one run instead of three.
#include <algorithm>
#include <map>

#include "internal.h"
#include "tma.cuh"

namespace afq {

namespace {

constexpr int kProducerThreads = 128;     // one warpgroup (setmaxnreg is warpgroup-wide)
// epilogue warps: 3 (warps 1..3 of the producer's warpgroup) or 7 (a second warpgroup of them; 8 consumer warps only)
constexpr int kSmemMax = 232448;          // 227 KB opt-in limit per CTA
constexpr int kMaxTasks = 512;            // (gamma, walker, row pair) lane tasks per tile: 16 KB of partial sums
constexpr int kMaxWarps = 12;

struct XwsArgs {
  double* expart;      // [ngroups][nw] complex
  double* X;           // [n_chol][nw] complex
  int M, ns, off, n_chol, nw;
  int G, Wn;           // gammas / walkers per tile
  int Gp, Wp;          // gammas / walkers per epilogue pass
  int ldt;             // staging row stride (doubles)
  int stages, nbuf;
  int rowsA, rowsB;    // rows TMA writes per stage; the stage holds round-up-to-8 of each
  int ntile_w, ntiles;
  int accumulate;
  int pair;            // 1: A rows are [2 planes][G][ns]
  unsigned rect[kMaxWarps];   // r0 | mi << 8 | c0 << 16 | ni << 24, in 8 x 8 blocks
};

template <int NCW, int MI, int NI, int EW>
struct XwsCfg {
  static constexpr int NCT = NCW * 32;
  static constexpr int OTHER = (EW + 1) * 32;           // producer warp + epilogue warps
  static constexpr int THREADS = NCT + OTHER;
  static constexpr int EPT = EW * 32;
  // register file: THREADS * R0 at launch (R0 from __launch_bounds__), then PREGS for the producer's
  // warpgroup and CREGS for the consumers
  static constexpr int R0 = (65536 / THREADS) / 8 * 8;
  static constexpr int PREGS = NCW == 12 ? 40 : 56;
  static constexpr int CREGS_ = ((THREADS * R0 - OTHER * PREGS) / NCT) / 8 * 8;
  static constexpr int CREGS = CREGS_ > 232 ? 232 : CREGS_;
};


// K = M loop of one tile for a warp rectangle of MU x NU blocks known at compile time (no predicates in the DMMA
// stream); GENERIC: rectangle sizes from registers (small or odd problems), predicated.
// Ring state of a consumer: soff = byte offset of the current stage, sbar = 8 * stage index, ph = its parity,
// prev = 8 * index of the stage to release (lagged release, tma.cuh) or -1.
struct Ring { uint32_t soff, sbar, ph; int prev; };

template <int MI, int NI, int MU, int NU, bool GENERIC>
__device__ __forceinline__ void xws_kloop(double (&acc)[MI][NI][2], uint32_t full_u32, uint32_t empty_u32, int KT,
                                          uint32_t ring_bytes, uint32_t stage_bytes, Ring& r, uint32_t a0, uint32_t b0,
                                          int lane, int mi, int ni) {
  for (int kt = 0; kt < KT; ++kt) {
    mbar_wait_u32(full_u32 + r.sbar, r.ph);
    if (r.prev >= 0 && lane == 0) mbar_arrive_u32(empty_u32 + r.prev);
    r.prev = (int)r.sbar;
    const uint32_t sa = a0 + r.soff, sb = b0 + r.soff;
    r.soff += stage_bytes; r.sbar += 8;
    if (r.soff == ring_bytes) { r.soff = 0; r.sbar = 0; r.ph ^= 1; }
#pragma unroll
    for (int kp = 0; kp < 2; ++kp) {
      const uint32_t x = kp ? 64u : 0u;       // the second k pair of a row sits 64 bytes further, modulo the swizzle
      double2 af[MU];
#pragma unroll
      for (int i = 0; i < MU; ++i)
        if (!GENERIC || i < mi) af[i] = lds128((sa + i * 1024) ^ x);
#pragma unroll
      for (int j = 0; j < NU; ++j) {
        if (!GENERIC || j < ni) {
          const double2 bf = lds128((sb + j * 1024) ^ x);
#pragma unroll
          for (int i = 0; i < MU; ++i)
            if (!GENERIC || i < mi) dmma884(acc[i][j][0], acc[i][j][1], af[i].x, bf.x);
#pragma unroll
          for (int i = 0; i < MU; ++i)
            if (!GENERIC || i < mi) dmma884(acc[i][j][0], acc[i][j][1], af[i].y, bf.y);
        }
      }
    }
  }
}

template <int NCW, int MI, int NI, int EW>
__global__ void __launch_bounds__(XwsCfg<NCW, MI, NI, EW>::THREADS, 1)
exchange_ws_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB,
                   const __grid_constant__ XwsArgs a) {
  using Cfg = XwsCfg<NCW, MI, NI, EW>;
  constexpr int NCT = Cfg::NCT, kEpiThreads = Cfg::EPT, kEpiWarps = EW;
  // SWIZZLE_128B tiles need a 1024-byte aligned base
  extern __shared__ __align__(1024) unsigned char smem[];
  if (smem_u32(smem) & 1023u) __trap();
  const int S = a.stages;
  const int TAr = (a.rowsA + 7) & ~7, TBr = (a.rowsB + 7) & ~7;
  const uint32_t stage_bytes = (uint32_t)(TAr + TBr) * 128u;
  const int ns = a.ns, ldt = a.ldt;
  const int planes = a.pair ? 2 : 1;
  const int srows = planes * a.Gp * ns;                 // staging rows per buffer
  const int nitems = a.G * a.Wn;
  unsigned char* tiles = smem;
  double* stg = reinterpret_cast<double*>(smem + (size_t)S * stage_bytes);
  double* part = stg + (size_t)a.nbuf * srows * ldt;                  // [nitems][row pairs][4]
  uint64_t* full = reinterpret_cast<uint64_t*>(part + (size_t)nitems * ((ns + 1) >> 1) * 4);
  uint64_t* empty = full + S;
  uint64_t* sfull = empty + S;                                        // staging buffer written
  uint64_t* sempty = sfull + 2;                                       // staging buffer read

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KT = (a.M + 15) >> 4;
  const int npass_g = (a.G + a.Gp - 1) / a.Gp, npass_w = (a.Wn + a.Wp - 1) / a.Wp;

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
    for (int b = 0; b < 2; ++b) { mbar_init(&sfull[b], NCT); mbar_init(&sempty[b], kEpiThreads); }
    fence_barrier_init();
  }
  // rows of the A / B tiles that TMA never writes (round-up to 8 rows) must read as finite numbers
  {
    uint4* z = reinterpret_cast<uint4*>(tiles);
    const int n16 = (int)(S * stage_bytes / 16);
    for (int i = tid; i < n16; i += Cfg::THREADS) z[i] = make_uint4(0, 0, 0, 0);
  }
  fence_proxy_async();
  __syncthreads();

  if (warp >= NCW) {
    reg_dealloc<Cfg::PREGS>();
    if (warp == NCW) {
      // ---------------------------------------------------------------------- producer
      if (lane == 0) {
        prefetch_tensormap(&tmA);
        prefetch_tensormap(&tmB);
        const uint32_t bytes = (uint32_t)(a.rowsA + a.rowsB) * 128u;
        uint32_t it = 0;
        for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
          const int g0 = (tile / a.ntile_w) * a.G, w0 = (tile % a.ntile_w) * a.Wn;
          for (int kt = 0; kt < KT; ++kt, ++it) {
            const int s = it % S;
            const uint32_t ph = (it / S) & 1;
            mbar_wait(&empty[s], ph ^ 1);
            mbar_expect_tx(&full[s], bytes);
            unsigned char* sa = tiles + (size_t)s * stage_bytes;
            tma_load_4d(sa, &tmA, &full[s], kt * 16, a.off, g0, 0);
            tma_load_4d(sa + TAr * 128, &tmB, &full[s], kt * 16, a.off, 0, w0);
          }
        }
      }
      return;
    }
    // ------------------------------------------------------------------------ epilogue warps
    // One lane per (vector, walker, row pair): lane task (item, ii) forms the i < j part of
    //   tr(T T) = sum_i T_ii^2 + 2 sum_{i<j} T_ij T_ji
    // for the rows i = ii and i = ns - 1 - ii, which together hold ns - 1 pairs for every ii: all lanes run the same
    // trip count, no shuffles, and neighbouring lanes are ldt + 1 doubles apart in both operands (conflict free).
    const int et = tid - (NCW + 1) * 32, ew = warp - NCW - 1;
    const int h = (ns + 1) >> 1;                            // row pairs per item
    int hp = 1;
    while (hp < h) hp <<= 1;
    const uint32_t plane_off = (uint32_t)(a.Gp * ns * ldt * 8);   // second plane of the staging buffer (pair mode)
    const uint32_t ns8 = (uint32_t)ns * 8, ldt8 = (uint32_t)ldt * 8;
    const uint32_t stg_e = smem_u32(stg), buf_bytes_e = (uint32_t)(srows * ldt * 8), part_e = smem_u32(part);
    uint32_t e = 0;
    for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
      const int tg = tile / a.ntile_w;
      const int g0 = tg * a.G, w0 = (tile % a.ntile_w) * a.Wn;
      for (int pg = 0; pg < npass_g; ++pg)
        for (int pw = 0; pw < npass_w; ++pw, ++e) {
          const int gp0 = pg * a.Gp, wp0 = pw * a.Wp;
          const int Gpc = min(a.Gp, a.G - gp0), Wpc = min(a.Wp, a.Wn - wp0);
          const int buf = e % a.nbuf;
          mbar_wait(&sfull[buf], (e / a.nbuf) & 1);
          const uint32_t sb = stg_e + (uint32_t)buf * buf_bytes_e;
          const int ntask = Gpc * Wpc * h;
          for (int task = et; task < ntask; task += kEpiThreads) {
            const int item = task / h, ii = task - item * h;
            const int gl = item / Wpc, wl = item - gl * Wpc;
            const uint32_t p0 = sb + (uint32_t)((gl * ns * ldt + wl * 2 * ns) * 8);   // plane 0: [i][re j | im j]
            const int i2 = ns - 1 - ii, n1 = ns - 1 - ii;                             // n1 pairs in row ii, ii in row i2
            // byte addresses of T_ij (row walk, +8 per pair) and T_ji (column walk, +8 ldt per pair)
            uint32_t aij = p0 + (uint32_t)((ii * ldt + ii + 1) * 8), aji = p0 + (uint32_t)(((ii + 1) * ldt + ii) * 8);
            const int nk = (i2 == ii) ? n1 : ns - 1;        // odd ns: the middle row is its own partner
            // two pairs per trip on separate accumulators: an FP64 add or multiply of these warps queues behind the
            // consumers' DMMAs (same pipe), so the dependent chain is what takes the time
            double vr = 0.0, vi = 0.0, ur = 0.0, ui = 0.0;
            for (int k = 0; k < nk; k += 2) {
              if (k == n1) {                                // switch to row i2
                aij = p0 + (uint32_t)((i2 * ldt + i2 + 1) * 8);
                aji = p0 + (uint32_t)(((i2 + 1) * ldt + i2) * 8);
              }
              double ar = lds64(aij), ai = lds64(aij + ns8);
              double br = lds64(aji), bi = lds64(aji + ns8);
              if (a.pair) {
                ar -= lds64(aij + plane_off + ns8); ai += lds64(aij + plane_off);
                br -= lds64(aji + plane_off + ns8); bi += lds64(aji + plane_off);
              }
              aij += 8; aji += ldt8;
              vr += ar * br - ai * bi;
              vi += ar * bi + ai * br;
              if (k + 1 < nk) {
                if (k + 1 == n1) {
                  aij = p0 + (uint32_t)((i2 * ldt + i2 + 1) * 8);
                  aji = p0 + (uint32_t)(((i2 + 1) * ldt + i2) * 8);
                }
                double cr = lds64(aij), ci = lds64(aij + ns8);
                double dr = lds64(aji), di = lds64(aji + ns8);
                if (a.pair) {
                  cr -= lds64(aij + plane_off + ns8); ci += lds64(aij + plane_off);
                  dr -= lds64(aji + plane_off + ns8); di += lds64(aji + plane_off);
                }
                aij += 8; aji += ldt8;
                ur += cr * dr - ci * di;
                ui += cr * di + ci * dr;
              }
            }
            vr += ur; vi += ui;
            vr *= 2.0; vi *= 2.0;
            double xr = 0.0, xi = 0.0;
            for (int q = 0; q < (i2 == ii ? 1 : 2); ++q) {                    // the two diagonal elements
              const uint32_t o = p0 + (uint32_t)((q ? i2 : ii) * (ldt + 1) * 8);
              double ar = lds64(o), ai = lds64(o + ns8);
              if (a.pair) { ar -= lds64(o + plane_off + ns8); ai += lds64(o + plane_off); }
              vr += ar * ar - ai * ai;
              vi += 2.0 * ar * ai;
              xr += ar; xi += ai;
            }
            const uint32_t c = part_e + (uint32_t)((((gp0 + gl) * a.Wn + wp0 + wl) * h + ii) * 32);
            sts64(c, vr); sts64(c + 8, vi); sts64(c + 16, xr); sts64(c + 24, xi);
          }
          // the stores above depend on every value read from the buffer
          mbar_arrive(&sempty[buf]);
        }
      // fixed-order sums over the tile's vectors and row pairs, between two barriers of the epilogue warps (the
      // second one frees the table for the next tile)
      named_bar_sync(2, kEpiThreads);
      // one warp per walker of the tile; a group of hp lanes (hp = h rounded up to a power of two) sums the row
      // pairs of one vector, 32 / hp vectors at a time, in a fixed order
      for (int wl = ew; wl < a.Wn; wl += kEpiWarps) {
        const int w = w0 + wl;
        const int sub = lane / hp, k = lane & (hp - 1);
        double sr = 0.0, si = 0.0;
        for (int gl0 = 0; gl0 < a.G; gl0 += 32 / hp) {
          const int gl = gl0 + sub;
          const bool valid = gl < a.G && k < h;
          double vr = 0.0, vi = 0.0, xr = 0.0, xi = 0.0;
          if (valid) {
            const uint32_t c = part_e + (uint32_t)(((gl * a.Wn + wl) * h + k) * 32);
            vr = lds64(c); vi = lds64(c + 8); xr = lds64(c + 16); xi = lds64(c + 24);
          }
          for (int o = hp >> 1; o > 0; o >>= 1) {
            vr += __shfl_xor_sync(0xffffffffu, vr, o);
            vi += __shfl_xor_sync(0xffffffffu, vi, o);
            xr += __shfl_xor_sync(0xffffffffu, xr, o);
            xi += __shfl_xor_sync(0xffffffffu, xi, o);
          }
          sr += vr; si += vi;
          if (k == 0 && gl < a.G && w < a.nw && g0 + gl < a.n_chol) {
            double* xo = a.X + ((size_t)(g0 + gl) * a.nw + w) * 2;
            if (a.accumulate) { xo[0] += xr; xo[1] += xi; } else { xo[0] = xr; xo[1] = xi; }
          }
        }
        for (int o = 16; o >= hp; o >>= 1) {
          sr += __shfl_xor_sync(0xffffffffu, sr, o);
          si += __shfl_xor_sync(0xffffffffu, si, o);
        }
        if (lane == 0 && w < a.nw) {
          double* eo = a.expart + ((size_t)tg * a.nw + w) * 2;
          eo[0] = sr; eo[1] = si;
        }
      }
      named_bar_sync(2, kEpiThreads);
    }
    return;
  }

  // -------------------------------------------------------------------- consumer warps
  reg_alloc<Cfg::CREGS>();
  const int g = lane >> 2, t = lane & 3;
  const int p = rperm(g);
  const unsigned rc = a.rect[warp];
  const int r0 = rc & 255, mi = (rc >> 8) & 255, c0 = (rc >> 16) & 255, ni = rc >> 24;
  const uint32_t lane0 = (uint32_t)(p * 128 + ((t ^ p) << 4));
  const uint32_t tiles_u32 = smem_u32(tiles);
  const uint32_t a0 = tiles_u32 + (uint32_t)r0 * 1024u + lane0;
  const uint32_t b0 = tiles_u32 + (uint32_t)(TAr * 128) + (uint32_t)c0 * 1024u + lane0;
  const uint32_t full_u32 = smem_u32(full), empty_u32 = smem_u32(empty);
  const uint32_t ring_bytes = (uint32_t)S * stage_bytes;
  const uint32_t stg_u32 = smem_u32(stg), buf_bytes = (uint32_t)(srows * ldt * 8);
  const uint32_t sfull_u32 = smem_u32(sfull), sempty_u32 = smem_u32(sempty);
  const int Gns = a.G * ns, rows_all = planes * Gns;

  // the rectangle is one of (MI | MI - 1) x (NI | NI - 1) for every plan of a production shape
  const int variant = (mi == MI && ni == NI) ? 0 : (mi == MI - 1 && ni == NI) ? 1 : (mi == MI && ni == NI - 1) ? 2
                      : (mi == MI - 1 && ni == NI - 1) ? 3 : 4;
  uint32_t d = 0;
  Ring ring = {0u, 0u, 0u, -1};
  for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    switch (variant) {
      case 0: xws_kloop<MI, NI, MI, NI, false>(acc, full_u32, empty_u32, KT, ring_bytes, stage_bytes, ring, a0, b0, lane, mi, ni); break;
      case 1: xws_kloop<MI, NI, MI - 1, NI, false>(acc, full_u32, empty_u32, KT, ring_bytes, stage_bytes, ring, a0, b0, lane, mi, ni); break;
      case 2: xws_kloop<MI, NI, MI, NI - 1, false>(acc, full_u32, empty_u32, KT, ring_bytes, stage_bytes, ring, a0, b0, lane, mi, ni); break;
      case 3: xws_kloop<MI, NI, MI - 1, NI - 1, false>(acc, full_u32, empty_u32, KT, ring_bytes, stage_bytes, ring, a0, b0, lane, mi, ni); break;
      default: xws_kloop<MI, NI, MI, NI, true>(acc, full_u32, empty_u32, KT, ring_bytes, stage_bytes, ring, a0, b0, lane, mi, ni); break;
    }

    // ---------------------------------------------------------------- dump, one pass at a time
    // (32-bit shared addresses, one predicate bit per store: this code runs on the DMMA warps' time)
    for (int pg = 0; pg < npass_g; ++pg)
      for (int pw = 0; pw < npass_w; ++pw, ++d) {
        const int gp0 = pg * a.Gp, wp0 = pw * a.Wp;
        const int rlo = gp0 * ns, rhi = min(a.Gp, a.G - gp0) * ns + rlo;
        const int clo = wp0 * 2 * ns, chi = min(a.Wp, a.Wn - wp0) * 2 * ns + clo;
        unsigned m0 = 0, m1 = 0;               // bit j: column 8 (c0 + j) + t (+ 4) belongs to this pass
#pragma unroll
        for (int j = 0; j < NI; ++j) {
          const int c = 8 * (c0 + j) + t;
          m0 |= (j < ni && c >= clo && c < chi) ? 1u << j : 0u;
          m1 |= (j < ni && c + 4 >= clo && c + 4 < chi) ? 1u << j : 0u;
        }
        uint32_t buf_u32 = stg_u32;
        uint32_t bar_off = 0;
        if (a.nbuf == 2 && (d & 1)) { buf_u32 += buf_bytes; bar_off = 8; }
        mbar_wait_u32(sempty_u32 + bar_off, (a.nbuf == 2 ? (d >> 1) & 1 : d & 1) ^ 1);
#pragma unroll
        for (int i = 0; i < MI; ++i) {
          const int r = 8 * (r0 + i) + p;
          const int pl = r >= Gns ? 1 : 0;
          const int rr = r - pl * Gns;
          if (i < mi && r < rows_all && rr >= rlo && rr < rhi) {
            const uint32_t row = buf_u32 + (uint32_t)(((pl * a.Gp * ns + rr - rlo) * ldt + 8 * c0 + t - clo) * 8);
#pragma unroll
            for (int j = 0; j < NI; ++j) {
              if (m0 >> j & 1) sts64(row + j * 64, acc[i][j][0]);
              if (m1 >> j & 1) sts64(row + j * 64 + 32, acc[i][j][1]);
            }
          }
        }
        mbar_arrive_u32(sfull_u32 + bar_off);
      }
  }
}

struct Plan {
  int inst = -1;      // index into kInst
  int WM = 0;         // warp grid rows
  int ncw = 0, G = 0, Wn = 0, Gp = 0, Wp = 0, ldt = 0, stages = 0, nbuf = 1;
  int rowsA = 0, rowsB = 0;
  unsigned rect[kMaxWarps] = {};
  size_t smem = 0;
  double eff = 0.0;     // useful share of the issued DMMA blocks
  double score = 0.0;   // useful flops per modelled cycle
  double bpf = 1e30;    // operand bytes per useful flop (shared-memory fill traffic out of L2)
};

struct Inst { int NCW, MI, NI, EW; };
constexpr Inst kInst[] = {{8, 5, 7, 3}, {8, 7, 5, 3}, {8, 6, 6, 3}, {12, 4, 7, 3}, {12, 7, 4, 3}, {12, 5, 5, 3},
                          {12, 5, 4, 3}, {12, 4, 5, 3}, {8, 5, 7, 7}, {8, 7, 5, 7}, {8, 6, 6, 7}};
constexpr int kNumInst = sizeof(kInst) / sizeof(kInst[0]);

// staging row stride: stride mod 16 in {6, 10} spreads the accumulator dump (8 rows x 4 columns per store
// instruction) over all banks exactly twice and keeps the column reads of the epilogue warps 4-way at worst
int staging_stride(int cols) {
  int l = cols;
  while (l % 16 != 6 && l % 16 != 10) ++l;
  return l;
}

// Deal nbr x nbc blocks to a WM x WN grid of near-equal rectangles and the rectangles to warp ids so that the
// four sub-partitions (warp id mod 4) carry about the same number of DMMA blocks.  Returns the largest
// sub-partition load; fails (-1) if a rectangle exceeds MI x NI.
int deal_rectangles(int nbr, int nbc, int WM, int WN, int MI, int NI, unsigned* rect) {
  const int ncw = WM * WN;
  struct R { int r0, mi, c0, ni; };
  std::vector<R> rs;
  for (int wn = 0; wn < WN; ++wn)
    for (int wm = 0; wm < WM; ++wm) {
      R r;
      r.mi = nbr / WM + (wm < nbr % WM ? 1 : 0);
      r.r0 = wm * (nbr / WM) + std::min(wm, nbr % WM);
      r.ni = nbc / WN + (wn < nbc % WN ? 1 : 0);
      r.c0 = wn * (nbc / WN) + std::min(wn, nbc % WN);
      if (r.mi > MI || r.ni > NI) return -1;
      rs.push_back(r);
    }
  std::stable_sort(rs.begin(), rs.end(), [](const R& x, const R& y) { return x.mi * x.ni > y.mi * y.ni; });
  int load[4] = {0, 0, 0, 0}, cnt[4] = {0, 0, 0, 0};
  for (const R& r : rs) {           // largest first, to the lightest sub-partition that still has a warp slot
    int best = -1;
    for (int s = 0; s < 4; ++s)
      if (cnt[s] < ncw / 4 && (best < 0 || load[s] < load[best])) best = s;
    const int warp = best + 4 * cnt[best];
    rect[warp] = (unsigned)r.r0 | ((unsigned)r.mi << 8) | ((unsigned)r.c0 << 16) | ((unsigned)r.ni << 24);
    load[best] += r.mi * r.ni;
    cnt[best] += 1;
  }
  return std::max(std::max(load[0], load[1]), std::max(load[2], load[3]));
}

// shared memory beside the ring and the staging buffers: partial-sum table, barriers, alignment slack
size_t fixed_smem(int ns, int nitems) {
  return (size_t)nitems * ((ns + 1) / 2) * 32 + 16 * 8 + 64;
}

// Cycle model of one tile on one SM (measured on B200, profiles/r2_exchange.md): the main loop runs at 64 clocks per
// DMMA block and k-tile on the busiest sub-partition unless the fill of the stage out of L2 is slower (c5 sustains
// 21 B/clk/SM at 92 % of the DMMA peak; 30 taken as the ceiling); every pass costs the DMMA warps a dump; the
// epilogue warps need about 150 + 30 (ns - 1) clocks per round of 96 lane tasks and stall the consumers when a tile
// has more passes than staging buffers, or when they cannot keep up with a short K loop.
// clocks per pair of an epilogue lane while the DMMA pipe is saturated (its FP64 operations queue behind the DMMAs);
// c2: 224 lane tasks of 15 pairs on 96 lanes held a 25 k-clock main loop up at 37 k clocks per tile
constexpr double kEpiTrip = 150.0;

std::vector<Plan> enumerate_plans(int ns, bool pair, int KT) {
  const int planes = pair ? 2 : 1;
  const int h = (ns + 1) / 2;
  auto t_epi = [&](int items, int ew) { return 300.0 + ((items * h + 32 * ew - 1) / (32 * ew)) * kEpiTrip * (ns - 1); };
  std::vector<Plan> cands;
  for (int c = 0; c < kNumInst; ++c) {
    const Inst& I = kInst[c];
    for (int WM = 1; WM <= I.NCW; ++WM) {
      if (I.NCW % WM) continue;
      const int WN = I.NCW / WM;
      const int Gmax = std::min(255, 8 * WM * I.MI / (planes * ns)), Wmax = std::min(255, 8 * WN * I.NI / (2 * ns));
      for (int G = 1; G <= Gmax; ++G)
        for (int Wn = 1; Wn <= Wmax; ++Wn) {
          if (G * Wn * ((ns + 1) / 2) > kMaxTasks) continue;
          Plan p;
          p.inst = c; p.ncw = I.NCW; p.G = G; p.Wn = Wn; p.WM = WM;
          p.rowsA = planes * G * ns; p.rowsB = Wn * 2 * ns;
          const int nbr = (p.rowsA + 7) / 8, nbc = (p.rowsB + 7) / 8;
          const int maxload = deal_rectangles(nbr, nbc, WM, WN, I.MI, I.NI, p.rect);
          if (maxload < 0) continue;
          const double useful = (double)p.rowsA * p.rowsB;
          const double bytes = (double)(p.rowsA + p.rowsB) * 128.0;
          p.eff = useful / (256.0 * maxload);
          p.bpf = bytes / useful;
          const size_t stage = (size_t)(8 * nbr + 8 * nbc) * 128;
          const size_t fixed = fixed_smem(ns, G * Wn);
          for (int S = 3; S >= 2; --S) {
            if (S * stage + fixed >= (size_t)kSmemMax) continue;
            const size_t left = (size_t)kSmemMax - fixed - S * stage;
            // as few passes as fit beside the ring; two buffers as soon as there is more than one pass
            int bp = 1 << 30;
            Plan q = p;
            for (int Gp = G; Gp >= 1; --Gp)
              for (int Wp = Wn; Wp >= 1; --Wp) {
                const int passes = ((G + Gp - 1) / Gp) * ((Wn + Wp - 1) / Wp);
                const int nbuf = passes > 1 ? 2 : 1;
                const int ldt = staging_stride(Wp * 2 * ns);
                const size_t need = (size_t)nbuf * planes * Gp * ns * ldt * 8;
                if (need > left || passes >= bp) continue;
                bp = passes;
                q.Gp = Gp; q.Wp = Wp; q.ldt = ldt; q.nbuf = nbuf; q.stages = S;
                q.smem = S * stage + need + fixed;
              }
            if (bp == 1 << 30) continue;
            // 12 consumer warps run on 152 registers (a few spills in the k loop), 8 on 224: measured 2 % apart
            double main = KT * std::max(64.0 * maxload, bytes / 30.0) * (S == 2 ? 1.03 : 1.0) * (I.NCW == 12 ? 1.02 : 1.0);
            const double dump = bp * (I.NCW / 4) * (6.0 * I.MI * I.NI + 150.0);
            const double epi_pass = t_epi(q.Gp * q.Wp, I.EW);
            const double stall = std::max(0, bp - q.nbuf) * epi_pass;
            const double epi_all = bp * epi_pass + 300.0;
            // rectangles other than (MI | MI - 1) x (NI | NI - 1) run the predicated k loop
            bool generic = false;
            for (int w = 0; w < I.NCW; ++w) {
              const int mi = (q.rect[w] >> 8) & 255, ni = q.rect[w] >> 24;
              generic = generic || mi < I.MI - 1 || ni < I.NI - 1;
            }
            if (generic) main *= 1.15;
            // measured: seven epilogue warps pay off while the K loop is short (c2, c3), cost 5 % at c5 (200
            // instead of 224 consumer registers)
            if (I.EW == 7) main *= KT <= 32 ? 0.98 : 1.05;
            const double t_tile = std::max(main + 800.0 + dump + stall, epi_all);
            q.score = useful * KT / t_tile;
            cands.push_back(q);
          }
        }
    }
  }
  return cands;
}

// Plans found by sweeping every candidate on a B200 (afqmc_exchange_plan_pin; profiles/r2_exchange.md), for the
// shapes of BASELINE.json's configs; any other shape takes the model's choice.
struct Tuned { int ns, KT, pair, ncw, mi, ni, wm, G, Wn, ew; };
constexpr Tuned kTuned[] = {
    {16, 7, 0, 8, 5, 7, 4, 9, 3, 7},    // c2 alpha block: 144 x 96 tiles, 7 epilogue warps (short K loop)
    {14, 7, 0, 8, 7, 5, 1, 4, 8, 7},    // c2 beta block: 56 x 224 tiles
    {50, 19, 0, 8, 5, 7, 4, 3, 1, 7},   // c3
    {40, 44, 0, 12, 5, 4, 4, 4, 1, 3},  // c4: 160 x 80 tiles in one pass
    {42, 75, 0, 12, 4, 7, 4, 3, 2, 3},  // c5: 126 x 168 tiles, three passes through two buffers
    {50, 19, 1, 12, 4, 5, 4, 1, 1, 3},  // complex c3 shapes
};

Plan make_plan(int ns, bool pair, int KT) {
  const std::vector<Plan> cands = enumerate_plans(ns, pair, KT);
  for (const Tuned& t : kTuned) {
    if (t.ns != ns || t.KT != KT || (t.pair != 0) != pair) continue;
    const Plan* pick = nullptr;
    for (const Plan& p : cands)
      if (p.ncw == t.ncw && kInst[p.inst].MI == t.mi && kInst[p.inst].NI == t.ni && kInst[p.inst].EW == t.ew &&
          p.WM == t.wm && p.G == t.G && p.Wn == t.Wn && (!pick || p.stages > pick->stages))
        pick = &p;
    if (pick) return *pick;
  }
  // the most useful work per cycle; among plans within 1 % of it the one that moves the fewest bytes per flop (the
  // squarest tile), then the deeper ring
  Plan best;
  double top = 0.0;
  for (const Plan& p : cands) top = std::max(top, p.score);
  for (const Plan& p : cands) {
    if (p.score < 0.99 * top) continue;
    if (best.inst < 0 || p.bpf < best.bpf - 1e-12 || (p.bpf < best.bpf + 1e-12 && p.stages > best.stages)) best = p;
  }
  return best;
}

template <int NCW, int MI, int NI, int EW>
int launch_xws(const ExArgs& e, const Plan& p, cudaStream_t st) {
  using Cfg = XwsCfg<NCW, MI, NI, EW>;
  auto kern = exchange_ws_kernel<NCW, MI, NI, EW>;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  }
  const int nsm = sm_count_current();
  const bool pair = e.plane_stride != 0;
  TensorMap tmA, tmB;
  {
    const uint64_t dims[4] = {(uint64_t)e.M, (uint64_t)e.Nt, (uint64_t)e.n_chol, (uint64_t)(pair ? 2 : 1)};
    const uint64_t str[3] = {(uint64_t)e.M * 8, (uint64_t)e.Nt * e.M * 8,
                             pair ? (uint64_t)e.plane_stride * 8 : (uint64_t)e.n_chol * e.Nt * e.M * 8};
    const uint32_t box[4] = {16, (uint32_t)e.ns, (uint32_t)p.G, (uint32_t)(pair ? 2 : 1)};
    if (make_tensor_map_f64(&tmA, e.Lrot, 4, dims, str, box) != 0) return -1;
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
  a.G = p.G; a.Wn = p.Wn; a.Gp = p.Gp; a.Wp = p.Wp; a.ldt = p.ldt; a.stages = p.stages; a.nbuf = p.nbuf;
  a.rowsA = p.rowsA; a.rowsB = p.rowsB;
  a.ntile_w = (e.nw + p.Wn - 1) / p.Wn;
  a.ntiles = a.ntile_w * ((e.n_chol + p.G - 1) / p.G);
  a.accumulate = e.accumulate;
  a.pair = pair ? 1 : 0;
  for (int w = 0; w < kMaxWarps; ++w) a.rect[w] = p.rect[w];
  const int grid = a.ntiles < nsm ? a.ntiles : nsm;
  kern<<<grid, Cfg::THREADS, p.smem, st>>>(tmA, tmB, a);
  return 1;
}

std::mutex g_plan_mu;
std::map<long, Plan> g_plan_cache;

// By value, copied under the lock: a pin from another host thread may overwrite the entry at any time, and a launch
// must see one plan from its first field to its last.
Plan cached_plan(int ns, bool pair, int M) {
  const int KT = (M + 15) / 16;
  const long key = ((long)KT << 8 | ns) << 1 | (pair ? 1 : 0);
  std::lock_guard<std::mutex> lk(g_plan_mu);
  auto it = g_plan_cache.find(key);
  if (it == g_plan_cache.end()) it = g_plan_cache.emplace(key, make_plan(ns, pair, KT)).first;
  return it->second;
}

}  // namespace

bool exchange_ws_usable(int M, const void* Lrot, const void* ThT) {
  return (M % 2 == 0) && (((uintptr_t)Lrot | (uintptr_t)ThT) & 15) == 0;
}

int exchange_ws_group_size(int ns, int M, bool pair) { return cached_plan(ns, pair, M).G; }

double exchange_ws_efficiency(int ns, int M, bool pair) { return cached_plan(ns, pair, M).eff; }

// Tuning hook: replace the plan of (ns, M, pair) by the candidate with this warp count, rectangle bound, warp grid
// and tile (the deepest ring that fits); false if there is no such candidate.
bool exchange_ws_pin(int ns, int M, bool pair, int ncw, int mi, int ni, int wm, int G, int Wn, int ew) {
  const int KT = (M + 15) / 16;
  const std::vector<Plan> cands = enumerate_plans(ns, pair, KT);
  const Plan* pick = nullptr;
  for (const Plan& p : cands)
    if (p.ncw == ncw && kInst[p.inst].MI == mi && kInst[p.inst].NI == ni && kInst[p.inst].EW == ew && p.WM == wm &&
        p.G == G && p.Wn == Wn &&
        (!pick || p.stages > pick->stages))
      pick = &p;
  if (!pick) return false;
  const long key = ((long)KT << 8 | ns) << 1 | (pair ? 1 : 0);
  std::lock_guard<std::mutex> lk(g_plan_mu);
  g_plan_cache[key] = *pick;
  return true;
}

// Forget the pin of (ns, M, pair), or every pin with ns <= 0: the next use computes the library's own choice again.
void exchange_ws_unpin(int ns, int M, bool pair) {
  std::lock_guard<std::mutex> lk(g_plan_mu);
  if (ns <= 0) { g_plan_cache.clear(); return; }
  const int KT = (M + 15) / 16;
  g_plan_cache.erase(((long)KT << 8 | ns) << 1 | (pair ? 1 : 0));
}

// human-readable plan (bench / tests)
void exchange_ws_describe(int ns, int M, bool pair, char* out, int n) {
  const Plan p = cached_plan(ns, pair, M);
  if (p.inst < 0) { snprintf(out, n, "no plan"); return; }
  snprintf(out, n, "warps %d+%d grid %dx%d (<=%dx%d blocks each) G %d Wn %d tile %dx%d eff %.3f stages %d passes %dx%d nbuf %d ldt %d smem %zu",
           p.ncw, kInst[p.inst].EW, p.WM, p.ncw / p.WM, kInst[p.inst].MI, kInst[p.inst].NI, p.G, p.Wn, p.rowsA, p.rowsB, p.eff, p.stages,
           (p.G + p.Gp - 1) / p.Gp, (p.Wn + p.Wp - 1) / p.Wp, p.nbuf, p.ldt, p.smem);
}

// returns launches issued, -1 if the tensor maps could not be encoded, -2 if the plan needs more partial-sum rows
// than the caller allocated
int run_exchange_ws(const ExArgs& e, cudaStream_t st) {
  const Plan p = cached_plan(e.ns, e.plane_stride != 0, e.M);
  if (p.inst < 0) return -1;
  if (e.ngroups_cap > 0 && (e.n_chol + p.G - 1) / p.G != e.ngroups_cap) return -2;   // the reduce sums exactly cap rows
  switch (p.inst) {
    case 0: return launch_xws<8, 5, 7, 3>(e, p, st);
    case 1: return launch_xws<8, 7, 5, 3>(e, p, st);
    case 2: return launch_xws<8, 6, 6, 3>(e, p, st);
    case 3: return launch_xws<12, 4, 7, 3>(e, p, st);
    case 4: return launch_xws<12, 7, 4, 3>(e, p, st);
    case 5: return launch_xws<12, 5, 5, 3>(e, p, st);
    case 6: return launch_xws<12, 5, 4, 3>(e, p, st);
    case 7: return launch_xws<12, 4, 5, 3>(e, p, st);
    case 8: return launch_xws<8, 5, 7, 7>(e, p, st);
    case 9: return launch_xws<8, 7, 5, 7>(e, p, st);
    case 10: return launch_xws<8, 6, 6, 7>(e, p, st);
  }
  return -1;
}

}  // namespace afq
