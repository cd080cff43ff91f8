// vhs_tc.cu - V_HS build in emulated single precision on the 5th-generation tensor cores
// (mixed precision: "single precision is used for propagations and double precision is used for
// local energy estimation"; Eq. 9):
//     A[(w, plane)][p][q] = sum_g Cf[(w, plane)][g] * L[g][p][q]
//
// FP64 has no tcgen05 kind, FP32 neither (kind::tf32 keeps 10 mantissa bits).  Single precision is
// therefore EMULATED: every double x is split once into three bfloat16 numbers x = h + m + l + O(2^-24 x)
// (h = bf16(x), m = bf16(x - h), l = bf16(x - h - m)), and the product of two such numbers keeps the six
// terms of order <= 2:  hh + hm + mh + hl + lh + mm.  A bf16 x bf16 product is exact in FP32 and
// tcgen05.mma.kind::f16 accumulates in FP32 in tensor memory, so the result carries the 24 significant bits
// of an FP32 GEMM with FP32 accumulation.
//
// Data: only tiles touching the upper triangle are kept - this kernel's own tiles of 8 p x 16 q (128 elements,
// 1200 = 150 x 8 = 75 x 16) -, K-MAJOR (gamma contiguous) and plane-major, so that two neighbouring tiles of one
// plane form one 256-row canonical SWIZZLE_64B K-major UMMA operand in shared memory:
//     Lb[3 planes][tile][128 n = (pl, qj)][Gp]   bf16, Gp = n_chol rounded up to 64, zero padded   (setup)
//     Ab[3 planes][Rp rows = (w, plane)][Gp]     bf16, Rp = rows rounded up to 128                 (per step)
// 6 bytes per kept element of L: 21.0 GB at M = 1200, Nchol = 4800 (dense FP64: 55.3 GB).
//
// Kernel: one persistent CTA per SM, 6 warps; a work unit is a PAIR of tiles x 128 rows.  Warp 0: TMA
// producer - per stage of 32 gamma one box {32 g, 128 rows, 3 planes} of Ab and one box {32 g, 128 n, 2 tiles,
// 3 planes} of Lb (72 KB), ring of 3 stages with mbarrier full/empty pairs.  Warp 1: allocates the 512 columns
// of tensor memory and issues tcgen05.mma M = 128, N = 256, K = 16: 2 k-steps x 6 plane pairs per stage;
// tcgen05.commit frees the stage and, after the last one, publishes the accumulator set.  Warps 2-5: epilogue -
// tcgen05.ld (one accumulator row = one (walker, plane) row of A per thread), 32 x 32 warp transposes so that
// a store instruction writes 128-byte runs of q (direct, [p][q]) or 64-byte runs of p (mirrored, [q][p]) of ONE
// row.  The hh plane pair has its own accumulator (the tensor core truncates when it adds: see the MMA
// loop), so the 512 columns hold ONE set of two N = 256 accumulators and the MMA warp waits while the
// epilogue drains it (about 2 % of a unit; TMA keeps filling the ring meanwhile).  Measured and what
// bounds it: profiles/r1v5_tc_c5.md.
#include <cuda_bf16.h>

#include <vector>

#include "internal.h"
#include "tma.cuh"
#include "tc.cuh"

namespace afq {

namespace {

constexpr int TC_GPAD = 64;                     // gamma extent of the split tensors is padded to this
constexpr int TC_BK = 32;                       // gamma per stage: 64 bytes of bf16 = one SWIZZLE_64B row
constexpr int TC_M = 128, TC_N = 128;
constexpr int TC_NT = 2;                        // N tiles per work unit: one A stage feeds both
constexpr int TC_PT = 8, TC_QT = 16;            // tile = 8 p x 16 q: 128-byte runs of q, 64-byte mirrored runs of p
constexpr int TC_PLANE = TC_M * TC_BK * 2;      // bytes of one plane of one 128-row operand in a stage (8 KB)
constexpr int TC_OPER = 3 * TC_PLANE;           // 24 KB
constexpr int TC_STAGE = (1 + TC_NT) * TC_OPER; // 72 KB: A, B tile 0, B tile 1
constexpr int TC_STAGES = 3;
constexpr int TC_ACC = 1;                       // accumulator sets in tensor memory; a set = TWO accumulators of
                                                // TC_NT x 128 columns: D1 for the hh plane pair, D2 for the other five
constexpr int TC_TMEM_COLS = 512;
constexpr int TC_THREADS = 192;
// instruction descriptor: M = 128, N = 256 (both tiles of a pair)
constexpr uint32_t kIdesc = umma_idesc_bf16(TC_M, TC_NT * TC_N);
constexpr size_t TC_SMEM = (size_t)TC_STAGES * TC_STAGE + 1024 + 256 + 1024;   // + alignment, barriers, row table

// Lb[plane][t][n][g] from the dense L[g][p][q]; grid (ntile, Gp / 64), 256 threads
__global__ void __launch_bounds__(256) split_L_kernel(const double* __restrict__ L, __nv_bfloat16* __restrict__ Lb,
                                                      const int* __restrict__ tiles, int M, int n_chol, int Gp) {
  __shared__ double sm[32][TC_N + 1];
  const int t = blockIdx.x, g00 = blockIdx.y * 64;
  const int tn = tiles[t];
  const int p0 = (tn >> 16) * TC_PT, q0 = (tn & 0xffff) * TC_QT;
  const size_t MM = (size_t)M * M;
  for (int pass = 0; pass < 2; ++pass) {
    const int g0 = g00 + pass * 32;
    for (int idx = threadIdx.x; idx < 32 * TC_N; idx += 256) {
      const int gl = idx / TC_N, n = idx % TC_N;
      const int p = p0 + n / TC_QT, q = q0 + n % TC_QT, g = g0 + gl;
      sm[gl][n] = (g < n_chol && p < M && q < M) ? L[(size_t)g * MM + (size_t)p * M + q] : 0.0;
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < 32 * TC_N; idx += 256) {
      const int n = idx / 32, gl = idx % 32;
      __nv_bfloat16 h, m, l;
      split3(sm[gl][n], h, m, l);
      const size_t o = ((size_t)t * TC_N + n) * Gp + g0 + gl, plane = (size_t)gridDim.x * TC_N * Gp;
      Lb[o] = h;
      Lb[o + plane] = m;
      Lb[o + 2 * plane] = l;
    }
    __syncthreads();
  }
}

// Ab[plane][r][g] from Cf[r][g]; rows >= rows and g >= n_chol are zero
__global__ void __launch_bounds__(256) split_cf_kernel(const double* __restrict__ Cf, __nv_bfloat16* __restrict__ Ab,
                                                       int rows, int n_chol, int Rp, int Gp) {
  const int r = blockIdx.y;
  const size_t plane = (size_t)Rp * Gp;
  for (int g = blockIdx.x * blockDim.x + threadIdx.x; g < Gp; g += gridDim.x * blockDim.x) {
    const double x = (r < rows && g < n_chol) ? Cf[(size_t)r * n_chol + g] : 0.0;
    __nv_bfloat16 h, m, l;
    split3(x, h, m, l);
    const size_t o = (size_t)r * Gp + g;
    Ab[o] = h;
    Ab[o + plane] = m;
    Ab[o + 2 * plane] = l;
  }
}

struct TcArgs {
  double* Cb[kMaxGroup];   // output base per block of rpm rows (as vhs_ws.cu)
  int rpm;
  const int* tiles;        // [ntile_n] packed (pb << 16 | qb)
  int M, rows, KT;         // KT = Gp / TC_BK
  int ntile_n, npairs, mtiles;
  // EPI = 1 (plain row-major output, split over K): C[ks][row][n], n < N
  double* C;
  long ldc, sCsplit;
  int N, nsplit, KTs;      // KTs: k stages per slice
};

template <int EPI>
__device__ __forceinline__ void unit_decode(const TcArgs& a, int u, int& pr, int& mt, int& kbeg, int& kend) {
  if (EPI == 1) {
    const int ks = u % a.nsplit, rest = u / a.nsplit;
    mt = rest % a.mtiles; pr = rest / a.mtiles;
    kbeg = ks * a.KTs; kend = min(a.KT, kbeg + a.KTs);
  } else {
    pr = u / a.mtiles; mt = u % a.mtiles;
    kbeg = 0; kend = a.KT;
  }
}

// EPI = 0: V_HS - symmetric scatter of the tiles of the tile list (direct + mirrored stores).
// EPI = 1: plain GEMM C[row][n] = sum_k A[row][k] B[n][k] over 256-column blocks of B rows, split over K
//          (force bias X = Theta^T . Lrot: K = Nt M is long, N = n_chol short).
template <int EPI>
__global__ void __launch_bounds__(TC_THREADS, 1)
vhs_tc_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB, const TcArgs a) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)TC_STAGES * TC_STAGE);
  uint64_t* empty = full + TC_STAGES;
  uint64_t* tfull = empty + TC_STAGES;
  uint64_t* tempty = tfull + TC_ACC;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + TC_ACC);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // work unit = (pair of N tiles, 128-row block[, K slice])
  const int nunits = a.npairs * a.mtiles * (EPI == 1 ? a.nsplit : 1);

  if (tid == 0) {
    for (int s = 0; s < TC_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    for (int s = 0; s < TC_ACC; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], 4); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<TC_TMEM_COLS>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------------ TMA producer
    if (lane == 0) {
      prefetch_tensormap(&tmA);
      prefetch_tensormap(&tmB);
      uint32_t it = 0;
      for (int u = blockIdx.x; u < nunits; u += gridDim.x) {
        int pr, mt, kbeg, kend;
        unit_decode<EPI>(a, u, pr, mt, kbeg, kend);
        for (int kt = kbeg; kt < kend; ++kt, ++it) {
          const int s = it % TC_STAGES;
          mbar_wait(&empty[s], ((it / TC_STAGES) & 1) ^ 1);
          mbar_expect_tx(&full[s], TC_STAGE);
          unsigned char* sa = smem + (size_t)s * TC_STAGE;
          tma_load_3d(sa, &tmA, &full[s], kt * TC_BK, mt * TC_M, 0);
          // both tiles of the pair in one box; a tile index past the end reads as zeros
          tma_load_4d(sa + TC_OPER, &tmB, &full[s], kt * TC_BK, 0, pr * TC_NT, 0);
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ MMA issuer (lane 0)
    uint32_t it = 0, tc = 0;
    for (int u = blockIdx.x; u < nunits; u += gridDim.x, ++tc) {
      const int acc = tc % TC_ACC;
      mbar_wait(&tempty[acc], ((tc / TC_ACC) & 1) ^ 1);
      tc_fence_after();
      // The tensor core adds into its FP32 accumulator with truncation.  Adding the five small plane pairs
      // (<= 2^-8 of hh) to the same accumulator would cost a truncation of the LARGE sum each time; kept apart,
      // the large sum sees one update per 16 gamma and the bias drops six-fold.  The epilogue adds D1 + D2.
      const uint32_t d1 = tmem_base + (uint32_t)acc * (2 * TC_NT * TC_N), d2 = d1 + TC_NT * TC_N;
      int pr_, mt_, kbeg, kend;
      unit_decode<EPI>(a, u, pr_, mt_, kbeg, kend);
      for (int kt = kbeg; kt < kend; ++kt, ++it) {
        const int s = it % TC_STAGES;
        mbar_wait(&full[s], (it / TC_STAGES) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t sa = smem_u32(smem + (size_t)s * TC_STAGE), sb = sa + TC_OPER;
          // plane pairs (A plane, B plane), small terms first: lh hl mm mh hm hh
          const int pa[6] = {2, 0, 1, 1, 0, 0}, pb[6] = {0, 2, 1, 0, 1, 0};
#pragma unroll
          for (int k = 0; k < TC_BK / 16; ++k) {
#pragma unroll
            for (int q = 0; q < 6; ++q) {
              const uint64_t da = umma_desc(sa + pa[q] * TC_PLANE + k * 32);
              const uint64_t db = umma_desc(sb + pb[q] * (TC_NT * TC_PLANE) + k * 32);   // 256 rows: tile 0, tile 1
              if (q == 5) umma_bf16(d1, da, db, kIdesc, ((kt - kbeg) | k) != 0 ? 1u : 0u);
              else umma_bf16(d2, da, db, kIdesc, ((kt - kbeg) | k | q) != 0 ? 1u : 0u);
            }
          }
          umma_commit(&empty[s]);                       // stage free when these MMAs have read it
          if (kt == kend - 1) umma_commit(&tfull[acc]);  // accumulators complete
        }
        __syncwarp();
      }
    }
  } else {
    // ------------------------------------------------------------------ epilogue warps 2..5
    // A thread owns one accumulator row (tensor-memory lane) = one (walker, plane) row of A.  Tiles
    // strictly above the diagonal are transposed across the warp 32 x 32 values at a time, so that one
    // store instruction writes, for ONE row, two 128-byte runs of q (direct) or four 64-byte runs of p
    // (mirrored) instead of 32 scattered 8-byte pieces.
    const int quarter = warp & 3;                 // tensor-memory lanes 32 quarter .. 32 quarter + 31
    const size_t MM = (size_t)a.M * a.M;
    double** rowp = reinterpret_cast<double**>(tmem_slot + 4) + quarter * 32;   // this warp's 32 row bases
    uint32_t tc = 0;
    int mt_cur = -1;
    for (int u = blockIdx.x; u < nunits; u += gridDim.x, ++tc) {
      const int acc = tc % TC_ACC;
      int pr, mt, kbeg, kend;
      unit_decode<EPI>(a, u, pr, mt, kbeg, kend);
      if (EPI == 1) {
        const int r = mt * TC_M + quarter * 32 + lane;
        __syncwarp();
        rowp[lane] = r < a.rows ? a.C + (size_t)(kbeg / a.KTs) * a.sCsplit + (size_t)r * a.ldc : nullptr;
        __syncwarp();
      } else if (mt != mt_cur) {
        const int r = mt * TC_M + quarter * 32 + lane;
        __syncwarp();
        rowp[lane] = r < a.rows ? a.Cb[r / a.rpm] + (size_t)(r % a.rpm) * MM : nullptr;
        __syncwarp();
        mt_cur = mt;
      }
      double* Cr = rowp[lane];
      mbar_wait(&tfull[acc], (tc / TC_ACC) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int nt = 0; nt < TC_NT; ++nt) {
        const int tl = pr * TC_NT + nt;
        const uint32_t taddr = tmem_base + (uint32_t)(acc * 2 * TC_NT + nt) * TC_N + ((uint32_t)(quarter * 32) << 16);
        float v[4][32];                           // v[c][j]: n = 32 c + j, p = p0 + n / 16, q = q0 + n % 16
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          float v2[32];
          tmem_ld32(taddr + c * 32, v[c]);
          tmem_ld32(taddr + TC_NT * TC_N + c * 32, v2);
#pragma unroll
          for (int j = 0; j < 32; ++j) v[c][j] += v2[j];
        }
        if (nt == TC_NT - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty[acc]);    // the accumulators may be overwritten from here on
        }
        if (tl >= a.ntile_n) continue;
        if (EPI == 1) {
          // plain rows: after the transpose of block c, lane l holds column 128 tl + 32 c + l of row i
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            warp_transpose32(v[c], lane);
            const int n = tl * TC_N + 32 * c + lane;
            if (n < a.N) {
#pragma unroll
              for (int i = 0; i < 32; ++i) {
                double* R = rowp[i];
                if (R) R[n] = (double)v[c][i];
              }
            }
          }
          continue;
        }
        const int tn = a.tiles[tl];
        const int p0 = (tn >> 16) * TC_PT, q0 = (tn & 0xffff) * TC_QT;
        const bool fast = (q0 >= p0 + TC_PT) && (p0 + TC_PT <= a.M) && (q0 + TC_QT <= a.M);
        if (fast) {
          // mirrored: block b holds q = q0 + 4 b + j / 8, p = p0 + j % 8
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            float t[32];
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int n = (j % 8) * TC_QT + 4 * b + j / 8;
              t[j] = v[n / 32][n % 32];
            }
            warp_transpose32(t, lane);
            const size_t off = (size_t)(q0 + 4 * b + lane / 8) * a.M + p0 + lane % 8;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              double* R = rowp[i];
              if (R) R[off] = (double)t[i];
            }
          }
          // direct: block c holds p = p0 + 2 c + j / 16, q = q0 + j % 16
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            warp_transpose32(v[c], lane);
            const size_t off = (size_t)(p0 + 2 * c + lane / 16) * a.M + q0 + lane % 16;
#pragma unroll
            for (int i = 0; i < 32; ++i) {
              double* R = rowp[i];
              if (R) R[off] = (double)v[c][i];
            }
          }
        } else if (Cr) {
          // tiles on the diagonal or the matrix edge: element by element from the thread's own row
#pragma unroll
          for (int c = 0; c < 4; ++c) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int n = 32 * c + j;
              const int pp = p0 + n / TC_QT, qq = q0 + n % TC_QT;
              if (pp >= a.M || qq >= a.M || qq < pp) continue;
              const double x = (double)v[c][j];
              Cr[(size_t)pp * a.M + qq] = x;
              if (qq > pp) Cr[(size_t)qq * a.M + pp] = x;
            }
          }
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<TC_TMEM_COLS>(tmem_base);
  }
}

}  // namespace

// ---------------------------------------------------------------------------------- host side
// (p-block, q-block) tiles of 8 x 16 elements that touch the upper triangle q >= p, row-major
int vhs_tc_tile_list(int M, std::vector<int>* out) {
  out->clear();
  const int npb = (M + TC_PT - 1) / TC_PT, nqb = (M + TC_QT - 1) / TC_QT;
  for (int pb = 0; pb < npb; ++pb)
    for (int qb = 0; qb < nqb; ++qb)
      if (qb * TC_QT + TC_QT - 1 >= pb * TC_PT) out->push_back((pb << 16) | qb);
  return (int)out->size();
}
int vhs_tc_gamma_padded(int n_chol) { return (n_chol + TC_GPAD - 1) / TC_GPAD * TC_GPAD; }
int vhs_tc_rows_padded(int rows) { return (rows + TC_M - 1) / TC_M * TC_M; }
size_t vhs_tc_L_elems(int ntile_n, int n_chol) { return (size_t)ntile_n * 3 * TC_N * vhs_tc_gamma_padded(n_chol); }
size_t vhs_tc_cf_elems(int rows, int n_chol) { return (size_t)3 * vhs_tc_rows_padded(rows) * vhs_tc_gamma_padded(n_chol); }

int run_vhs_tc_split_L(const double* L, void* Lb, const int* tiles_dev, int ntile_n, int M, int n_chol,
                       cudaStream_t st) {
  const int Gp = vhs_tc_gamma_padded(n_chol);
  // grid.x up to 2^31 - 1 tiles; grid.y = Gp / 64 <= 65535 (n_chol < 4.2e6)
  split_L_kernel<<<dim3(ntile_n, Gp / 64), 256, 0, st>>>(L, (__nv_bfloat16*)Lb, tiles_dev, M, n_chol, Gp);
  return 1;
}

// A (scattered by owner as run_vhs_ws_scatter) from Cf [rows][n_chol] and the split tensor Lb; Ab is scratch
int run_vhs_tc(const double* Cf, void* Ab, const void* Lb, double* const* Cb, int nmember, int rows_per_member,
               const int* tiles_dev, int ntile_n, int M, int n_chol, cudaStream_t st) {
  if (nmember < 1 || nmember > kMaxGroup || rows_per_member < 1) return -1;
  const int rows = nmember * rows_per_member;
  const int Gp = vhs_tc_gamma_padded(n_chol), Rp = vhs_tc_rows_padded(rows);
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(vhs_tc_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM);
    cudaFuncSetAttribute(vhs_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM);
  }
  const int nsm = sm_count_current();
  split_cf_kernel<<<dim3((Gp + 255) / 256, Rp), 256, 0, st>>>(Cf, (__nv_bfloat16*)Ab, rows, n_chol, Rp, Gp);
  TensorMap tmA, tmB;
  {
    const uint64_t dims[3] = {(uint64_t)Gp, (uint64_t)Rp, 3};
    const uint64_t str[2] = {(uint64_t)Gp * 2, (uint64_t)Rp * Gp * 2};
    const uint32_t box[3] = {TC_BK, TC_M, 3};
    if (make_tensor_map_bf16(&tmA, Ab, 3, dims, str, box, 64) != 0) return -1;
  }
  {
    const uint64_t dims[4] = {(uint64_t)Gp, TC_N, (uint64_t)ntile_n, 3};
    const uint64_t str[3] = {(uint64_t)Gp * 2, (uint64_t)TC_N * Gp * 2, (uint64_t)ntile_n * TC_N * Gp * 2};
    const uint32_t box[4] = {TC_BK, TC_N, TC_NT, 3};
    if (make_tensor_map_bf16(&tmB, Lb, 4, dims, str, box, 64) != 0) return -1;
  }
  TcArgs a;
  for (int r = 0; r < kMaxGroup; ++r) a.Cb[r] = r < nmember ? Cb[r] : nullptr;
  a.rpm = rows_per_member;
  a.tiles = tiles_dev; a.M = M; a.rows = rows; a.KT = Gp / TC_BK;
  a.ntile_n = ntile_n; a.npairs = (ntile_n + TC_NT - 1) / TC_NT; a.mtiles = Rp / TC_M;
  const long nt = (long)a.npairs * a.mtiles;
  const int grid = nt < nsm ? (int)nt : nsm;
  a.C = nullptr; a.ldc = 0; a.sCsplit = 0; a.N = 0; a.nsplit = 1; a.KTs = a.KT;
  vhs_tc_kernel<0><<<grid, TC_THREADS, TC_SMEM, st>>>(tmA, tmB, a);
  return 2;
}

// ---- force bias on the same kernel: X[s][row][g] = sum_{k in slice s} ThT[row][k] Lrot[g][k] -------------
int fb_tc_rows_padded(int n_chol) { return (n_chol + TC_NT * TC_N - 1) / (TC_NT * TC_N) * (TC_NT * TC_N); }
size_t fb_tc_L_elems(int n_chol, int K) { return (size_t)3 * fb_tc_rows_padded(n_chol) * vhs_tc_gamma_padded(K); }
size_t fb_tc_T_elems(int rows, int K) { return (size_t)3 * vhs_tc_rows_padded(rows) * vhs_tc_gamma_padded(K); }

// K slices so that (pairs x row blocks x slices) fills the SMs; every slice is non-empty
int fb_tc_split(int rows, int n_chol, int K, int max_split) {
  const int nsm = sm_count_current();
  const int KT = vhs_tc_gamma_padded(K) / TC_BK;
  const long base = (long)(fb_tc_rows_padded(n_chol) / (TC_NT * TC_N)) * (vhs_tc_rows_padded(rows) / TC_M);
  int best = 1;
  double best_cost = 1e300;
  for (int s = 1; s <= max_split; ++s) {
    const int KTs = (KT + s - 1) / s;
    if ((long)KTs * (s - 1) >= KT && s > 1) continue;
    const double cost = (double)((base * s + nsm - 1) / nsm) * (KTs + 8);
    if (cost < best_cost) { best_cost = cost; best = s; }
  }
  return best;
}

// Lrb[3][rows padded to 256][Kp] from Lrot [n_chol][K] (setup)
int run_fb_tc_split_L(const double* Lrot, void* Lrb, int n_chol, int K, cudaStream_t st) {
  const int Kp = vhs_tc_gamma_padded(K), Rp = fb_tc_rows_padded(n_chol);
  split_cf_kernel<<<dim3((Kp + 255) / 256 > 64 ? 64 : (Kp + 255) / 256, Rp), 256, 0, st>>>(Lrot, (__nv_bfloat16*)Lrb, n_chol, K,
                                                                                          Rp, Kp);
  return 1;
}

int run_fb_tc(const double* ThT, void* Tbuf, const void* Lrb, double* Xp, long ldc, long sCsplit, int rows, int n_chol,
              int K, int split, cudaStream_t st) {
  const int Kp = vhs_tc_gamma_padded(K), Rp = vhs_tc_rows_padded(rows), Np = fb_tc_rows_padded(n_chol);
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(vhs_tc_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM);
    cudaFuncSetAttribute(vhs_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM);
  }
  const int nsm = sm_count_current();
  split_cf_kernel<<<dim3((Kp + 255) / 256 > 64 ? 64 : (Kp + 255) / 256, Rp), 256, 0, st>>>(ThT, (__nv_bfloat16*)Tbuf, rows, K, Rp,
                                                                                          Kp);
  TensorMap tmA, tmB;
  {
    const uint64_t dims[3] = {(uint64_t)Kp, (uint64_t)Rp, 3};
    const uint64_t str[2] = {(uint64_t)Kp * 2, (uint64_t)Rp * Kp * 2};
    const uint32_t box[3] = {TC_BK, TC_M, 3};
    if (make_tensor_map_bf16(&tmA, Tbuf, 3, dims, str, box, 64) != 0) return -1;
  }
  const int ntile = Np / TC_N;
  {
    const uint64_t dims[4] = {(uint64_t)Kp, TC_N, (uint64_t)ntile, 3};
    const uint64_t str[3] = {(uint64_t)Kp * 2, (uint64_t)TC_N * Kp * 2, (uint64_t)Np * Kp * 2};
    const uint32_t box[4] = {TC_BK, TC_N, TC_NT, 3};
    if (make_tensor_map_bf16(&tmB, Lrb, 4, dims, str, box, 64) != 0) return -1;
  }
  TcArgs a;
  for (int r = 0; r < kMaxGroup; ++r) a.Cb[r] = nullptr;
  a.rpm = 1; a.tiles = nullptr; a.M = 0; a.rows = rows; a.KT = Kp / TC_BK;
  a.ntile_n = ntile; a.npairs = ntile / TC_NT; a.mtiles = Rp / TC_M;
  a.C = Xp; a.ldc = ldc; a.sCsplit = sCsplit; a.N = n_chol;
  a.nsplit = split < 1 ? 1 : split; a.KTs = (a.KT + a.nsplit - 1) / a.nsplit;
  const long nt = (long)a.npairs * a.mtiles * a.nsplit;
  const int grid = nt < nsm ? (int)nt : nsm;
  vhs_tc_kernel<1><<<grid, TC_THREADS, TC_SMEM, st>>>(tmA, tmB, a);
  return 2;
}

}  // namespace afq
