// taylor_tc.cu - Taylor propagation T_n = A T_{n-1} / n, Acc += T_n (Eq. 12)
// in emulated single precision on the tcgen05 tensor cores, the second half of the mixed-precision mode
// ("single precision is used for propagations"; reading S24).  Same arithmetic as
// vhs_tc.cu: operands split into three bfloat16 numbers, six plane pairs, FP32 accumulation in tensor memory.
//
// The complex product is ONE real GEMM per walker: with T stored as real columns (re, im interleaved, N2 = 2 Nt)
//     A T = [Ar | Ai] * [T ; J T],   (J T)[k][2j] = -T[k][2j+1],  (J T)[k][2j+1] = T[k][2j],
// i.e. K = 2 Kp (Kp = M rounded up to 32, zero padded), both operands K-major:
//     Abf[w][3 planes][M rows][2 Kp]      bf16   [Ar row | Ai row]          (split_A_kernel, once per step)
//     Tb [w][3 planes][Np rows][2 Kp]     bf16   [T^T row | (J T)^T row]    (Np = N2 rounded up to 16)
// The epilogue of order n scales by 1/n, adds the term to the FP64 running sum Acc (walker layout) and writes
// the split, transposed term straight into the Tb of order n + 1 (lanes = consecutive k: 64-byte runs).
//
// Kernel: persistent CTA per SM, work unit = (walker, 128 rows of A); warp 0 TMA producer (boxes {32 k, 128
// rows, 3 planes} of Abf and {32 k, Np rows, 3 planes} of Tb), warp 1 tcgen05.mma M = 128, N = Np, K = 16
// (2 k-steps x 6 plane pairs per stage; hh into its own accumulator), warps 2-5 epilogue; two accumulator
// sets in tensor memory when Np <= 128.
#include "internal.h"
#include "tc.cuh"
#include "tma.cuh"

namespace afq {

namespace {

constexpr int TY_BK = 32;
constexpr int TY_M = 128;
constexpr int TY_APLANE = TY_M * TY_BK * 2;     // 8 KB
constexpr int TY_AOPER = 3 * TY_APLANE;         // 24 KB
constexpr int TY_ACC = 2;
constexpr int TY_TMEM_COLS = 512;
constexpr int TY_THREADS = 192;
constexpr int TY_SMEM_CAP = 232448;

// Abf[w][plane][m][reim * Kp + q] from A[w][reim][m][q]; grid (M, nw)
__global__ void __launch_bounds__(256) split_A_kernel(const double* __restrict__ A, __nv_bfloat16* __restrict__ Abf,
                                                      int M, int Kp) {
  const int m = blockIdx.x, w = blockIdx.y;
  const size_t MM = (size_t)M * M, plane = (size_t)M * 2 * Kp;
  __nv_bfloat16* out = Abf + (size_t)w * 3 * plane + (size_t)m * 2 * Kp;
  for (int idx = threadIdx.x; idx < 2 * Kp; idx += blockDim.x) {
    const int reim = idx / Kp, q = idx % Kp;
    const double x = q < M ? A[((size_t)w * 2 + reim) * MM + (size_t)m * M + q] : 0.0;
    __nv_bfloat16 h, mm, l;
    split3(x, h, mm, l);
    out[idx] = h;
    out[idx + plane] = mm;
    out[idx + 2 * plane] = l;
  }
}

// E1b[plane][m][q] (row stride 2 Kp, second half unused) from E1[m][q] - delta_mq: the one-body half step is
// applied as phi + (E1 - 1) phi with the identity part kept in FP64, so that the truncating FP32 accumulation
// acts on the small correction only (E1 = expm(-dt/2 h_mod) is 1 + O(dt)); grid M
__global__ void __launch_bounds__(256) split_E1_kernel(const double* __restrict__ E1, __nv_bfloat16* __restrict__ E1b,
                                                       int M, int Kp) {
  const int m = blockIdx.x;
  const size_t plane = (size_t)M * 2 * Kp;
  __nv_bfloat16* out = E1b + (size_t)m * 2 * Kp;
  for (int q = threadIdx.x; q < Kp; q += blockDim.x) {
    const double x = q < M ? E1[(size_t)m * M + q] - (q == m ? 1.0 : 0.0) : 0.0;
    __nv_bfloat16 h, mm, l;
    split3(x, h, mm, l);
    out[q] = h;
    out[q + plane] = mm;
    out[q + 2 * plane] = l;
  }
}

// Tb[w][plane][n][k] = T[w][k][n], Tb[w][plane][n][Kp + k] = (J T)[k][n]; zero for n >= N2 or k >= M.
// grid (Kp / 32, nw), 256 threads; T is [nw][M][N2] doubles (the walker layout)
__global__ void __launch_bounds__(256) split_T_kernel(const double* __restrict__ T, __nv_bfloat16* __restrict__ Tb,
                                                      int M, int N2, int Np, int Kp) {
  extern __shared__ double tsm[];                 // [32][N2 + 1]
  const int k0 = blockIdx.x * 32, w = blockIdx.y;
  const int ld = N2 + 1;
  for (int idx = threadIdx.x; idx < 32 * N2; idx += blockDim.x) {
    const int kl = idx / N2, n = idx % N2;
    tsm[kl * ld + n] = (k0 + kl < M) ? T[((size_t)w * M + k0 + kl) * N2 + n] : 0.0;
  }
  __syncthreads();
  const size_t plane = (size_t)Np * 2 * Kp;
  __nv_bfloat16* out = Tb + (size_t)w * 3 * plane;
  for (int idx = threadIdx.x; idx < 32 * Np; idx += blockDim.x) {
    const int n = idx / 32, kl = idx % 32;
    double t = 0.0, jt = 0.0;
    if (n < N2) {
      t = tsm[kl * ld + n];
      jt = (n & 1) ? tsm[kl * ld + n - 1] : -tsm[kl * ld + n + 1];
    }
    __nv_bfloat16 h, m, l;
    split3(t, h, m, l);
    size_t o = (size_t)n * 2 * Kp + k0 + kl;
    out[o] = h; out[o + plane] = m; out[o + 2 * plane] = l;
    split3(jt, h, m, l);
    o += Kp;
    out[o] = h; out[o + plane] = m; out[o + 2 * plane] = l;
  }
}

struct TyArgs {
  double* Acc;             // [nw][M][N2] running sum, FP64
  __nv_bfloat16* Tnext;    // Tb of the next order, or nullptr for the last one
  double alpha;            // 1 / n
  int assign;              // Acc = term instead of Acc += term
  const double* Src;       // assign only: Acc = Src + term (the operator is 1 + Aop; nullptr: none)
  int a_shared;            // the A operand is one matrix for all walkers
  int M, N2, Np, Kp, nw;
  int KT, mtiles, stages;
  uint32_t idesc;
  int nacc, d2off;         // accumulator sets in tensor memory (2 if Np <= 128), column offset of D2 in a set
  int b_plane;             // bytes of one plane of the B operand in a stage (Np * 64)
  int stage_bytes;
};

__global__ void __launch_bounds__(TY_THREADS, 1)
taylor_tc_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB, const TyArgs a) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  const int S = a.stages;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)S * a.stage_bytes);
  uint64_t* empty = full + S;
  uint64_t* tfull = empty + S;
  uint64_t* tempty = tfull + TY_ACC;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(tempty + TY_ACC);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nunits = a.nw * a.mtiles;            // work unit = (walker, 128 rows of A)

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    for (int s = 0; s < TY_ACC; ++s) { mbar_init(&tfull[s], 1); mbar_init(&tempty[s], 4); }
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc<TY_TMEM_COLS>(tmem_slot);
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
        const int w = u / a.mtiles, mt = u % a.mtiles;
        for (int kt = 0; kt < a.KT; ++kt, ++it) {
          const int s = it % S;
          mbar_wait(&empty[s], ((it / S) & 1) ^ 1);
          mbar_expect_tx(&full[s], (uint32_t)a.stage_bytes);
          unsigned char* sa = smem + (size_t)s * a.stage_bytes;
          tma_load_4d(sa, &tmA, &full[s], kt * TY_BK, mt * TY_M, 0, a.a_shared ? 0 : w);   // rows past M: zeros
          tma_load_4d(sa + TY_AOPER, &tmB, &full[s], kt * TY_BK, 0, 0, w);
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------ MMA issuer (lane 0)
    uint32_t it = 0, tc = 0;
    for (int u = blockIdx.x; u < nunits; u += gridDim.x, ++tc) {
      const int acc = tc % a.nacc;
      mbar_wait(&tempty[acc], ((tc / a.nacc) & 1) ^ 1);
      tc_fence_after();
      // D1: the hh plane pair; D2: the five small ones (truncating accumulation, see vhs_tc.cu)
      const uint32_t d1 = tmem_base + (uint32_t)acc * 256, d2 = d1 + a.d2off;
      for (int kt = 0; kt < a.KT; ++kt, ++it) {
        const int s = it % S;
        mbar_wait(&full[s], (it / S) & 1);
        tc_fence_after();
        if (lane == 0) {
          const uint32_t sa = smem_u32(smem + (size_t)s * a.stage_bytes), sb = sa + TY_AOPER;
          const int pa[6] = {2, 0, 1, 1, 0, 0}, pb[6] = {0, 2, 1, 0, 1, 0};   // lh hl mm mh hm hh
#pragma unroll
          for (int k = 0; k < TY_BK / 16; ++k) {
#pragma unroll
            for (int q = 0; q < 6; ++q) {
              const uint64_t da = umma_desc(sa + pa[q] * TY_APLANE + k * 32);
              const uint64_t db = umma_desc(sb + pb[q] * a.b_plane + k * 32);
              if (q == 5) umma_bf16(d1, da, db, a.idesc, (kt | k) != 0 ? 1u : 0u);
              else umma_bf16(d2, da, db, a.idesc, (kt | k | q) != 0 ? 1u : 0u);
            }
          }
          umma_commit(&empty[s]);
          if (kt == a.KT - 1) umma_commit(&tfull[acc]);
        }
        __syncwarp();
      }
    }
  } else {
    // ------------------------------------------------------------------ epilogue warps 2..5
    // thread = one row m of the term: scale, add to the FP64 running sum, write the split transposed term
    // (and J times it) into the B operand of the next order: lanes are consecutive k = m.
    const int quarter = warp & 3;
    const size_t bplane = (size_t)a.Np * 2 * a.Kp;
    const float alpha = (float)a.alpha;
    uint32_t tc = 0;
    for (int u = blockIdx.x; u < nunits; u += gridDim.x, ++tc) {
      const int acc = tc % a.nacc;
      const int w = u / a.mtiles, mt = u % a.mtiles;
      const int m = mt * TY_M + quarter * 32 + lane;
      mbar_wait(&tfull[acc], (tc / a.nacc) & 1);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (uint32_t)acc * 256 + ((uint32_t)(quarter * 32) << 16);
      double* accrow = a.Acc + ((size_t)w * a.M + m) * a.N2;
      __nv_bfloat16* tn = a.Tnext ? a.Tnext + (size_t)w * 3 * bplane + m : nullptr;
      const int nchunks = (a.N2 + 31) / 32;
#pragma unroll 1
      for (int c = 0; c < nchunks; ++c) {
        float v[32], v2[32];
        tmem_ld32(taddr + c * 32, v);
        tmem_ld32(taddr + a.d2off + c * 32, v2);
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] += v2[j];
        if (c == nchunks - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(&tempty[acc]);
        }
        if (m >= a.M) continue;
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const int n = 32 * c + j;
          if (n >= a.N2) continue;
          float t = v[j] * alpha;
          if (a.assign) {
            if (a.Src) {
              const double full = a.Src[((size_t)w * a.M + m) * a.N2 + n] + (double)t;
              accrow[n] = full;
              t = (float)full;                     // what the next order sees
            } else {
              accrow[n] = (double)t;
            }
          } else {
            accrow[n] += (double)t;
          }
          if (tn) {
            // an FP32 number is exactly three bfloat16 numbers
            const __nv_bfloat16 h = __float2bfloat16_rn(t);
            const float r1 = t - __bfloat162float(h);
            const __nv_bfloat16 mm = __float2bfloat16_rn(r1);
            const __nv_bfloat16 l = __float2bfloat16_rn(r1 - __bfloat162float(mm));
            __nv_bfloat16* o = tn + (size_t)n * 2 * a.Kp;
            o[0] = h; o[bplane] = mm; o[2 * bplane] = l;
            // (J T)[k][n ^ 1] = (n odd ? -t : +t)
            __nv_bfloat16* oj = tn + (size_t)(n ^ 1) * 2 * a.Kp + a.Kp;
            if (n & 1) { oj[0] = __hneg(h); oj[bplane] = __hneg(mm); oj[2 * bplane] = __hneg(l); }
            else { oj[0] = h; oj[bplane] = mm; oj[2 * bplane] = l; }
          }
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc<TY_TMEM_COLS>(tmem_base);
  }
}

int round_up(int v, int m) { return (v + m - 1) / m * m; }

}  // namespace

// ---------------------------------------------------------------------------------- host side
size_t taylor_tc_A_elems(int nw, int M) { return (size_t)nw * 3 * M * 2 * round_up(M, TY_BK); }
size_t taylor_tc_T_elems(int nw, int M, int N2) { return (size_t)nw * 3 * round_up(N2, 16) * 2 * round_up(M, TY_BK); }
bool taylor_tc_usable(int N2) { return N2 % 2 == 0 && round_up(N2, 16) <= 256; }

// Abf <- planar complex A [nw][2][M][M]
int taylor_tc_prepare_A(const double* A, void* Abf, int nw, int M, cudaStream_t st) {
  split_A_kernel<<<dim3(M, nw), 256, 0, st>>>(A, (__nv_bfloat16*)Abf, M, round_up(M, TY_BK));
  return 1;
}
// E1b (layout of ONE walker of Abf, real half only) <- real E1 [M][M]
int taylor_tc_prepare_E1(const double* E1, void* E1b, int M, cudaStream_t st) {
  split_E1_kernel<<<M, 256, 0, st>>>(E1, (__nv_bfloat16*)E1b, M, round_up(M, TY_BK));
  return 1;
}
// Tb <- T [nw][M][N2] (walker layout): [T^T | (J T)^T] rows
int taylor_tc_prepare_T(const double* T, void* Tb, int nw, int M, int N2, cudaStream_t st) {
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr))
    cudaFuncSetAttribute(split_T_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 32 * 257 * 8);
  const int Kp = round_up(M, TY_BK);
  split_T_kernel<<<dim3(Kp / 32, nw), 256, (size_t)32 * (N2 + 1) * 8, st>>>(T, (__nv_bfloat16*)Tb, M, N2,
                                                                            round_up(N2, 16), Kp);
  return 1;
}

// Out (+)= alpha * Aop * T per walker, where T is given by its split planes Tb and
//   real_shared = false: Aop = the walker's complex A (Abf of taylor_tc_prepare_A), K = 2 Kp
//   real_shared = true : Aop = one real matrix for all walkers (E1b of taylor_tc_prepare_E1), K = Kp
// assign: Out = [Src +] ... instead of Out += ...; Tnext (or nullptr) receives the split planes of the result.
// Returns launches or -1.
int taylor_tc_apply(const void* Aplanes, bool real_shared, const void* Tb, void* Tnext, double* Out, bool assign,
                    const double* Src, double alpha, int nw, int M, int N2, cudaStream_t st) {
  if (!taylor_tc_usable(N2)) return -1;
  const int Kp = round_up(M, TY_BK), Np = round_up(N2, 16);
  const int b_plane = Np * TY_BK * 2, stage = TY_AOPER + 3 * b_plane;
  int S = (TY_SMEM_CAP - 1024 - 256) / stage;
  if (S > 8) S = 8;
  if (S < 2) return -1;
  const size_t smem = (size_t)S * stage + 1024 + 256;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr))
    cudaFuncSetAttribute(taylor_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TY_SMEM_CAP);
  const int nsm = sm_count_current();
  TensorMap tmA, tmB;
  {
    const uint64_t dims[4] = {(uint64_t)2 * Kp, (uint64_t)M, 3, (uint64_t)(real_shared ? 1 : nw)};
    const uint64_t str[3] = {(uint64_t)2 * Kp * 2, (uint64_t)M * 2 * Kp * 2, (uint64_t)3 * M * 2 * Kp * 2};
    const uint32_t box[4] = {TY_BK, TY_M, 3, 1};
    if (make_tensor_map_bf16(&tmA, Aplanes, 4, dims, str, box, 64) != 0) return -1;
  }
  {
    const uint64_t dims[4] = {(uint64_t)2 * Kp, (uint64_t)Np, 3, (uint64_t)nw};
    const uint64_t str[3] = {(uint64_t)2 * Kp * 2, (uint64_t)Np * 2 * Kp * 2, (uint64_t)3 * Np * 2 * Kp * 2};
    const uint32_t box[4] = {TY_BK, (uint32_t)Np, 3, 1};
    if (make_tensor_map_bf16(&tmB, Tb, 4, dims, str, box, 64) != 0) return -1;
  }
  TyArgs a;
  a.Acc = Out; a.Tnext = (__nv_bfloat16*)Tnext; a.alpha = alpha; a.assign = assign ? 1 : 0;
  a.a_shared = real_shared ? 1 : 0; a.Src = Src;
  a.M = M; a.N2 = N2; a.Np = Np; a.Kp = Kp; a.nw = nw;
  a.KT = (real_shared ? Kp : 2 * Kp) / TY_BK; a.mtiles = (M + TY_M - 1) / TY_M; a.stages = S;
  a.idesc = umma_idesc_bf16(TY_M, Np); a.b_plane = b_plane; a.stage_bytes = stage;
  a.nacc = Np <= 128 ? 2 : 1; a.d2off = Np <= 128 ? 128 : 256;
  const long nu = (long)nw * a.mtiles;
  const int grid = nu < nsm ? (int)nu : nsm;
  taylor_tc_kernel<<<grid, TY_THREADS, smem, st>>>(tmA, tmB, a);
  return 1;
}

}  // namespace afq
