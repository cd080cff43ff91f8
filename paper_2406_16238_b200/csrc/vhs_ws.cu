// vhs_ws.cu - V_HS build (Eq. 9; "VHS step" PAPER.md:318):
//     A[(w, plane)][p][q] = sum_g Cf[(w, plane)][g] * L[g][p][q]
// warp-specialised TMA version that uses the symmetry L_g = L_g^T (8-fold real symmetry,
// PAPER.md:189; the paper's pack_chol, stores the same half): only tiles that
// touch the upper triangle (q >= p) are computed, straight out of the caller's DENSE L, and
// every element is stored twice, at [p][q] and mirrored at [q][p].  Half the flops and half
// the L bytes of the dense contraction, same result (each element of A is written once, from
// the upper-triangle entry of L).
//
// Tile: 128 rows (w, plane) x (8 p x 16 q) (1200 = 150 x 8 = 75 x 16: no ragged tile at the headline size).
// Producer: per 16-gamma stage one box of Cf (k-major, 128 x 16) and eight boxes {16 q, 1 p, 16 gamma} of L,
// all SWIZZLE_128B.  Consumers: 8 warps of 64 x 32 (8 x 4 DMMA blocks); a warp owns one q-octet and 4 p rows,
// so the mirrored store is 32 contiguous bytes per (row, q).
#include <vector>

#include "internal.h"
#include "tma.cuh"

namespace afq {

namespace {

constexpr int kProd = 128;
constexpr int BMv = 128, PT = 8, QT = 16, BKv = 16;
constexpr int NCWv = 8, NCTv = NCWv * 32, THREADSv = NCTv + kProd;
constexpr int A_BYTES = BMv * 128, B_BOX = BKv * 128, B_BYTES = PT * (QT / 16) * B_BOX;
constexpr int STAGE_BYTESv = A_BYTES + B_BYTES;    // 32 KB
constexpr int STAGESv = 6;
constexpr size_t SMEMv = (size_t)STAGESv * STAGE_BYTESv + 1024 + 256;

struct VhsArgs {
  double* Cb[kMaxGroup];  // output base per block of rpm rows: row r -> Cb[r / rpm] + (r % rpm) M M
  int rpm;
  const int* tiles;     // [ntile_n] packed (pb << 16 | qb)
  int M, n_chol, rows;  // rows = 2 nw
  int ntile_n, mtiles;
};

template <bool PACKED>
__global__ void __launch_bounds__(THREADSv, 1)
vhs_ws_kernel(const __grid_constant__ TensorMap tmA, const __grid_constant__ TensorMap tmB, const VhsArgs a) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)STAGESv * STAGE_BYTESv);
  uint64_t* empty = full + STAGESv;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KT = (a.n_chol + BKv - 1) / BKv;
  const int ntiles = a.ntile_n * a.mtiles;

  if (tid == 0) {
    for (int s = 0; s < STAGESv; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCWv); }
    fence_barrier_init();
  }
  __syncthreads();

  if (warp >= NCWv) {
    reg_dealloc<24>();
    if (warp == NCWv && lane == 0) {
      prefetch_tensormap(&tmA);
      prefetch_tensormap(&tmB);
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int tl = tile / a.mtiles;                // position in the upper-triangle tile list
        const int tn = a.tiles[tl], mt = tile % a.mtiles;
        const int p0 = (tn >> 16) * PT, q0 = (tn & 0xffff) * QT;
        for (int kt = 0; kt < KT; ++kt, ++it) {
          const int s = it % STAGESv;
          mbar_wait(&empty[s], ((it / STAGESv) & 1) ^ 1);
          mbar_expect_tx(&full[s], STAGE_BYTESv);
          unsigned char* sa = smem + (size_t)s * STAGE_BYTESv;
          tma_load_2d(sa, &tmA, &full[s], kt * BKv, mt * BMv);
          unsigned char* sb = sa + A_BYTES;
#pragma unroll
          for (int pl = 0; pl < PT; ++pl)
#pragma unroll
            for (int qb = 0; qb < QT / 16; ++qb)
              if (PACKED)   // tile-packed copy [tile][gamma][pl][q]: box (pl, qb) of tile tl
                tma_load_4d(sb + (pl * (QT / 16) + qb) * B_BOX, &tmB, &full[s], 0, pl * (QT / 16) + qb, kt * BKv, tl);
              else
                tma_load_3d(sb + (pl * (QT / 16) + qb) * B_BOX, &tmB, &full[s], q0 + 16 * qb, p0 + pl, kt * BKv);
        }
      }
    }
    return;
  }

  reg_alloc<240>();
  constexpr int MI = 8, NI = 4;
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp & 1, wn = warp >> 1;       // wn: (q-octet, p-half) of the 8 p x 16 q tile
  const int p = rperm(g);
  // A (k-major, 16-byte loads): chunk (4 kp + t) of row 8 b + p
  const uint32_t la0 = (uint32_t)(p * 128 + ((t ^ p) << 4));
  const uint32_t la1 = (uint32_t)(p * 128 + (((t ^ p) ^ 4) << 4));
  // B (n-major, 8-byte loads): box (j, qb) row k = 8 kp + 2 t + par, element q = 8 h + g
  const int hh = wn & 1, ph = wn >> 1;            // q-octet 0..1 of the 16-q box, p rows 4 ph .. 4 ph + 3
  const int chunk = 4 * hh + (g >> 1);
  uint32_t lb[2][2];                              // [kp][par]
#pragma unroll
  for (int kp = 0; kp < 2; ++kp)
#pragma unroll
    for (int par = 0; par < 2; ++par) {
      const int k = 8 * kp + 2 * t + par;
      lb[kp][par] = (uint32_t)(4 * ph * B_BOX + k * 128 + ((chunk ^ (k & 7)) << 4) + (g & 1) * 8);
    }
  const uint32_t smem_u = smem_u32(smem);
  const uint32_t aoff = (uint32_t)(wm * MI) * 1024u;
  const size_t MM = (size_t)a.M * a.M;

  uint32_t it = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int tn = a.tiles[tile / a.mtiles], mt = tile % a.mtiles;
    const int p0 = (tn >> 16) * PT, q0 = (tn & 0xffff) * QT;

    double acc[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    for (int kt = 0; kt < KT; ++kt, ++it) {
      const int s = it % STAGESv;
      mbar_wait(&full[s], (it / STAGESv) & 1);
      consumer_release_prev(empty, it, STAGESv, lane);
      const uint32_t sa = smem_u + (uint32_t)s * STAGE_BYTESv + aoff;
      const uint32_t sb = smem_u + (uint32_t)s * STAGE_BYTESv + A_BYTES;
#pragma unroll
      for (int kp = 0; kp < 2; ++kp) {
        double2 af[MI];
#pragma unroll
        for (int i = 0; i < MI; ++i) af[i] = lds128(sa + i * 1024 + (kp ? la1 : la0));
        double b0[NI], b1[NI];
#pragma unroll
        for (int j = 0; j < NI; ++j) {
          b0[j] = lds64(sb + j * (QT / 16) * B_BOX + lb[kp][0]);
          b1[j] = lds64(sb + j * (QT / 16) * B_BOX + lb[kp][1]);
        }
#pragma unroll
        for (int j = 0; j < NI; ++j)
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], af[i].x, b0[j]);
#pragma unroll
        for (int j = 0; j < NI; ++j)
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][j][0], acc[i][j][1], af[i].y, b1[j]);
      }
    }

    // ---- epilogue: direct store at [p][q] (q >= p) and mirrored store at [q][p] (q > p)
    const int ql = q0 + 8 * hh;                    // first q of this warp's octet
    const int pw = p0 + 4 * ph;                    // first of this warp's 4 p rows
    if (ql + 7 < pw) continue;                     // entirely below the diagonal: nothing to keep
    const int q = ql + 2 * t;                      // this lane's q, q + 1
    const bool fast = (ql >= pw + 4) && (pw + 4 <= a.M) && (ql + 8 <= a.M);
#pragma unroll
    for (int i = 0; i < MI; ++i) {
      const int r = mt * BMv + 8 * (wm * MI + i) + p;
      if (r >= a.rows) continue;
      double* Cr = a.Cb[r / a.rpm] + (size_t)(r % a.rpm) * MM;
      if (fast) {
#pragma unroll
        for (int j = 0; j < NI; ++j)
          *reinterpret_cast<double2*>(Cr + (size_t)(pw + j) * a.M + q) = make_double2(acc[i][j][0], acc[i][j][1]);
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          double* d = Cr + (size_t)(q + e) * a.M + pw;
          *reinterpret_cast<double2*>(d) = make_double2(acc[i][0][e], acc[i][1][e]);
          *reinterpret_cast<double2*>(d + 2) = make_double2(acc[i][2][e], acc[i][3][e]);
        }
      } else {
#pragma unroll
        for (int j = 0; j < NI; ++j) {
          const int pp = pw + j;
          if (pp >= a.M) continue;
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int qq = q + e;
            if (qq >= a.M || qq < pp) continue;
            Cr[(size_t)pp * a.M + qq] = acc[i][j][e];
            if (qq > pp) Cr[(size_t)qq * a.M + pp] = acc[i][j][e];
          }
        }
      }
    }
  }
}

// Lpk[t][g][pl][q] = L[g][p0(t) + pl][q0(t) + q] (zero outside the matrix); grid (ntile_n, gamma chunks)
__global__ void __launch_bounds__(PT * QT) pack_tiles_kernel(const double* L, double* Lpk, const int* tiles, int M,
                                                             int n_chol) {
  const int t = blockIdx.x;
  const int tn = tiles[t];
  const int p = (tn >> 16) * PT + threadIdx.x / QT, q = (tn & 0xffff) * QT + threadIdx.x % QT;
  const bool in = p < M && q < M;
  const size_t MM = (size_t)M * M;
  for (int g = blockIdx.y; g < n_chol; g += gridDim.y)
    Lpk[((size_t)t * n_chol + g) * (PT * QT) + threadIdx.x] = in ? L[(size_t)g * MM + (size_t)p * M + q] : 0.0;
}

}  // namespace

size_t vhs_ws_packed_doubles(int ntile_n, int n_chol) { return (size_t)ntile_n * n_chol * PT * QT; }

int run_pack_tiles(const double* L, double* Lpk, const int* tiles_dev, int ntile_n, int M, int n_chol,
                   cudaStream_t st) {
  const int gy = n_chol < 64 ? n_chol : 64;
  pack_tiles_kernel<<<dim3(ntile_n, gy), PT * QT, 0, st>>>(L, Lpk, tiles_dev, M, n_chol);
  return 1;
}

// host: list of (p-block, q-block) tiles that intersect the upper triangle, row-major
int vhs_ws_tile_list(int M, std::vector<int>* out) {
  out->clear();
  const int npb = (M + PT - 1) / PT, nqb = (M + QT - 1) / QT;
  for (int pb = 0; pb < npb; ++pb)
    for (int qb = 0; qb < nqb; ++qb)
      if (qb * QT + QT - 1 >= pb * PT) out->push_back((pb << 16) | qb);
  return (int)out->size();
}

bool vhs_ws_usable(int M, int n_chol, const void* L, const void* Cf, const void* C) {
  return (M % 2 == 0) && (n_chol % 2 == 0) && M < 65536 * PT &&
         ((((uintptr_t)L | (uintptr_t)Cf | (uintptr_t)C) & 15) == 0);
}

// algorithmic flops actually needed with the symmetric half: 2 * rows * n_chol * M (M + 1) / 2 * 2
int run_vhs_ws(const double* Cf, const double* L, double* C, const int* tiles_dev, int ntile_n, int M,
               int n_chol, int rows, bool packed, cudaStream_t st) {
  double* Cb[1] = {C};
  return run_vhs_ws_scatter(Cf, L, Cb, 1, rows, tiles_dev, ntile_n, M, n_chol, packed, st, 0);
}

int run_vhs_ws_scatter(const double* Cf, const double* L, double* const* Cb, int nmember, int rows_per_member,
                       const int* tiles_dev, int ntile_n, int M, int n_chol, bool packed, cudaStream_t st, long ldcf) {
  if (nmember < 1 || nmember > kMaxGroup || rows_per_member < 1) return -1;
  if (ldcf <= 0) ldcf = n_chol;                  // row stride of Cf (a column block of a wider matrix otherwise)
  if (ldcf & 1) return -1;
  const int rows = nmember * rows_per_member;
  static uint64_t attr = 0;
  if (auto once_ = first_use_on_device(&attr)) {
    cudaFuncSetAttribute(vhs_ws_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEMv);
    cudaFuncSetAttribute(vhs_ws_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEMv);
  }
  const int nsm = sm_count_current();
  TensorMap tmA, tmB;
  {
    const uint64_t dims[2] = {(uint64_t)n_chol, (uint64_t)rows};
    const uint64_t str[1] = {(uint64_t)ldcf * 8};
    const uint32_t box[2] = {BKv, BMv};
    if (make_tensor_map_f64(&tmA, Cf, 2, dims, str, box) != 0) return -1;
  }
  if (packed) {   // L = the tile-packed copy [ntile_n][n_chol][PT * QT / 16][16]
    const uint64_t dims[4] = {16, (uint64_t)(PT * QT / 16), (uint64_t)n_chol, (uint64_t)ntile_n};
    const uint64_t str[3] = {128, (uint64_t)PT * QT * 8, (uint64_t)n_chol * PT * QT * 8};
    const uint32_t box[4] = {16, 1, BKv, 1};
    if (make_tensor_map_f64(&tmB, L, 4, dims, str, box) != 0) return -1;
  } else {
    const uint64_t dims[3] = {(uint64_t)M, (uint64_t)M, (uint64_t)n_chol};
    const uint64_t str[2] = {(uint64_t)M * 8, (uint64_t)M * M * 8};
    const uint32_t box[3] = {16, 1, BKv};
    if (make_tensor_map_f64(&tmB, L, 3, dims, str, box) != 0) return -1;
  }
  VhsArgs a;
  for (int r = 0; r < kMaxGroup; ++r) a.Cb[r] = r < nmember ? Cb[r] : nullptr;
  a.rpm = rows_per_member;
  a.tiles = tiles_dev; a.M = M; a.n_chol = n_chol; a.rows = rows;
  a.ntile_n = ntile_n; a.mtiles = (rows + BMv - 1) / BMv;
  const long nt = (long)a.ntile_n * a.mtiles;
  const int grid = nt < nsm ? (int)nt : nsm;
  if (packed) vhs_ws_kernel<true><<<grid, THREADSv, SMEMv, st>>>(tmA, tmB, a);
  else vhs_ws_kernel<false><<<grid, THREADSv, SMEMv, st>>>(tmA, tmB, a);
  return 1;
}

}  // namespace afq
