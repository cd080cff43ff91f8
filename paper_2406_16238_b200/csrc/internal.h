// internal.h - declarations shared by the translation units of libafqmc (not installed).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/afqmc.h"
#include "gemm.cuh"

namespace afq {

constexpr int kMaxOcc = 64;     // largest occupied block (columns per spin) supported
constexpr int kMaxTaylor = 16;
constexpr int kMaxGroup = 8;    // members of a distributed-Hamiltonian group

// Per-device one-off work (cudaFuncSetAttribute is per device; handles may live on different devices of one
// process, and may be driven from different host threads).  Usage:
//     if (auto once = first_use_on_device(&mask)) { cudaFuncSetAttribute(...); }
// The guard holds a process-wide mutex for the whole if statement and marks the device as done only when it is
// destroyed, so a second thread can never launch the kernel between "bit set" and "attribute set".
inline std::mutex& device_once_mutex() {
  static std::mutex m;
  return m;
}
struct OnceGuard {
  std::unique_lock<std::mutex> lk;
  uint64_t* mask = nullptr;
  uint64_t bit = 0;
  bool first = false;
  OnceGuard() = default;
  OnceGuard(OnceGuard&& o) noexcept : lk(std::move(o.lk)), mask(o.mask), bit(o.bit), first(o.first) { o.mask = nullptr; }
  explicit operator bool() const { return first; }
  ~OnceGuard() { if (first && mask) *mask |= bit; }
};
inline OnceGuard first_use_on_device(uint64_t* mask) {
  int dev = 0;
  cudaGetDevice(&dev);
  OnceGuard g;
  g.lk = std::unique_lock<std::mutex>(device_once_mutex());
  g.mask = mask;
  g.bit = 1ull << (dev & 63);
  g.first = (*mask & g.bit) == 0;
  return g;
}
// largest dynamic shared-memory size requested so far on the current device; the guard is true if `bytes`
// exceeds it (same locking as above; the new size is recorded when the guard is destroyed)
struct GrowGuard {
  std::unique_lock<std::mutex> lk;
  size_t* slot = nullptr;
  size_t bytes = 0;
  bool grow = false;
  GrowGuard() = default;
  GrowGuard(GrowGuard&& o) noexcept : lk(std::move(o.lk)), slot(o.slot), bytes(o.bytes), grow(o.grow) { o.slot = nullptr; }
  explicit operator bool() const { return grow; }
  ~GrowGuard() { if (grow && slot) *slot = bytes; }
};
inline GrowGuard grow_on_device(size_t* cur /* [64] */, size_t bytes) {
  int dev = 0;
  cudaGetDevice(&dev);
  GrowGuard g;
  g.lk = std::unique_lock<std::mutex>(device_once_mutex());
  g.slot = &cur[dev & 63];
  g.bytes = bytes;
  g.grow = bytes > *g.slot;
  return g;
}
// SM count of the current device (cached per device)
inline int sm_count_current() {
  static std::atomic<int> n[64];
  int dev = 0;
  cudaGetDevice(&dev);
  int v = n[dev & 63].load(std::memory_order_relaxed);
  if (!v) {
    cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
    if (v <= 0) v = 148;
    n[dev & 63].store(v, std::memory_order_relaxed);
  }
  return v;
}

enum GemmKind { GEMM_KN = 0, GEMM_NK = 1, GEMM_KMKN = 2, GEMM_CPLX_KN = 3 };

// gemm.cu
// Fills the vec* fields, picks a tile configuration and launches.  Returns launches issued.
int run_gemm(GemmKind kind, GemmArgs a, cudaStream_t st);

// small.cu ---------------------------------------------------------------------------------
struct OTArgs {                 // overlap / Theta / one-body energy, one CTA per (block, walker)
  const double* W;              // walkers as doubles [nw][M][2*Nt]
  const double* trial;          // [M][Nt] (real part)
  const double* trial_im = nullptr;   // [M][Nt] imaginary part of a complex trial, else null; trialT then holds
                                      // the planes (Re psi^T, -Im psi^T), [2][Nt][M]
  const double* hrot;           // [Nt][M] (only with want_e1)
  double* det;                  // [nw][nblk] complex: det(psi_s^T phi_s)
  double* ThT;                  // [nw][2][Nt][M] planar transpose of Theta (want_theta)
  double* e1;                   // [nw][nblk] complex partial one-body energy (want_e1)
  int M, Nt, nblk;
  int off[2], ns[2];
  int want_theta, want_e1;
  // DMMA route (all three set): trial^T [Nt][M], scratch O [nw][Nt][Nt] complex, scratch Aop [nw][2Nt][2Nt]
  const double* trialT;
  double* Obuf;
  double* Aop;
};
int run_overlap_theta(const OTArgs& a, int nw, cudaStream_t st);

struct ShiftArgs {              // a4: force bias -> shifted fields and scalars, one CTA per walker
  const double* Xp;             // [splitK][2*nw][n_chol] partial sums of X (planar re/im rows)
  long sXp;                     // stride between partial slices
  int nsplit;
  const double* m;              // [n_chol]
  const double* x;              // [nw][n_chol] aux fields
  double* X;                    // [nw][2][n_chol] summed X incl. spin factor (kept for diagnostics)
  double* Cf;                   // [nw][2][n_chol]: rows of the V_HS GEMM: (sqrt(dt) Im xs, -sqrt(dt) Re xs)
  double* cfb;                  // [nw] complex
  double* cmf;                  // [nw] complex
  int n_chol;
  double spin_factor, sqrt_dt;
  double xbar_bound = 0.0;      // > 0: |xbar_g| capped (afqmc_params::xbar_bound)
};
int run_field_shift(const ShiftArgs& a, int nw, cudaStream_t st);

struct WeightArgs {
  const double* det_old;        // [nw][nblk] complex
  const double* det_new;        // [nw][nblk] complex
  const double* cfb;
  const double* cmf;
  double* weights;              // [nw] in/out
  double* ovlp;                 // [nw] complex out: overlap of the new walkers
  int nblk, rhf;
  double expo;                  // -dt (E_const - E_shift)
  double dt = 0.0, ehyb_bound = 0.0;   // > 0: |I| bounded (afqmc_params::ehyb_bound)
};
int run_weight_update(const WeightArgs& a, int nw, cudaStream_t st);

struct QRArgs {                 // thin QR per (block, walker), in place: Cholesky-QR passes until orthonormal
  double* W;                    // [nw][M][2*Nt]
  double* detR;                 // [nw][nblk] real: multiplied by prod diag(R) of this pass
  int M, Nt, nblk;
  int off[2], ns[2];
  int* shifted = nullptr;       // device counter of shifted (breakdown) passes, may be null
};
int run_cholqr_pass(const QRArgs& a, int nw, cudaStream_t st);
int run_ovlp_div_detR(double* ovlp, const double* detR, int nblk, int rhf, int nw, cudaStream_t st);
int run_fill(double* p, double v, long n, cudaStream_t st);

// exchange.cu ------------------------------------------------------------------------------
struct ExArgs {
  const double* Lrot;           // [n_chol][Nt][M]
  const double* ThT;            // [nw][2][Nt][M]
  double* expart;               // [ngroups][nw] complex: sum over the group's g of tr(T T)
  double* X;                    // [n_chol][nw] complex: tr(T_g) (accumulated over spin blocks)
  int M, Nt, n_chol, nw;
  int off, ns;                  // spin block
  int accumulate;               // 1: add to expart / X (second spin block)
  int ngroups_cap = 0;          // > 0: rows of `expart` the caller allocated and sums; exchange_ws refuses (-2) a plan that writes another count
                                // (a plan pinned after the handle was created)
  long plane_stride = 0;        // != 0 (exchange_ws only): Lrot = Lr + i Li, the imaginary plane starts plane_stride
                                // doubles after Lrot; T is then the complex product and X = tr(T) of it
};
int exchange_group_size(int ns);            // gamma per CTA tile for this block size
int run_exchange(const ExArgs& a, cudaStream_t st);
// exchange_ws.cu: warp-specialised TMA version (needs even M and 16-byte aligned operands)
bool exchange_ws_usable(int M, const void* Lrot, const void* ThT);
int exchange_ws_group_size(int ns, int M, bool pair = false);      // the plan depends on the K = M loop length
double exchange_ws_efficiency(int ns, int M, bool pair = false);
void exchange_ws_describe(int ns, int M, bool pair, char* out, int n);
bool exchange_ws_pin(int ns, int M, bool pair, int ncw, int mi, int ni, int wm, int G, int Wn, int ew);
void exchange_ws_unpin(int ns, int M, bool pair);
int run_exchange_ws(const ExArgs& a, cudaStream_t st);

struct EnergyArgs {
  const double* expart; int ngroups;
  const double* X;              // [n_chol][nw] complex
  const double* e1;             // [nw][nblk] complex
  double* E_out;                // [nw][3] complex
  int n_chol, nw, nblk;
  double spin_factor;
};
int run_energy_reduce(const EnergyArgs& a, cudaStream_t st);
int run_energy_reduce2(const EnergyArgs& a, const double* expart2, int ngroups2, cudaStream_t st);

// vhs_ws.cu: symmetric-half V_HS build on the warp-specialised TMA pipeline
bool vhs_ws_usable(int M, int n_chol, const void* L, const void* Cf, const void* C);
int vhs_ws_tile_list(int M, std::vector<int>* out);
int run_vhs_ws(const double* Cf, const double* L, double* C, const int* tiles_dev, int ntile_n, int M,
               int n_chol, int rows, bool packed, cudaStream_t st);
// the same contraction with the output rows scattered by blocks of rows_per_member rows: row r goes
// to Cb[r / rows_per_member] + (r % rows_per_member) * M * M (distributed Hamiltonian: the partial
// V_HS of a walker is stored straight into its owner's receive slot, possibly peer memory)
int run_vhs_ws_scatter(const double* Cf, const double* L, double* const* Cb, int nmember, int rows_per_member,
                       const int* tiles_dev, int ntile_n, int M, int n_chol, bool packed, cudaStream_t st,
                       long ldcf = 0);
// tile-packed upper triangle of L (the paper's pack_chol): [ntile_n][n_chol][8][16]
size_t vhs_ws_packed_doubles(int ntile_n, int n_chol);
int run_pack_tiles(const double* L, double* Lpk, const int* tiles_dev, int ntile_n, int M, int n_chol,
                   cudaStream_t st);

// vhs_tc.cu: V_HS build in emulated single precision (bf16 x 3 on tcgen05, FP32 accumulation in TMEM)
int vhs_tc_gamma_padded(int n_chol);
int vhs_tc_tile_list(int M, std::vector<int>* out);   // its own 8 p x 16 q tiles touching the upper triangle
size_t vhs_tc_L_elems(int ntile_n, int n_chol);      // bf16 elements of the split tile tensor
size_t vhs_tc_cf_elems(int rows, int n_chol);        // bf16 elements of the split coefficient scratch
int run_vhs_tc_split_L(const double* L, void* Lb, const int* tiles_dev, int ntile_n, int M, int n_chol,
                       cudaStream_t st);
int run_vhs_tc(const double* Cf, void* Ab, const void* Lb, double* const* Cb, int nmember, int rows_per_member,
               const int* tiles_dev, int ntile_n, int M, int n_chol, cudaStream_t st);

// force bias on the same tcgen05 kernel (plain epilogue, split over K = Nt M)
size_t fb_tc_L_elems(int n_chol, int K);
size_t fb_tc_T_elems(int rows, int K);
int fb_tc_split(int rows, int n_chol, int K, int max_split);
int run_fb_tc_split_L(const double* Lrot, void* Lrb, int n_chol, int K, cudaStream_t st);
int run_fb_tc(const double* ThT, void* Tbuf, const void* Lrb, double* Xp, long ldc, long sCsplit, int rows, int n_chol,
              int K, int split, cudaStream_t st);

// taylor_tc.cu: Taylor propagation in the same emulated single precision (bf16 x 3 on tcgen05)
size_t taylor_tc_A_elems(int nw, int M);
size_t taylor_tc_T_elems(int nw, int M, int N2);
bool taylor_tc_usable(int N2);
int taylor_tc_prepare_A(const double* A, void* Abf, int nw, int M, cudaStream_t st);
int taylor_tc_prepare_E1(const double* E1, void* E1b, int M, cudaStream_t st);
int taylor_tc_prepare_T(const double* T, void* Tb, int nw, int M, int N2, cudaStream_t st);
int taylor_tc_apply(const void* Aplanes, bool real_shared, const void* Tb, void* Tnext, double* Out, bool assign,
                    const double* Src, double alpha, int nw, int M, int N2, cudaStream_t st);

// gemm_ws.cu: warp-specialised TMA GEMMs (return -1 when the shapes/alignment cannot be served)
// stream-K scratch of one caller (stream): accumulators of the tiles cut by a chunk boundary + one flag per CTA
struct KnStreamK { double* part; size_t part_doubles; int* flag; int flags; int force = 0; };
int run_gemm_ws_kn(const double* A, long lda, long sPlane, long sA, bool cplx, const double* B, long ldb, long sB,
                   double* C, double* C2, long ldc, long sC, int M, int N, int K, int batch, double alpha,
                   int mode, cudaStream_t st, const KnStreamK* sk = nullptr);
int gemm_ws_nk_split(int M, int N, int K, int max_split);
int run_gemm_ws_nk(const double* A, long lda, const double* B, long ldb, double* C, long ldc, long sCsplit,
                   int M, int N, int K, int split, cudaStream_t st);

// block.cu: population control (comb), walker permutation, estimator sums
int run_comb(double* weights, const double* xi, double* cum, int* map, int nw, cudaStream_t st);
int run_permute_rows(void* rows, void* tmp, const int* map, long row_bytes, int nw, cudaStream_t st);
int run_estimators(const double* weights, const double* E, double* out4, int nw, cudaStream_t st);

// shard.cu: fixed-order reductions of the per-member receive slots (distributed Hamiltonian)
int run_sum_slots(double* dst, const double* const* slots, int G, long n, cudaStream_t st);
int run_push_e2(double* dst, const double* E, int n, cudaStream_t st);
int run_energy_finish(double* E_out, const double* e1, const double* const* slots, int G, int nblk, double sf,
                      int nw, cudaStream_t st);

// cplx.cu: complex Cholesky vectors on the real kernels
struct CShiftArgs {
  const double* Xp; long sXp; int nsplit;     // [split][2 nw][nv] partial sums over the nv = 2 nf planes
  const double* m;                            // [nf] (the first nf entries of the mean field of the planes)
  const double* x;                            // [nw][nf]
  double *X, *Cf, *cfb, *cmf;                 // X [nw][2][nf]; Cf [nw][2][nv]
  int nf;
  double spin_factor, sqrt_dt;
  double xbar_bound = 0.0;
};
struct CEnergyArgs {
  const double* Xr; const double* Xi;         // tr(T) of the Re / Im plane runs, [nf][nw] complex
  const double* expart[3][2]; int ngroups[2]; // sums of tr(TT) of the runs r, i, r + i per spin block
  const double* e1r; const double* e1i;       // [nw][nblk] complex: Re(h)rot . Theta, Im(h)rot . Theta
  double* E_out;
  int nf, nw, nblk;
  double spin_factor;
  int pair = 0;                               // 1: Xr holds tr(T) of the complex T, expart[0] its tr(T T) (one run)
};
int run_hermitian_planes(const double* L_cplx, double* Ks, int M, int n, cudaStream_t st);
int run_add(double* dst, const double* a, const double* b, long n, cudaStream_t st);
int run_add_scaled(double* dst, const double* a, const double* b, double sb, long n, cudaStream_t st);   // dst = a + sb b
// A[r][p][q] += sign(q - p) * B[r][p][q] for `rows` matrices of M x M (B: an antisymmetric sum computed by the
// symmetric-half V_HS kernel, i.e. correct above the diagonal and mirrored with the wrong sign below)
int run_add_antisym(double* A, const double* B, int rows, int M, cudaStream_t st);
int run_deinterleave(double* planar, const double* inter, int M, cudaStream_t st);       // [2][M][M] <- [M][2M]
int run_caxpby_identity(double* P, double a, double idval, int M, cudaStream_t st);    // interleaved complex P
int run_field_shift_cplx(const CShiftArgs& a, int nw, cudaStream_t st);
int run_energy_cplx(const CEnergyArgs& a, cudaStream_t st);
int run_e1(const OTArgs& a, int nw, cudaStream_t st);    // small.cu: one-body energy sum only

// fused_small.cu: whole step / whole local energy in one kernel per call for small systems (c1-sized)
struct SmallArgs {
  double* W;                    // [nw][M][Nt] complex, in/out (step), in (energy)
  const double* trial;          // [M][Nt]
  const double* Lrot;           // [n_chol][Nt][M]
  const double* hrot;           // [Nt][M]
  const double* m;              // [n_chol]
  const double* x;              // [nw][n_chol]
  const double* L;              // [n_chol][M][M]
  const double* E1;             // [M][M]
  double* weights;              // [nw]
  double* ovlp;                 // [nw] complex
  double* Xdbg;                 // [nw][2][n_chol] or null (afqmc_debug_read 0)
  double* Adbg;                 // [nw][2][M][M] or null (afqmc_debug_read 1)
  double* E_out;                // [nw][3] complex
  int M, Nt, nblk, n_chol, K, rhf, gchunk, lchunk;
  int off[2], ns[2];
  double sf, sqrt_dt, dt, expo, xbar_bound, ehyb_bound;
};
bool small_path_fits(int M, int Nt, int nsmax, int n_chol);
int run_small_step(SmallArgs a, int nw, cudaStream_t st);
int run_small_energy(SmallArgs a, int nw, cudaStream_t st);

// setup.cu ---------------------------------------------------------------------------------
int run_mean_field(const double* L, const double* P, double* m, int M, int n_chol, cudaStream_t st);
int run_sum_mL(const double* L, const double* m, double* out, int M, int n_chol, cudaStream_t st);
// hmod = h1 - 0.5 * sum_s part[s] + mL
int run_hmod(const double* h1, const double* part, int nsplit, const double* mL, double* hmod, int M,
             cudaStream_t st);
int run_axpby_identity(double* P, double a, double idval, int M, cudaStream_t st);  // P = a P + idval I
int run_scale_copy(double* dst, const double* src, double a, long n, cudaStream_t st);

}  // namespace afq
