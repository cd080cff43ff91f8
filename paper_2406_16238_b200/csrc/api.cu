// api.cu - the C ABI of libafqmc (include/afqmc.h): handle, setup, and the stream-ordered
// sequence of kernels that makes one walker step / one local-energy evaluation.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "internal.h"

using namespace afq;

struct afqmc_handle {
  afqmc_params p;
  int M = 0, Nt = 0, nblk = 1, off[2] = {0, 0}, ns[2] = {0, 0};
  int n_chol = 0, maxw = 0, K = 6, rhf = 1;
  double sf = 2.0;
  int dev = 0;                 // CUDA device of the handle (that of L_chol); every entry point switches to it
  cudaStream_t st = nullptr;
  bool own_stream = false;
  const double* L = nullptr;
  std::vector<void*> allocs;
  // constants
  double *h1 = nullptr, *trial = nullptr, *trialT = nullptr, *Lrot = nullptr, *hrot = nullptr;
  double* trial_im = nullptr;   // complex trial: Im psi [M][Nt]; trialT is then [2][Nt][M] = (Re psi^T, -Im psi^T)
  double *m = nullptr, *hmod = nullptr, *E1 = nullptr, *Xs = nullptr, *Pa = nullptr, *Pb = nullptr;
  double E_const = 0.0, e_shift = 0.0, e_trial = NAN, hmod_norm1 = 0.0, dt_cached = NAN;
  // per-step workspaces
  double *det_old = nullptr, *det_new = nullptr, *ThT = nullptr, *Xp = nullptr, *X = nullptr, *Cf = nullptr;
  double *cfb = nullptr, *cmf = nullptr, *A = nullptr, *T0 = nullptr, *T1 = nullptr, *Acc = nullptr;
  double *ovlp = nullptr, *detR = nullptr;
  double *expart[2] = {nullptr, nullptr}, *Xe = nullptr, *e1 = nullptr;
  int exgroups[2] = {0, 0};
  // staging for host-pointer calls
  double *stW = nullptr, *stWt = nullptr, *stX = nullptr, *stE = nullptr;
  // population control / estimators
  double *cum = nullptr, *xi_dev = nullptr, *est_dev = nullptr, *ovlp_tmp = nullptr;
  int* pmap = nullptr;
  KnStreamK sk = {nullptr, 0, nullptr, 0};   // stream-K scratch of the batched KN GEMMs (gemm_ws.cu)
  int* qr_shifted = nullptr;     // device counter: shifted Cholesky-QR passes (ill-conditioned walkers) so far
  // CUDA graphs of whole blocks (afqmc_run_block on device buffers), keyed by the call's arguments
  struct BlockGraph {
    const void *W, *wt, *x, *xi, *E, *est;
    int nw, n_steps, pop_every, ortho_phase;
    double dt;
    int seen;                 // eager runs so far with this key (the 2nd call captures)
    cudaGraphExec_t exec;
    int64_t launches;
  };
  std::vector<BlockGraph> graphs;
  bool graph_on = true;
  int64_t graph_replays = 0;
  // distributed Hamiltonian (afqmc_shard_*): group of G members, this one holds a gamma slice
  int G = 1, rank = 0, mwg = 0;                 // mwg = G * maxw: walkers of the whole group
  bool shard_ready = true, peers_set = false;
  double *theta_buf = nullptr, *a_slots = nullptr, *scal_slots = nullptr, *e_slots = nullptr;
  double *hmod_part = nullptr, *setup_buf = nullptr, *e1zero = nullptr, *Etmp = nullptr, *scal_sum = nullptr;
  double Ec_part = 0.0, e2trial_part = 0.0, e1b_trial = 0.0;
  double* peer[4][kMaxGroup] = {};              // [theta, a, scal, e][member]
  double *Obuf = nullptr, *Aop = nullptr;       // overlap / inverse operands of the DMMA overlap-Theta route
  bool ot_gemm = false;
  int fb_split = 1;
  bool small = false;   // whole step / local energy in one kernel each (fused_small.cu)
  bool ws = false;      // warp-specialised TMA kernels (even M); else the cp.async kernels
  bool ws_vhs = false;
  int* vhs_tiles = nullptr;
  double* Lpk = nullptr;   // tile-packed upper triangle of L (pack_chol)
  void *Lb = nullptr, *Ab = nullptr;   // mixed precision: bf16 x 3 split tiles of L, split coefficients
  int* tc_tiles = nullptr;
  int tc_ntile = 0;
  // complex Cholesky vectors (cplx.cu): n_chol counts the 4n real planes, nf = 2n fields
  bool cplx = false;
  int nf = 0;
  double *hmod_c = nullptr, *cbuf = nullptr;    // complex: planar h_mod; scratch of the complex expm (8 M^2)
  double* A2 = nullptr;                         // complex: antisymmetric part of V_HS before the sign fix
  double *Ks = nullptr, *hrot_i = nullptr, *Lrot_sum = nullptr, *E1c = nullptr, *e1i = nullptr, *Xe_s = nullptr;
  double* expart_c[2][2] = {{nullptr, nullptr}, {nullptr, nullptr}};   // [set i / set r+i][spin block]
  int exgroups_c[2] = {0, 0};
  std::vector<double> hm_host;                  // h_mod, planar (re, im), for the host expm
  void *Abf = nullptr, *Tb0 = nullptr, *Tb1 = nullptr;   // mixed precision: split A and Taylor terms
  void* E1b = nullptr;                                    // mixed precision: split one-body propagator
  void *Lrb = nullptr, *Tfb = nullptr;                    // mixed precision: split Lrot and Theta^T (force bias)
  int fb_tc_nsplit = 1;
  int vhs_ntile = 0;
  long step_count = 0;
  int last_nw = 0;
  int64_t launches = 0;
  std::string err;
  // per-stage event timing (afqmc_set_profiling)
  bool prof = false;
  std::vector<cudaEvent_t> ev_free;
  struct Bracket { int stage; cudaEvent_t a, b; };
  std::vector<Bracket> ev_pending;
  double stage_ms[AFQMC_STAGE_COUNT] = {0};
  int64_t stage_n[AFQMC_STAGE_COUNT] = {0};
};

// message of the last failed afqmc_create / handle-less call ON THIS HOST THREAD (afqmc_last_error(NULL))
static thread_local std::string g_create_err;

namespace {

// switch to the handle's device for the duration of an API call
struct DevGuard {
  int prev = -1;
  bool sw = false;
  explicit DevGuard(int dev) {
    cudaGetDevice(&prev);
    if (prev != dev) { cudaSetDevice(dev); sw = true; }
  }
  ~DevGuard() { if (sw) cudaSetDevice(prev); }
};

int device_of(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return -1; }
  return (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) ? at.device : -1;
}

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  cudaError_t e = cudaPointerGetAttributes(&at, p);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int fail(afqmc_handle* h, int code, const std::string& msg) {
  if (h) h->err = msg; else g_create_err = msg;
  return code;
}

int check_cuda(afqmc_handle* h, const char* where) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(h, AFQMC_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
  return AFQMC_OK;
}

double* dalloc(afqmc_handle* h, size_t n_doubles) {
  void* p = nullptr;
  if (n_doubles == 0) n_doubles = 2;
  if (cudaMalloc(&p, n_doubles * sizeof(double)) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  h->allocs.push_back(p);
  return (double*)p;
}

void dfree_one(afqmc_handle* h, double* p) {
  for (auto& q : h->allocs)
    if (q == p) { cudaFree(q); q = nullptr; }
}

// copy `n` doubles from a host-or-device pointer to a device buffer on the stream
void to_device(afqmc_handle* h, double* dst, const void* src, size_t n) {
  cudaMemcpyAsync(dst, src, n * sizeof(double), cudaMemcpyDefault, h->st);
}

// Brackets the launches of one stage with two events when profiling is on.
struct StageTimer {
  afqmc_handle* h;
  int stage;
  cudaEvent_t a = nullptr, b = nullptr;
  static cudaEvent_t get(afqmc_handle* h) {
    cudaEvent_t e = nullptr;
    if (!h->ev_free.empty()) { e = h->ev_free.back(); h->ev_free.pop_back(); }
    else if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; }
    return e;
  }
  StageTimer(afqmc_handle* h_, int stage_) : h(h_), stage(stage_) {
    if (!h->prof) return;
    a = get(h); b = get(h);
    if (a && b) cudaEventRecord(a, h->st);
  }
  ~StageTimer() {
    if (!h->prof || !a || !b) return;
    cudaEventRecord(b, h->st);
    h->ev_pending.push_back({stage, a, b});
  }
};

GemmArgs gemm_args() {
  GemmArgs a;
  memset(&a, 0, sizeof(a));
  a.batch = 1;
  a.splitK = 1;
  a.alpha = 1.0;
  return a;
}

// E1 = expm(-dt/2 h_mod) by scaling and squaring of a degree-16 Taylor polynomial (Horner),
// every product on the DMMA GEMM.  (The oracle uses an eigendecomposition instead: reading S6.)
// complex Hermitian h_mod (complex Cholesky vectors): E1 = expm(-dt/2 h_mod) by scaling and squaring of a
// degree-18 Taylor polynomial (Horner) on the device, as the real case: every product is the planar-complex
// DMMA GEMM (A planar, B and C interleaved), with a de-interleave between the squarings.  The oracle uses eigh.
void build_E1_complex(afqmc_handle* h, double dt) {
  StageTimer tm(h, AFQMC_STAGE_E1_BUILD);
  const int M = h->M;
  const long MM = (long)M * M;
  double nrm = 0.5 * fabs(dt) * h->hmod_norm1;
  int s = 0;
  while (nrm > 0.25 && s < 40) { nrm *= 0.5; ++s; }
  double* X = h->cbuf;              // planar scaled argument   [2][MM]
  double* P = h->cbuf + 2 * MM;     // interleaved              [M][2M]
  double* Q = h->cbuf + 4 * MM;     // interleaved
  double* Pp = h->cbuf + 6 * MM;    // planar copy of P for the squarings
  h->launches += run_scale_copy(X, h->hmod_c, -0.5 * dt / std::ldexp(1.0, s), 2 * MM, h->st);
  h->launches += run_fill(P, 0.0, 2 * MM, h->st);
  h->launches += run_caxpby_identity(P, 0.0, 1.0, M, h->st);
  auto cgemm = [&](const double* Apl, const double* B, double* C, double alpha) {
    GemmArgs g = gemm_args();
    g.A = Apl; g.A2 = Apl + MM; g.lda = M; g.B = B; g.ldb = 2 * M; g.C = C; g.ldc = 2 * M;
    g.M = M; g.N = 2 * M; g.K = M; g.alpha = alpha;
    h->launches += run_gemm(GEMM_CPLX_KN, g, h->st);
  };
  for (int k = 18; k >= 1; --k) {                 // Horner: P <- 1 + X P / k
    cgemm(X, P, Q, 1.0 / k);
    h->launches += run_caxpby_identity(Q, 1.0, 1.0, M, h->st);
    std::swap(P, Q);
  }
  for (int i = 0; i < s; ++i) {
    h->launches += run_deinterleave(Pp, P, M, h->st);
    cgemm(Pp, P, Q, 1.0);
    std::swap(P, Q);
  }
  h->launches += run_deinterleave(h->E1c, P, M, h->st);
  h->dt_cached = dt;
}

void build_E1(afqmc_handle* h, double dt) {
  if (h->cplx) { build_E1_complex(h, dt); return; }
  StageTimer tm(h, AFQMC_STAGE_E1_BUILD);
  const int M = h->M;
  const long MM = (long)M * M;
  double nrm = 0.5 * fabs(dt) * h->hmod_norm1;
  int s = 0;
  while (nrm > 0.25 && s < 40) { nrm *= 0.5; ++s; }
  h->launches += run_scale_copy(h->Xs, h->hmod, -0.5 * dt / std::ldexp(1.0, s), MM, h->st);
  h->launches += run_fill(h->Pa, 0.0, MM, h->st);
  h->launches += run_axpby_identity(h->Pa, 0.0, 1.0, M, h->st);
  double *P = h->Pa, *Q = h->Pb;
  for (int k = 16; k >= 1; --k) {
    GemmArgs g = gemm_args();
    g.A = h->Xs; g.lda = M; g.B = P; g.ldb = M; g.C = Q; g.ldc = M;
    g.M = M; g.N = M; g.K = M; g.alpha = 1.0 / k;
    h->launches += run_gemm(GEMM_KN, g, h->st);
    h->launches += run_axpby_identity(Q, 1.0, 1.0, M, h->st);
    std::swap(P, Q);
  }
  for (int i = 0; i < s; ++i) {
    GemmArgs g = gemm_args();
    g.A = P; g.lda = M; g.B = P; g.ldb = M; g.C = Q; g.ldc = M;
    g.M = M; g.N = M; g.K = M;
    h->launches += run_gemm(GEMM_KN, g, h->st);
    std::swap(P, Q);
  }
  h->launches += run_scale_copy(h->E1, P, 1.0, MM, h->st);
  if (h->E1b) h->launches += taylor_tc_prepare_E1(h->E1, h->E1b, M, h->st);
  h->dt_cached = dt;
}

OTArgs ot_args(afqmc_handle* h, const double* W, double* det, int want_theta, int want_e1,
               double* ThT = nullptr) {
  OTArgs a;
  a.W = W; a.trial = h->trial; a.trial_im = h->trial_im; a.hrot = h->hrot; a.det = det; a.ThT = ThT ? ThT : h->ThT; a.e1 = h->e1;
  a.M = h->M; a.Nt = h->Nt; a.nblk = h->nblk;
  for (int b = 0; b < 2; ++b) { a.off[b] = h->off[b]; a.ns[b] = h->ns[b]; }
  a.want_theta = want_theta; a.want_e1 = want_e1;
  a.trialT = h->ot_gemm ? h->trialT : nullptr; a.Obuf = h->Obuf; a.Aop = h->Aop;
  return a;
}

SmallArgs small_args(afqmc_handle* h, double* W) {
  SmallArgs a{};
  a.W = W; a.trial = h->trial; a.Lrot = h->Lrot; a.hrot = h->hrot; a.m = h->m; a.L = h->L; a.E1 = h->E1;
  a.ovlp = h->ovlp; a.Xdbg = h->X; a.Adbg = h->A;
  a.M = h->M; a.Nt = h->Nt; a.nblk = h->nblk; a.n_chol = h->n_chol; a.K = h->K; a.rhf = h->rhf;
  for (int b = 0; b < 2; ++b) { a.off[b] = h->off[b]; a.ns[b] = h->ns[b]; }
  a.sf = h->sf; a.xbar_bound = h->p.xbar_bound; a.ehyb_bound = h->p.ehyb_bound;
  return a;
}

// exchange + Coulomb + final sums for the nw walkers whose Theta^T sits in h->ThT; e1 [nw][nblk]
int energy_from_theta(afqmc_handle* h, const double* e1, double* E_out, int nw) {
  for (int b = 0; b < h->nblk; ++b) {
    StageTimer tm(h, AFQMC_STAGE_EXCHANGE);
    ExArgs e;
    e.Lrot = h->Lrot; e.ThT = h->ThT; e.expart = h->expart[b]; e.X = h->Xe;
    e.M = h->M; e.Nt = h->Nt; e.n_chol = h->n_chol; e.nw = nw;
    e.off = h->off[b]; e.ns = h->ns[b]; e.accumulate = b > 0; e.ngroups_cap = h->exgroups[b];
    if (h->ws) {
      const int r = run_exchange_ws(e, h->st);
      if (r == -2) return fail(h, AFQMC_ERR_INVALID, "exchange: the tile plan was changed (afqmc_exchange_plan_pin) after this handle was created");
      if (r < 0) return fail(h, AFQMC_ERR_CUDA, "exchange: tensor map encode failed");
      h->launches += r;
    } else {
      h->launches += run_exchange(e, h->st);
    }
  }
  StageTimer tm(h, AFQMC_STAGE_E_REDUCE);
  EnergyArgs r;
  r.expart = h->expart[0]; r.ngroups = h->exgroups[0];
  r.X = h->Xe; r.e1 = e1; r.E_out = E_out;
  r.n_chol = h->n_chol; r.nw = nw; r.nblk = h->nblk; r.spin_factor = h->sf;
  h->launches += run_energy_reduce2(r, h->nblk > 1 ? h->expart[1] : nullptr, h->exgroups[1], h->st);
  return AFQMC_OK;
}

// complex Cholesky vectors: Lrot = Lr + i Li as two planes
int local_energy_complex_device(afqmc_handle* h, const double* W, double* E_out, int nw) {
  const int nf = h->nf;
  {
    StageTimer tm(h, AFQMC_STAGE_E_THETA);
    OTArgs a = ot_args(h, W, h->det_old, 1, 1);
    h->launches += run_overlap_theta(a, nw, h->st);           // e1 <- Re(h)rot . Theta
    a.hrot = h->hrot_i; a.e1 = h->e1i;
    h->launches += run_e1(a, nw, h->st);                      // e1i <- Im(h)rot . Theta
  }
  const size_t lsz = (size_t)nf * h->Nt * h->M;
  CEnergyArgs c;
  c.pair = h->ws ? 1 : 0;
  if (h->ws) {
    // ONE run: the tile's rows are [Re plane | Im plane] of the same vectors, T = Lrot Theta is put together as a
    // complex matrix by the epilogue warps (exchange_ws.cu, pair mode)
    for (int b = 0; b < h->nblk; ++b) {
      StageTimer tm(h, AFQMC_STAGE_EXCHANGE);
      ExArgs e;
      e.Lrot = h->Lrot; e.plane_stride = (long)lsz; e.ThT = h->ThT; e.expart = h->expart_c[0][b]; e.X = h->Xe;
      e.M = h->M; e.Nt = h->Nt; e.n_chol = nf; e.nw = nw;
      e.off = h->off[b]; e.ns = h->ns[b]; e.accumulate = b > 0; e.ngroups_cap = h->exgroups_c[b];
      const int r = run_exchange_ws(e, h->st);
      if (r == -2) return fail(h, AFQMC_ERR_INVALID, "exchange: the tile plan was changed (afqmc_exchange_plan_pin) after this handle was created");
      if (r < 0) return fail(h, AFQMC_ERR_CUDA, "exchange: tensor map encode failed");
      h->launches += r;
    }
    c.Xr = h->Xe; c.Xi = nullptr;
    for (int b = 0; b < 2; ++b) {
      c.expart[0][b] = h->expart_c[0][b]; c.expart[1][b] = nullptr; c.expart[2][b] = nullptr;
      c.ngroups[b] = h->exgroups_c[b];
    }
  } else {
    // odd M (no TMA): three runs of the cp.async kernel (Re planes, Im planes, their sum), cplx.cu
    const double* lrot[3] = {h->Lrot, h->Lrot + lsz, h->Lrot_sum};
    double* xe[3] = {h->Xe, h->Xe + (size_t)nf * h->mwg * 2, h->Xe_s};
    for (int k = 0; k < 3; ++k)
      for (int b = 0; b < h->nblk; ++b) {
        StageTimer tm(h, AFQMC_STAGE_EXCHANGE);
        ExArgs e;
        e.Lrot = lrot[k]; e.ThT = h->ThT; e.expart = k == 0 ? h->expart[b] : h->expart_c[k - 1][b]; e.X = xe[k];
        e.M = h->M; e.Nt = h->Nt; e.n_chol = nf; e.nw = nw;
        e.off = h->off[b]; e.ns = h->ns[b]; e.accumulate = b > 0;
        h->launches += run_exchange(e, h->st);
      }
    c.Xr = xe[0]; c.Xi = xe[1];
    for (int b = 0; b < 2; ++b) {
      c.expart[0][b] = h->expart[b]; c.expart[1][b] = h->expart_c[0][b]; c.expart[2][b] = h->expart_c[1][b];
      c.ngroups[b] = h->exgroups_c[b];
    }
  }
  StageTimer tm(h, AFQMC_STAGE_E_REDUCE);
  c.e1r = h->e1; c.e1i = h->e1i; c.E_out = E_out;
  c.nf = nf; c.nw = nw; c.nblk = h->nblk; c.spin_factor = h->sf;
  h->launches += run_energy_cplx(c, h->st);
  return AFQMC_OK;
}

int local_energy_device(afqmc_handle* h, const double* W, double* E_out, int nw) {
  if (h->cplx) return local_energy_complex_device(h, W, E_out, nw);
  if (h->small) {
    StageTimer tm(h, AFQMC_STAGE_FUSED_ENERGY);
    SmallArgs a = small_args(h, const_cast<double*>(W));
    a.E_out = E_out;
    h->launches += run_small_energy(a, nw, h->st);
    return AFQMC_OK;
  }
  {
    StageTimer tm(h, AFQMC_STAGE_E_THETA);
    h->launches += run_overlap_theta(ot_args(h, W, h->det_old, 1, 1), nw, h->st);
  }
  return energy_from_theta(h, h->e1, E_out, nw);
}

// One walker step on device buffers (rows a1-a10), stream ordered, no synchronisation.
// a3 + a4 for the nw walkers whose Theta^T sits in h->ThT (with this handle's Cholesky vectors)
int force_bias_shift_device(afqmc_handle* h, const double* x, double dt, int nw) {
  const int M = h->M, Nt = h->Nt, nc = h->n_chol;
  // a3: X[(w,part)][g] = sum_k ThT[(w,part)][k] Lrot[g][k], split over k
  int nsplit = h->fb_split;
  if (h->Lrb) {     // mixed precision: the shift xbar may be ANY complex vector (Eqs. 12, 16 hold for every
                    // xbar), so single precision here changes the sampling efficiency only, not the estimator
    StageTimer tm(h, AFQMC_STAGE_FORCE_BIAS);
    nsplit = h->fb_tc_nsplit;
    const int r = run_fb_tc(h->ThT, h->Tfb, h->Lrb, h->Xp, nc, (long)2 * h->mwg * nc, 2 * nw, nc, Nt * M, nsplit, h->st);
    if (r < 0) return fail(h, AFQMC_ERR_CUDA, "force bias (mixed precision): tensor map encode failed");
    h->launches += r;
  } else {
    StageTimer tm(h, AFQMC_STAGE_FORCE_BIAS);
    GemmArgs g = gemm_args();
    g.A = h->ThT; g.lda = (long)Nt * M; g.B = h->Lrot; g.ldb = (long)Nt * M;
    g.C = h->Xp; g.ldc = nc; g.M = 2 * nw; g.N = nc; g.K = Nt * M;
    g.splitK = h->fb_split; g.sCsplit = (long)2 * h->mwg * nc;
    int r = -1;
    if (h->ws)
      r = run_gemm_ws_nk(h->ThT, (long)Nt * M, h->Lrot, (long)Nt * M, h->Xp, nc, g.sCsplit, 2 * nw, nc, Nt * M,
                         h->fb_split, h->st);
    h->launches += r > 0 ? r : run_gemm(GEMM_NK, g, h->st);
  }
  // a4: shifted fields, scalars, V_HS coefficients
  if (h->cplx) {
    StageTimer tm(h, AFQMC_STAGE_FIELD_SHIFT);
    CShiftArgs c;
    c.Xp = h->Xp; c.sXp = (long)2 * h->mwg * nc; c.nsplit = nsplit; c.m = h->m; c.x = x;
    c.X = h->X; c.Cf = h->Cf; c.cfb = h->cfb; c.cmf = h->cmf; c.nf = h->nf;
    c.spin_factor = h->sf; c.sqrt_dt = sqrt(dt); c.xbar_bound = h->p.xbar_bound;
    h->launches += run_field_shift_cplx(c, nw, h->st);
  } else {
    StageTimer tm(h, AFQMC_STAGE_FIELD_SHIFT);
    ShiftArgs s;
    s.Xp = h->Xp; s.sXp = (long)2 * h->mwg * nc; s.nsplit = nsplit; s.m = h->m; s.x = x;
    s.X = h->X; s.Cf = h->Cf; s.cfb = h->cfb; s.cmf = h->cmf; s.n_chol = nc;
    s.spin_factor = h->sf; s.sqrt_dt = sqrt(dt); s.xbar_bound = h->p.xbar_bound;
    h->launches += run_field_shift(s, nw, h->st);
  }
  return AFQMC_OK;
}

void reortho_device(afqmc_handle* h, double* W, int nw, bool fix_overlaps);
int finish_step_device(afqmc_handle* h, double* W, double* wt, const double* cfb, const double* cmf, double dt, int nw);
int propagate_device(afqmc_handle* h, double* W, double* wt, const double* cfb, const double* cmf, double dt, int nw);

int step_device(afqmc_handle* h, double* W, double* wt, const double* x, double dt, int nw) {
  const int M = h->M, nc = h->n_chol;
  const long MM = (long)M * M;
  if (!(h->dt_cached == dt)) build_E1(h, dt);
  if (h->small) {
    {
      StageTimer tm(h, AFQMC_STAGE_FUSED_STEP);
      SmallArgs a = small_args(h, W);
      a.x = x; a.weights = wt;
      a.sqrt_dt = sqrt(dt); a.dt = dt; a.expo = -dt * (h->E_const - h->e_shift);
      h->launches += run_small_step(a, nw, h->st);
    }
    h->step_count += 1;
    h->last_nw = nw;
    if (h->p.ortho_every > 0 && h->step_count % h->p.ortho_every == 0) reortho_device(h, W, nw, true);
    return AFQMC_OK;
  }

  // a1/a2: overlap, Theta
  {
    StageTimer tm(h, AFQMC_STAGE_OVERLAP_THETA);
    h->launches += run_overlap_theta(ot_args(h, W, h->det_old, 1, 0), nw, h->st);
  }
  {
    const int rc = force_bias_shift_device(h, x, dt, nw);
    if (rc != AFQMC_OK) return rc;
  }
  // a5: A[(w,part)][pq] = sum_g Cf[(w,part)][g] L[g][pq]
  if (h->Lb) {
    StageTimer tm(h, AFQMC_STAGE_VHS);
    double* Cb[1] = {h->A};
    const int r = run_vhs_tc(h->Cf, h->Ab, h->Lb, Cb, 1, 2 * nw, h->tc_tiles, h->tc_ntile, M, nc, h->st);
    if (r < 0) return fail(h, AFQMC_ERR_CUDA, "vhs (mixed precision): tensor map encode failed");
    h->launches += r;
  } else if (h->cplx && h->A2) {
    StageTimer tm(h, AFQMC_STAGE_VHS);
    const int nf = h->nf;
    double* Cb1[1] = {h->A};
    double* Cb2[1] = {h->A2};
    const int r1 = run_vhs_ws_scatter(h->Cf, h->Ks, Cb1, 1, 2 * nw, h->vhs_tiles, h->vhs_ntile, M, nf, false, h->st, nc);
    const int r2 = run_vhs_ws_scatter(h->Cf + nf, h->Ks + (size_t)nf * MM, Cb2, 1, 2 * nw, h->vhs_tiles, h->vhs_ntile, M, nf,
                                      false, h->st, nc);
    if (r1 < 0 || r2 < 0) return fail(h, AFQMC_ERR_CUDA, "vhs (complex): tensor map encode failed");
    h->launches += r1 + r2;
    h->launches += run_add_antisym(h->A, h->A2, 2 * nw, M, h->st);
  } else if (h->ws_vhs) {
    StageTimer tm(h, AFQMC_STAGE_VHS);
    const int r = run_vhs_ws(h->Cf, h->Lpk ? h->Lpk : h->L, h->A, h->vhs_tiles, h->vhs_ntile, M, nc, 2 * nw,
                             h->Lpk != nullptr, h->st);
    if (r < 0) return fail(h, AFQMC_ERR_CUDA, "vhs: tensor map encode failed");
    h->launches += r;
  } else {
    StageTimer tm(h, AFQMC_STAGE_VHS);
    GemmArgs g = gemm_args();
    g.A = h->Cf; g.lda = nc; g.B = h->L; g.ldb = MM; g.C = h->A; g.ldc = MM;
    g.M = 2 * nw; g.N = (int)MM; g.K = nc;
    h->launches += run_gemm(GEMM_KN, g, h->st);
  }
  return propagate_device(h, W, wt, h->cfb, h->cmf, dt, nw);
}

// a10: thin QR with R_ii > 0 of every walker block, in place; h->detR [nw][nblk] = prod diag R per block
void reortho_device(afqmc_handle* h, double* W, int nw, bool fix_overlaps) {
  StageTimer tm(h, AFQMC_STAGE_REORTHO);
  QRArgs q;
  q.W = W; q.detR = h->detR; q.M = h->M; q.Nt = h->Nt; q.nblk = h->nblk;
  for (int b = 0; b < 2; ++b) { q.off[b] = h->off[b]; q.ns[b] = h->ns[b]; }
  q.shifted = h->qr_shifted;
  h->launches += run_fill(h->detR, 1.0, (long)nw * h->nblk, h->st);
  h->launches += run_cholqr_pass(q, nw, h->st);       // all passes in one launch (small.cu)
  if (fix_overlaps) h->launches += run_ovlp_div_detR(h->ovlp, h->detR, h->nblk, h->rhf, nw, h->st);
}

// a9-a10: overlap of the propagated walkers, phaseless weight update, re-orthonormalisation on schedule
int finish_step_device(afqmc_handle* h, double* W, double* wt, const double* cfb, const double* cmf, double dt, int nw) {
  const int M = h->M, Nt = h->Nt;
  // a9: new overlap and weights
  {
    StageTimer tm(h, AFQMC_STAGE_OVERLAP_NEW);
    h->launches += run_overlap_theta(ot_args(h, W, h->det_new, 0, 0), nw, h->st);
  }
  {
    StageTimer tm(h, AFQMC_STAGE_WEIGHT);
    WeightArgs a;
    a.det_old = h->det_old; a.det_new = h->det_new; a.cfb = cfb; a.cmf = cmf;
    a.weights = wt; a.ovlp = h->ovlp; a.nblk = h->nblk; a.rhf = h->rhf;
    a.expo = -dt * (h->E_const - h->e_shift);
    a.dt = dt; a.ehyb_bound = h->p.ehyb_bound;
    h->launches += run_weight_update(a, nw, h->st);
  }
  // a10: re-orthonormalisation
  h->step_count += 1;
  h->last_nw = nw;
  if (h->p.ortho_every > 0 && h->step_count % h->p.ortho_every == 0) reortho_device(h, W, nw, true);
  return AFQMC_OK;
}

// a6-a10 with A = V_HS in h->A and the overlap determinants of the incoming walkers in h->det_old
int propagate_device(afqmc_handle* h, double* W, double* wt, const double* cfb, const double* cmf, double dt, int nw) {
  const int M = h->M, Nt = h->Nt;
  const long MM = (long)M * M;
  if (!(h->dt_cached == dt)) build_E1(h, dt);
  if (h->Abf) {
    // mixed precision: a6, a7, a8 as bf16 x 3 GEMMs on tcgen05; the running sum of the Taylor terms is FP64
    const int N2 = 2 * Nt;
    int r = 0, bad = 0;
    {
      StageTimer tm(h, AFQMC_STAGE_ONE_BODY);       // Acc = T_0 = phi + (E1 - 1) phi; the split T_0 goes straight to Tb1
      h->launches += taylor_tc_prepare_T(W, h->Tb0, nw, M, N2, h->st);
      r = taylor_tc_apply(h->E1b, true, h->Tb0, h->Tb1, h->Acc, true, W, 1.0, nw, M, N2, h->st);
      bad |= r < 0; h->launches += r > 0 ? r : 0;
    }
    {
      StageTimer tm(h, AFQMC_STAGE_TAYLOR);         // Acc += A^n T_0 / n!
      h->launches += taylor_tc_prepare_A(h->A, h->Abf, nw, M, h->st);
      void* tb[2] = {h->Tb1, h->Tb0};
      for (int n = 1; n <= h->K; ++n) {
        const int cur = (n - 1) & 1;
        r = taylor_tc_apply(h->Abf, false, tb[cur], n < h->K ? tb[cur ^ 1] : nullptr, h->Acc, false, nullptr, 1.0 / n, nw, M, N2,
                            h->st);
        bad |= r < 0; h->launches += r > 0 ? r : 0;
      }
    }
    {
      StageTimer tm(h, AFQMC_STAGE_ONE_BODY);       // phi = Acc + (E1 - 1) Acc, into the caller's walkers
      h->launches += taylor_tc_prepare_T(h->Acc, h->Tb0, nw, M, N2, h->st);
      r = taylor_tc_apply(h->E1b, true, h->Tb0, nullptr, W, true, h->Acc, 1.0, nw, M, N2, h->st);
      bad |= r < 0; h->launches += r > 0 ? r : 0;
    }
    if (bad) return fail(h, AFQMC_ERR_CUDA, "propagation (mixed precision): tensor map encode failed");
    return finish_step_device(h, W, wt, cfb, cmf, dt, nw);
  }
  // a6: T0 = Acc = E1 phi
  const long wstride = (long)M * 2 * Nt;
  {
    StageTimer tm(h, AFQMC_STAGE_ONE_BODY);
    GemmArgs g = gemm_args();
    g.A = h->E1; g.lda = M; g.sA = 0; g.B = W; g.ldb = 2 * Nt; g.sB = wstride;
    g.C = h->T0; g.C2 = h->Acc; g.mode = 2; g.ldc = 2 * Nt; g.sC = wstride;
    g.M = M; g.N = 2 * Nt; g.K = M; g.batch = nw;
    int r = -1;
    if (h->cplx) {       // complex E1 (planar): the planar-complex GEMM of the Taylor terms with a shared operand
      g.A = h->E1c; g.A2 = h->E1c + MM;
      if (h->ws)
        r = run_gemm_ws_kn(h->E1c, M, MM, 0, true, W, 2 * Nt, wstride, h->T0, h->Acc, 2 * Nt, wstride, M, 2 * Nt, M,
                           nw, 1.0, 2, h->st, &h->sk);
      h->launches += r > 0 ? r : run_gemm(GEMM_CPLX_KN, g, h->st);
    } else {
      if (h->ws)
        r = run_gemm_ws_kn(h->E1, M, 0, 0, false, W, 2 * Nt, wstride, h->T0, h->Acc, 2 * Nt, wstride, M, 2 * Nt, M,
                           nw, 1.0, 2, h->st, &h->sk);
      h->launches += r > 0 ? r : run_gemm(GEMM_KN, g, h->st);
    }
  }
  // a7: T_n = A T_{n-1} / n, Acc += T_n
  {
    StageTimer tm(h, AFQMC_STAGE_TAYLOR);
    double *Tp = h->T0, *Tn = h->T1;
    for (int n = 1; n <= h->K; ++n) {
      GemmArgs g = gemm_args();
      g.A = h->A; g.A2 = h->A + MM; g.lda = M; g.sA = 2 * MM; g.B = Tp; g.ldb = 2 * Nt; g.sB = wstride;
      g.C = Tn; g.C2 = h->Acc; g.mode = 1; g.ldc = 2 * Nt; g.sC = wstride;
      g.M = M; g.N = 2 * Nt; g.K = M; g.batch = nw; g.alpha = 1.0 / n;
      int r = -1;
      if (h->ws)
        r = run_gemm_ws_kn(h->A, M, MM, 2 * MM, true, Tp, 2 * Nt, wstride, Tn, h->Acc, 2 * Nt, wstride, M, 2 * Nt,
                           M, nw, 1.0 / n, 1, h->st, &h->sk);
      h->launches += r > 0 ? r : run_gemm(GEMM_CPLX_KN, g, h->st);
      std::swap(Tp, Tn);
    }
  }
  // a8: phi = E1 Acc, written into the caller's walkers
  {
    StageTimer tm(h, AFQMC_STAGE_ONE_BODY);
    GemmArgs g = gemm_args();
    g.A = h->E1; g.lda = M; g.sA = 0; g.B = h->Acc; g.ldb = 2 * Nt; g.sB = wstride;
    g.C = W; g.ldc = 2 * Nt; g.sC = wstride; g.M = M; g.N = 2 * Nt; g.K = M; g.batch = nw;
    int r = -1;
    if (h->cplx) {
      g.A = h->E1c; g.A2 = h->E1c + MM;
      if (h->ws)
        r = run_gemm_ws_kn(h->E1c, M, MM, 0, true, h->Acc, 2 * Nt, wstride, W, nullptr, 2 * Nt, wstride, M, 2 * Nt, M,
                           nw, 1.0, 0, h->st, &h->sk);
      h->launches += r > 0 ? r : run_gemm(GEMM_CPLX_KN, g, h->st);
    } else {
      if (h->ws)
        r = run_gemm_ws_kn(h->E1, M, 0, 0, false, h->Acc, 2 * Nt, wstride, W, nullptr, 2 * Nt, wstride, M, 2 * Nt, M,
                           nw, 1.0, 0, h->st, &h->sk);
      h->launches += r > 0 ? r : run_gemm(GEMM_KN, g, h->st);
    }
  }
  return finish_step_device(h, W, wt, cfb, cmf, dt, nw);
}

// Comb on device buffers: map -> h->pmap, weights in place, walkers and stored overlaps permuted.
void population_control_device(afqmc_handle* h, double* W, double* wt, const double* xi_dev, int nw) {
  StageTimer tm(h, AFQMC_STAGE_POP_CONTROL);
  const long row_bytes = (long)h->M * h->Nt * 16;
  h->launches += run_comb(wt, xi_dev, h->cum, h->pmap, nw, h->st);
  h->launches += run_permute_rows(W, h->T0, h->pmap, row_bytes, nw, h->st);
  if (h->last_nw == nw) h->launches += run_permute_rows(h->ovlp, h->ovlp_tmp, h->pmap, 16, nw, h->st);
}

void estimators_device(afqmc_handle* h, const double* wt, const double* E, double* out4, int nw) {
  StageTimer tm(h, AFQMC_STAGE_ESTIMATORS);
  h->launches += run_estimators(wt, E, out4, nw, h->st);
}

// The block loop on device buffers: stream ordered, no host synchronisation (capturable).
int block_body_device(afqmc_handle* h, double* W, double* wt, const double* aux, const double* xi, double dt, int nw,
                      int n_steps, int pop_every, double* E, double* est) {
  int j = 0;
  for (int s = 0; s < n_steps; ++s) {
    const int rc = step_device(h, W, wt, aux + (size_t)s * nw * h->nf, dt, nw);
    if (rc != AFQMC_OK) return rc;
    if (pop_every > 0 && (s + 1) % pop_every == 0) population_control_device(h, W, wt, xi + j++, nw);
  }
  if (E) {
    const int rc = local_energy_device(h, W, E, nw);
    if (rc != AFQMC_OK) return rc;
    if (est) estimators_device(h, wt, E, est, nw);
  }
  return AFQMC_OK;
}

// afqmc_run_block on device buffers: the first call with a given argument set runs eagerly
// (it also pays every one-off cudaFuncSetAttribute), the second is captured into a CUDA graph,
// later ones replay it.  The graph bakes in the pointers, sizes, dt and the phase of the
// re-orthonormalisation schedule, which together form the key.
int block_graphed(afqmc_handle* h, double* W, double* wt, const double* aux, const double* xi, double dt, int nw,
                  int n_steps, int pop_every, double* E, double* est) {
  if (!h->graph_on || h->prof)
    return block_body_device(h, W, wt, aux, xi, dt, nw, n_steps, pop_every, E, est);
  if (!(h->dt_cached == dt)) build_E1(h, dt);
  const int phase = h->p.ortho_every > 0 ? (int)(h->step_count % h->p.ortho_every) : 0;
  afqmc_handle::BlockGraph* g = nullptr;
  for (auto& c : h->graphs)
    if (c.W == W && c.wt == wt && c.x == aux && c.xi == xi && c.E == E && c.est == est && c.nw == nw &&
        c.n_steps == n_steps && c.pop_every == pop_every && c.ortho_phase == phase && c.dt == dt)
      g = &c;
  if (!g) {
    if (h->graphs.size() >= 8) {
      if (h->graphs.front().exec) cudaGraphExecDestroy(h->graphs.front().exec);
      h->graphs.erase(h->graphs.begin());
    }
    h->graphs.push_back({W, wt, aux, xi, E, est, nw, n_steps, pop_every, phase, dt, 0, nullptr, 0});
    g = &h->graphs.back();
  }
  if (g->exec) {
    if (cudaGraphLaunch(g->exec, h->st) != cudaSuccess) return check_cuda(h, "cudaGraphLaunch");
    h->step_count += n_steps;
    h->last_nw = nw;
    h->launches += g->launches;
    h->graph_replays += 1;
    return AFQMC_OK;
  }
  if (g->seen++ == 0) return block_body_device(h, W, wt, aux, xi, dt, nw, n_steps, pop_every, E, est);
  // capture
  const long sc0 = h->step_count;
  const int64_t l0 = h->launches;
  cudaGraph_t graph = nullptr;
  if (cudaStreamBeginCapture(h->st, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
    cudaGetLastError();
    h->graph_on = false;
    return block_body_device(h, W, wt, aux, xi, dt, nw, n_steps, pop_every, E, est);
  }
  const int rc = block_body_device(h, W, wt, aux, xi, dt, nw, n_steps, pop_every, E, est);
  const cudaError_t ce = cudaStreamEndCapture(h->st, &graph);
  cudaGraphExec_t exec = nullptr;
  if (rc != AFQMC_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    cudaGetLastError();
    if (graph) cudaGraphDestroy(graph);
    h->graph_on = false;          // fall back to eager launches for good
    h->step_count = sc0;
    h->launches = l0;
    return block_body_device(h, W, wt, aux, xi, dt, nw, n_steps, pop_every, E, est);
  }
  cudaGraphDestroy(graph);
  g->exec = exec;
  g->launches = h->launches - l0;
  if (cudaGraphLaunch(exec, h->st) != cudaSuccess) return check_cuda(h, "cudaGraphLaunch");
  h->graph_replays += 1;
  return AFQMC_OK;
}

}  // namespace

extern "C" {

const char* afqmc_last_error(const afqmc_handle* h) { return h ? h->err.c_str() : g_create_err.c_str(); }

void afqmc_destroy(afqmc_handle* h) {
  if (!h) return;
  DevGuard dg_(h->dev);
  cudaStreamSynchronize(h->st);
  for (void* p : h->allocs)
    if (p) cudaFree(p);
  for (auto& g : h->graphs)
    if (g.exec) cudaGraphExecDestroy(g.exec);
  for (auto& br : h->ev_pending) { cudaEventDestroy(br.a); cudaEventDestroy(br.b); }
  for (cudaEvent_t e : h->ev_free) cudaEventDestroy(e);
  if (h->own_stream) cudaStreamDestroy(h->st);
  delete h;
}

int32_t afqmc_create(const double* h1, const double* L_chol, const double* trial, const afqmc_params* p,
                     afqmc_handle** out) {
  if (out) *out = nullptr;
  if (!h1 || !L_chol || !trial || !p || !out) return fail(nullptr, AFQMC_ERR_INVALID, "null argument");
  if (p->struct_size != (int32_t)sizeof(afqmc_params)) return fail(nullptr, AFQMC_ERR_INVALID, "bad struct_size");
  if (p->M <= 0 || p->n_chol <= 0 || p->max_walkers <= 0 || p->n_alpha <= 0 || p->n_beta < 0 ||
      p->ortho_every < 0 || p->taylor_order < 0 || (p->pack_chol != 0 && p->pack_chol != 1) || (p->mixed_precision != 0 && p->mixed_precision != 1) || (p->complex_chol != 0 && p->complex_chol != 1) || (p->walker_kind != 0 && p->walker_kind != 1) ||
      (p->complex_trial != 0 && p->complex_trial != 1) || (p->tuning_flags & ~1) != 0 || !(p->xbar_bound >= 0.0) || !(p->ehyb_bound >= 0.0))
    return fail(nullptr, AFQMC_ERR_INVALID, "bad parameter value");
  if (p->walker_kind == 0 && p->n_alpha != p->n_beta) return fail(nullptr, AFQMC_ERR_DIMS, "RHF walkers need n_alpha == n_beta");
  if (p->walker_kind == 1 && p->n_beta <= 0) return fail(nullptr, AFQMC_ERR_DIMS, "UHF walkers need n_beta > 0");
  if (p->n_alpha > p->M || p->n_beta > p->M) return fail(nullptr, AFQMC_ERR_DIMS, "more occupied orbitals than basis functions");
  if (p->taylor_order > kMaxTaylor) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "taylor_order > 16");
  if (p->n_alpha > kMaxOcc || p->n_beta > kMaxOcc) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "occupied block > 64 columns");
  // the per-walker kernels put the walker index in gridDim.y / gridDim.z (limit 65535)
  if (p->max_walkers > 65535) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "max_walkers > 65535");
  if (p->kernel_path < 0 || p->kernel_path > 3) return fail(nullptr, AFQMC_ERR_INVALID, "kernel_path must be 0, 1, 2 or 3");
  const bool cplx = p->complex_chol == 1;
  const bool ctrial = p->complex_trial == 1;
  if (ctrial && !cplx) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "complex_trial needs complex_chol = 1");
  const int nvec = cplx ? 4 * p->n_chol : p->n_chol;      // real planes the kernels run over
  if ((long)nvec * p->M >= (1L << 31)) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "n_chol * M >= 2^31");
  if (cplx && (p->pack_chol || p->mixed_precision || p->group_size > 1))
    return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "complex_chol cannot be combined with pack_chol, mixed_precision or a group");
  if (!is_device_ptr(L_chol)) return fail(nullptr, AFQMC_ERR_INVALID, "L_chol must be a device pointer");
  const int G = p->group_size > 0 ? p->group_size : 1;
  if (G > kMaxGroup) return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "group_size > 8");
  if (p->group_rank < 0 || p->group_rank >= G) return fail(nullptr, AFQMC_ERR_INVALID, "group_rank out of range");
  if (G > 1 && (p->M % 2 != 0 || p->n_chol % 2 != 0))
    return fail(nullptr, AFQMC_ERR_UNSUPPORTED, "a distributed Hamiltonian needs even M and an even local n_chol (TMA strides)");

  const int ldev = device_of(L_chol);
  DevGuard dg_(ldev >= 0 ? ldev : 0);
  // The inputs may have been produced on ANY stream of the caller (torch fills the 55 GB tensor on its own
  // stream); the handle's stream is non-blocking, so nothing orders it after them.  Setup is a one-off: drain
  // the device once so that L_chol, h1 and trial are complete before the first kernel reads them.
  if (cudaDeviceSynchronize() != cudaSuccess)
    return fail(nullptr, AFQMC_ERR_CUDA, std::string("device not ready at afqmc_create: ") + cudaGetErrorString(cudaGetLastError()));
  afqmc_handle* h = new (std::nothrow) afqmc_handle();
  if (!h) return fail(nullptr, AFQMC_ERR_ALLOC, "host allocation failed");
  h->p = *p;
  h->dev = ldev >= 0 ? ldev : 0;
  h->M = p->M; h->n_chol = nvec; h->maxw = p->max_walkers;
  h->cplx = cplx; h->nf = cplx ? 2 * p->n_chol : p->n_chol;
  h->G = G; h->rank = p->group_rank; h->mwg = G * p->max_walkers;
  h->shard_ready = G == 1;
  h->K = p->taylor_order ? p->taylor_order : 6;
  h->rhf = p->walker_kind == 0;
  h->sf = h->rhf ? 2.0 : 1.0;
  h->nblk = h->rhf ? 1 : 2;
  h->off[0] = 0; h->ns[0] = p->n_alpha;
  h->off[1] = p->n_alpha; h->ns[1] = h->rhf ? 0 : p->n_beta;
  h->Nt = h->rhf ? p->n_alpha : p->n_alpha + p->n_beta;
  h->L = L_chol;
  // TMA needs 16-byte global strides: even M.  kernel_path = 1 forces the cp.async kernels that odd M
  // takes anyway (tests cover both paths on the same inputs); a group always needs the TMA kernels.
  h->ws = (p->M % 2 == 0) && (G > 1 || p->kernel_path != 1);
  if (p->stream) {
    h->st = (cudaStream_t)p->stream;
  } else {
    if (cudaStreamCreateWithFlags(&h->st, cudaStreamNonBlocking) != cudaSuccess) {
      delete h;
      return fail(nullptr, AFQMC_ERR_CUDA, "cudaStreamCreate failed");
    }
    h->own_stream = true;
  }
  const int M = h->M, Nt = h->Nt, nc = h->n_chol, mw = h->maxw, mwg = h->mwg;
  const long MM = (long)M * M;
  auto bail = [&](int code, const std::string& msg) {
    std::string m2 = msg;
    afqmc_destroy(h);
    return fail(nullptr, code, m2);
  };

  // ---- host copies of the small inputs, checks, P_tot ------------------------------------
  std::vector<double> th((size_t)M * Nt), hh((size_t)MM), hi, ti;     // ti: Im psi (complex trial)
  if (ctrial) {
    std::vector<double> tc((size_t)2 * M * Nt);
    if (cudaMemcpy(tc.data(), trial, tc.size() * 8, cudaMemcpyDefault) != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "copy of the trial failed");
    ti.resize(th.size());
    for (size_t i = 0; i < th.size(); ++i) { th[i] = tc[2 * i]; ti[i] = tc[2 * i + 1]; }
  } else if (cudaMemcpy(th.data(), trial, th.size() * 8, cudaMemcpyDefault) != cudaSuccess) {
    return bail(AFQMC_ERR_CUDA, "copy of the trial failed");
  }
  if (cplx) {                                  // complex Hermitian h1: planes
    std::vector<double> hc((size_t)2 * MM);
    if (cudaMemcpy(hc.data(), h1, hc.size() * 8, cudaMemcpyDefault) != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "copy of h1 failed");
    hi.resize(MM);
    for (long i = 0; i < MM; ++i) { hh[i] = hc[2 * i]; hi[i] = hc[2 * i + 1]; }
    // the planes of the 2n Hermitian matrices replace the caller's tensor from here on
    h->Ks = dalloc(h, (size_t)nvec * MM);
    if (!h->Ks) return bail(AFQMC_ERR_ALLOC, "device allocation failed (Hermitian planes)");
    h->launches += run_hermitian_planes(L_chol, h->Ks, M, p->n_chol, h->st);
    h->L = h->Ks;
  } else if (cudaMemcpy(hh.data(), h1, hh.size() * 8, cudaMemcpyDefault) != cudaSuccess) {
    return bail(AFQMC_ERR_CUDA, "copy of h1 failed");
  }
  for (int b = 0; b < h->nblk; ++b)
    for (int i = 0; i < h->ns[b]; ++i)
      for (int j = i; j < h->ns[b]; ++j) {
        double s = 0.0, si = 0.0;        // (psi^+ psi)_ij = sum_q conj(psi_qi) psi_qj
        for (int q = 0; q < M; ++q) {
          const size_t qi = (size_t)q * Nt + h->off[b] + i, qj = (size_t)q * Nt + h->off[b] + j;
          s += th[qi] * th[qj];
          if (ctrial) { s += ti[qi] * ti[qj]; si += th[qi] * ti[qj] - ti[qi] * th[qj]; }
        }
        if (!(fabs(s - (i == j ? 1.0 : 0.0)) <= 1e-10) || !(fabs(si) <= 1e-10))
          return bail(AFQMC_ERR_TRIAL, "trial columns are not orthonormal to 1e-10");
      }
  // P = psi psi^+ = Pr + i Pi (times the spin factor); Pi = 0 for a real trial.  tT: planes (Re psi^T, -Im psi^T)
  std::vector<double> P((size_t)MM, 0.0), Pi, tT((size_t)(ctrial ? 2 : 1) * Nt * M);
  for (int q = 0; q < M; ++q)
    for (int i = 0; i < Nt; ++i) {
      tT[(size_t)i * M + q] = th[(size_t)q * Nt + i];
      if (ctrial) tT[(size_t)Nt * M + (size_t)i * M + q] = -ti[(size_t)q * Nt + i];
    }
  for (int i = 0; i < Nt; ++i)
    for (int a = 0; a < M; ++a) {
      const double f = h->sf * tT[(size_t)i * M + a];
      if (f == 0.0) continue;
      for (int c = 0; c < M; ++c) P[(size_t)a * M + c] += f * tT[(size_t)i * M + c];
    }
  if (ctrial) {
    Pi.assign((size_t)MM, 0.0);
    const double* nI = tT.data() + (size_t)Nt * M;           // -Im psi^T
    for (int i = 0; i < Nt; ++i)
      for (int a = 0; a < M; ++a) {
        const double ra = tT[(size_t)i * M + a], ia = -nI[(size_t)i * M + a];
        for (int c = 0; c < M; ++c) {
          const double rc = tT[(size_t)i * M + c], ic = -nI[(size_t)i * M + c];
          P[(size_t)a * M + c] += h->sf * ia * ic;             // Re (psi_a conj(psi_c)) = ra rc + ia ic
          Pi[(size_t)a * M + c] += h->sf * (ia * rc - ra * ic); // Im (psi_a conj(psi_c))
        }
      }
  }

  // ---- device constants ---------------------------------------------------------------
  h->h1 = dalloc(h, MM); h->trial = dalloc(h, (size_t)M * Nt); h->trialT = dalloc(h, tT.size());
  h->Lrot = dalloc(h, (size_t)nc * Nt * M); h->hrot = dalloc(h, (size_t)Nt * M); h->m = dalloc(h, nc);
  h->hmod = dalloc(h, MM); h->E1 = dalloc(h, MM); h->Xs = dalloc(h, MM); h->Pa = dalloc(h, MM); h->Pb = dalloc(h, MM);
  double* dP = dalloc(h, MM);
  double* mL = dalloc(h, MM);
  if (!h->h1 || !h->trial || !h->trialT || !h->Lrot || !h->hrot || !h->m || !h->hmod || !h->E1 || !h->Xs ||
      !h->Pa || !h->Pb || !dP || !mL)
    return bail(AFQMC_ERR_ALLOC, "device allocation failed (constants)");
  cudaMemcpyAsync(h->h1, hh.data(), MM * 8, cudaMemcpyHostToDevice, h->st);
  cudaMemcpyAsync(h->trial, th.data(), th.size() * 8, cudaMemcpyHostToDevice, h->st);
  cudaMemcpyAsync(h->trialT, tT.data(), tT.size() * 8, cudaMemcpyHostToDevice, h->st);
  cudaMemcpyAsync(dP, P.data(), MM * 8, cudaMemcpyHostToDevice, h->st);

  // m_g = tr(L_g P_tot); mL = sum_g m_g L_g
  h->launches += run_mean_field(h->L, dP, h->m, M, nc, h->st);
  if (ctrial) {
    // tr(K P) = <Re K, Pr> + <Im K, Pi> (elementwise; Im K and Pi antisymmetric): add the second term to the nf
    // entries that carry m.  mL is free scratch until run_sum_mL below.
    h->trial_im = dalloc(h, (size_t)M * Nt);
    double* mtmp = dalloc(h, h->nf);
    if (!h->trial_im || !mtmp) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex trial)");
    cudaMemcpyAsync(h->trial_im, ti.data(), ti.size() * 8, cudaMemcpyHostToDevice, h->st);
    cudaMemcpyAsync(mL, Pi.data(), MM * 8, cudaMemcpyHostToDevice, h->st);
    h->launches += run_mean_field(h->L + (size_t)h->nf * MM, mL, mtmp, M, h->nf, h->st);
    h->launches += run_add(h->m, h->m, mtmp, h->nf, h->st);
    cudaStreamSynchronize(h->st);           // Pi (host vector) and mtmp are released below
    dfree_one(h, mtmp);
  }
  h->launches += run_sum_mL(h->L, h->m, mL, M, nc, h->st);
  // sum_g L_g L_g = L2d^T L2d with L2d = L viewed as [(g,k)][M] (L_g symmetric), split over K
  {
    const int tiles = ((M + 127) / 128) * ((M + 127) / 128);
    int split = (296 + tiles - 1) / tiles;
    if (split > 32) split = 32;
    if (split < 1) split = 1;
    double* part = dalloc(h, (size_t)split * MM);
    if (!part) return bail(AFQMC_ERR_ALLOC, "device allocation failed (setup)");
    GemmArgs g = gemm_args();
    g.A = h->L; g.lda = M; g.B = h->L; g.ldb = M; g.C = part; g.ldc = M;
    g.M = M; g.N = M; g.K = nc * M; g.splitK = split; g.sCsplit = MM;
    h->launches += run_gemm(GEMM_KMKN, g, h->st);
    if (G > 1) {
      // this member's share of h_mod - h1 = sum over ITS gamma of (-1/2 L_g L_g + m_g L_g); the
      // group sum is added to h1 in afqmc_shard_setup_finish
      h->hmod_part = dalloc(h, MM);
      if (!h->hmod_part) return bail(AFQMC_ERR_ALLOC, "device allocation failed (setup)");
      h->launches += run_fill(h->Xs, 0.0, MM, h->st);
      h->launches += run_hmod(h->Xs, part, split, mL, h->hmod_part, M, h->st);
      h->launches += run_scale_copy(h->hmod, h->h1, 1.0, MM, h->st);    // placeholder until the finish
    } else {
      h->launches += run_hmod(h->h1, part, split, mL, h->hmod, M, h->st);
    }
    cudaStreamSynchronize(h->st);
    dfree_one(h, part);
  }
  // half rotation: Lrot[g] = trial^T L_g ; hrot = trial^T h1
  {
    GemmArgs g = gemm_args();
    g.A = h->trialT; g.lda = M; g.sA = 0; g.B = h->L; g.ldb = M; g.sB = MM;
    g.C = h->Lrot; g.ldc = M; g.sC = (long)Nt * M; g.M = Nt; g.N = M; g.K = M; g.batch = nc;
    // grid.z limit: batch in chunks of 32768
    for (int b0 = 0; b0 < nc; b0 += 32768) {
      GemmArgs gg = g;
      gg.B = g.B + (size_t)b0 * MM; gg.C = g.C + (size_t)b0 * Nt * M; gg.batch = std::min(32768, nc - b0);
      h->launches += run_gemm(GEMM_KN, gg, h->st);
    }
    if (ctrial) {
      // psi^+ K = (Re psi^T Kr + Im psi^T Ki) + i (Re psi^T Ki - Im psi^T Kr): the same batched GEMM with the plane
      // -Im psi^T, then the planes are combined in place (Lrot[0:nf] real part, Lrot[nf:2nf] imaginary part)
      double* t2 = dalloc(h, (size_t)nc * Nt * M);
      if (!t2) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex trial half rotation)");
      for (int b0 = 0; b0 < nc; b0 += 32768) {
        GemmArgs gg = g;
        gg.A = h->trialT + (size_t)Nt * M;
        gg.B = g.B + (size_t)b0 * MM; gg.C = t2 + (size_t)b0 * Nt * M; gg.batch = std::min(32768, nc - b0);
        h->launches += run_gemm(GEMM_KN, gg, h->st);
      }
      const long half = (long)h->nf * Nt * M;
      h->launches += run_add_scaled(h->Lrot, h->Lrot, t2 + half, -1.0, half, h->st);
      h->launches += run_add_scaled(h->Lrot + half, h->Lrot + half, t2, 1.0, half, h->st);
      cudaStreamSynchronize(h->st);
      dfree_one(h, t2);
    }
    GemmArgs g2 = gemm_args();
    g2.A = h->trialT; g2.lda = M; g2.B = h->h1; g2.ldb = M; g2.C = h->hrot; g2.ldc = M;
    g2.M = Nt; g2.N = M; g2.K = M;
    h->launches += run_gemm(GEMM_KN, g2, h->st);
  }
  // E_const and the 1-norm of h_mod on the host
  {
    std::vector<double> mh(nc), hm((size_t)MM);
    cudaMemcpyAsync(mh.data(), h->m, nc * 8, cudaMemcpyDeviceToHost, h->st);
    cudaMemcpyAsync(hm.data(), h->hmod, MM * 8, cudaMemcpyDeviceToHost, h->st);
    if (cudaStreamSynchronize(h->st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, std::string("setup kernels failed: ") + cudaGetErrorString(cudaPeekAtLastError()));
    double s = 0.0;
    const int nm = cplx ? h->nf : nc;          // complex: tr(Im K P) = 0, only the nf real planes carry m
    for (int g = 0; g < nm; ++g) s += mh[g] * mh[g];
    h->E_const = -0.5 * s;
    h->Ec_part = h->E_const;
    if (cplx) h->hm_host.assign(hm.begin(), hm.end());
    double n1 = 0.0;
    for (int c = 0; c < M; ++c) {
      double cs = 0.0;
      for (int r = 0; r < M; ++r) cs += fabs(hm[(size_t)r * M + c]);
      if (cs > n1) n1 = cs;
    }
    h->hmod_norm1 = n1;
  }
  if (cplx) {
    // Im h_mod = Im h1 - 1/2 (Z - Z^T) + sum_g m_g Im K_g,  Z = sum_g (Re K_g)^T (Im K_g)   (cplx.cu, header)
    const int nf = h->nf;
    const double* Ki = h->Ks + (size_t)nf * MM;
    const int tiles = ((M + 127) / 128) * ((M + 127) / 128);
    int split = (296 + tiles - 1) / tiles;
    if (split > 32) split = 32;
    if (split < 1) split = 1;
    double* part = dalloc(h, (size_t)split * MM);
    h->hrot_i = dalloc(h, (size_t)Nt * M);
    h->Lrot_sum = dalloc(h, (size_t)nf * Nt * M);
    h->E1c = dalloc(h, (size_t)2 * MM);
    if (!part || !h->hrot_i || !h->Lrot_sum || !h->E1c) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex setup)");
    GemmArgs g = gemm_args();
    g.A = h->Ks; g.lda = M; g.B = Ki; g.ldb = M; g.C = part; g.ldc = M;
    g.M = M; g.N = M; g.K = nf * M; g.splitK = split; g.sCsplit = MM;
    h->launches += run_gemm(GEMM_KMKN, g, h->st);
    h->launches += run_sum_mL(Ki, h->m, mL, M, nf, h->st);
    std::vector<double> zp((size_t)split * MM), mli((size_t)MM);
    cudaMemcpyAsync(zp.data(), part, zp.size() * 8, cudaMemcpyDeviceToHost, h->st);
    cudaMemcpyAsync(mli.data(), mL, MM * 8, cudaMemcpyDeviceToHost, h->st);
    // hrot_i = trial^T Im h1 (Xs is free scratch here); Lrot_sum = Lrot_re + Lrot_im for the cross term of tr(TT)
    cudaMemcpyAsync(h->Xs, hi.data(), MM * 8, cudaMemcpyHostToDevice, h->st);
    GemmArgs g2 = gemm_args();
    g2.A = h->trialT; g2.lda = M; g2.B = h->Xs; g2.ldb = M; g2.C = h->hrot_i; g2.ldc = M;
    g2.M = Nt; g2.N = M; g2.K = M;
    h->launches += run_gemm(GEMM_KN, g2, h->st);
    if (ctrial) {
      // psi^+ h = (Re psi^T hr + Im psi^T hi) + i (Re psi^T hi - Im psi^T hr).  The two Nt x M products go through
      // Lrot_sum (nf Nt M doubles, nf >= 2, filled only below): Nt exceeds M for UHF walkers past half filling, so an
      // M x M buffer such as Pa / Pb is too small for them.
      double* s0 = h->Lrot_sum;
      double* s1 = h->Lrot_sum + (size_t)Nt * M;
      GemmArgs g3 = g2;
      g3.A = h->trialT + (size_t)Nt * M; g3.C = s0;                     // -Im psi^T hi
      h->launches += run_gemm(GEMM_KN, g3, h->st);
      g3.B = h->h1; g3.C = s1;                                          // -Im psi^T hr
      h->launches += run_gemm(GEMM_KN, g3, h->st);
      h->launches += run_add_scaled(h->hrot, h->hrot, s0, -1.0, (long)Nt * M, h->st);
      h->launches += run_add_scaled(h->hrot_i, h->hrot_i, s1, 1.0, (long)Nt * M, h->st);
    }
    h->launches += run_add(h->Lrot_sum, h->Lrot, h->Lrot + (size_t)nf * Nt * M, (long)nf * Nt * M, h->st);
    if (cudaStreamSynchronize(h->st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "complex setup kernels failed");
    h->hm_host.resize((size_t)2 * MM);
    for (int r = 0; r < M; ++r)
      for (int c = 0; c < M; ++c) {
        double z = 0.0, zt = 0.0;
        for (int k = 0; k < split; ++k) {
          z += zp[(size_t)k * MM + (size_t)r * M + c];
          zt += zp[(size_t)k * MM + (size_t)c * M + r];
        }
        h->hm_host[MM + (size_t)r * M + c] = hi[(size_t)r * M + c] - 0.5 * (z - zt) + mli[(size_t)r * M + c];
      }
    h->hmod_c = dalloc(h, (size_t)2 * MM);
    h->cbuf = dalloc(h, (size_t)8 * MM);
    if (!h->hmod_c || !h->cbuf) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex expm)");
    cudaMemcpy(h->hmod_c, h->hm_host.data(), (size_t)2 * MM * 8, cudaMemcpyHostToDevice);
    {   // 1-norm of the complex h_mod for the scaling
      double n1 = 0.0;
      for (int c = 0; c < M; ++c) {
        double cs = 0.0;
        for (int r = 0; r < M; ++r) cs += hypot(h->hm_host[(size_t)r * M + c], h->hm_host[MM + (size_t)r * M + c]);
        if (cs > n1) n1 = cs;
      }
      h->hmod_norm1 = n1;
    }
    dfree_one(h, part);
    // The derivation needs sum_g (B_g x A_g - A_g x B_g) = 0 (a tensor with (ps|qr) = (qr|ps)).  Probe it with two
    // random Hermitian matrices U, V:  sum_g [tr(B_g U) tr(A_g V) - tr(A_g U) tr(B_g V)] must vanish, where
    // tr(K U) = sum Re K . Re U + sum Im K . Im U for Hermitian K, U.
    {
      const int n = p->n_chol;
      std::vector<double> pr((size_t)2 * MM), tr_all((size_t)4 * nc);
      double* probe = dalloc(h, 2 * MM);
      double* tro = dalloc(h, (size_t)4 * nc);
      if (!probe || !tro) return bail(AFQMC_ERR_ALLOC, "device allocation failed (symmetry probe)");
      uint64_t lcg = 0x9E3779B97F4A7C15ull;
      auto rnd = [&]() { lcg = lcg * 6364136223846793005ull + 1442695040888963407ull; return ((lcg >> 11) * (1.0 / 9007199254740992.0)) - 0.5; };
      for (int t = 0; t < 2; ++t) {
        for (int r = 0; r < M; ++r)
          for (int c = r; c < M; ++c) {
            const double a = rnd(), b = r == c ? 0.0 : rnd();
            pr[(size_t)r * M + c] = pr[(size_t)c * M + r] = a;                      // Re U symmetric
            pr[MM + (size_t)r * M + c] = b; pr[MM + (size_t)c * M + r] = -b;         // Im U antisymmetric
          }
        cudaMemcpyAsync(probe, pr.data(), 2 * MM * 8, cudaMemcpyHostToDevice, h->st);
        h->launches += run_mean_field(h->Ks, probe, tro + (size_t)(2 * t) * nc, M, nc, h->st);          // . Re U
        h->launches += run_mean_field(h->Ks, probe + MM, tro + (size_t)(2 * t + 1) * nc, M, nc, h->st); // . Im U
        cudaStreamSynchronize(h->st);
      }
      cudaMemcpy(tr_all.data(), tro, tr_all.size() * 8, cudaMemcpyDeviceToHost);
      // tr(K_g U) = (Re planes . Re U)[g] + (Im planes . Im U)[nf + g]
      auto trK = [&](int t, int g) { return tr_all[(size_t)(2 * t) * nc + g] + tr_all[(size_t)(2 * t + 1) * nc + nf + g]; };
      double f = 0.0, scale = 0.0;
      for (int g = 0; g < n; ++g) {
        const double aU = trK(0, g), bU = trK(0, n + g), aV = trK(1, g), bV = trK(1, n + g);
        f += bU * aV - aU * bV;
        scale += fabs(bU * aV) + fabs(aU * bV);
      }
      dfree_one(h, probe);
      dfree_one(h, tro);
      if (!(fabs(f) <= 1e-9 * scale + 1e-300))
        return bail(AFQMC_ERR_INVALID, "complex_chol: the vectors do not factorise a (ps|qr) = (qr|ps) symmetric tensor");
    }
  }
  dfree_one(h, dP);
  dfree_one(h, mL);

  // ---- workspaces ----------------------------------------------------------------------
  {
    const int tiles = ((2 * mwg + 127) / 128) * ((nc + 127) / 128);
    int split = (296 + tiles - 1) / tiles;
    const int kmax = std::max(1, (Nt * M) / 512);
    if (split > kmax) split = kmax;
    if (split > 16) split = 16;
    if (split < 1) split = 1;
    h->fb_split = h->ws ? gemm_ws_nk_split(2 * mwg, nc, Nt * M, 16) : split;
  }
  const size_t wsz = (size_t)mw * M * 2 * Nt;
  h->det_old = dalloc(h, (size_t)mw * 2 * 2); h->det_new = dalloc(h, (size_t)mw * 2 * 2);
  // Theta^T of every walker the force bias / exchange kernels see: the whole group's in a
  // distributed Hamiltonian (member r's walkers in slot r, written by member r)
  h->ThT = dalloc(h, (size_t)G * wsz); h->Xp = dalloc(h, (size_t)h->fb_split * 2 * mwg * nc);
  h->X = dalloc(h, (size_t)2 * mwg * nc); h->Cf = dalloc(h, (size_t)2 * mwg * nc);
  h->cfb = dalloc(h, 2 * mwg); h->cmf = dalloc(h, 2 * mwg);
  h->A = dalloc(h, (size_t)mw * 2 * MM);
  h->T0 = dalloc(h, wsz); h->T1 = dalloc(h, wsz); h->Acc = dalloc(h, wsz);
  h->ovlp = dalloc(h, 2 * mw); h->detR = dalloc(h, 2 * mw);
  for (int b = 0; b < h->nblk; ++b) {
    const int G = h->ws ? exchange_ws_group_size(h->ns[b], M) : exchange_group_size(h->ns[b]);
    h->exgroups[b] = (nc + G - 1) / G;
    h->expart[b] = dalloc(h, (size_t)h->exgroups[b] * mwg * 2);
  }
  h->Xe = dalloc(h, (size_t)nc * mwg * 2); h->e1 = dalloc(h, (size_t)mw * 2 * 2);
  h->Obuf = dalloc(h, (size_t)mw * Nt * 2 * Nt); h->Aop = dalloc(h, (size_t)mw * 4 * Nt * Nt);
  if (!h->Obuf || !h->Aop) return bail(AFQMC_ERR_ALLOC, "device allocation failed (overlap operands)");
  // kernel_path = 2: the one-kernel overlap / Theta route (tests); a group member always takes the GEMM route
  h->ot_gemm = h->ws && (G > 1 || p->kernel_path != 2);
  h->small = p->kernel_path == 0 && !cplx && !p->mixed_precision && !p->pack_chol && G == 1 &&
             small_path_fits(M, Nt, std::max(h->ns[0], h->ns[1]), nc);
  if (G > 1) {
    h->theta_buf = h->ThT;
    h->a_slots = dalloc(h, (size_t)G * mw * 2 * MM);
    h->scal_slots = dalloc(h, (size_t)G * mw * 4);
    h->e_slots = dalloc(h, (size_t)G * mw * 2);
    h->scal_sum = dalloc(h, (size_t)mw * 4);
    h->e1zero = dalloc(h, (size_t)mwg * 2 * 2);
    h->Etmp = dalloc(h, (size_t)mwg * 6);
    h->setup_buf = dalloc(h, (size_t)MM + 2);
    if (!h->a_slots || !h->scal_slots || !h->e_slots || !h->scal_sum || !h->e1zero || !h->Etmp || !h->setup_buf)
      return bail(AFQMC_ERR_ALLOC, "device allocation failed (distributed-Hamiltonian slots)");
    cudaMemsetAsync(h->e1zero, 0, (size_t)mwg * 2 * 2 * 8, h->st);
    h->peer[0][h->rank] = h->theta_buf; h->peer[1][h->rank] = h->a_slots;
    h->peer[2][h->rank] = h->scal_slots; h->peer[3][h->rank] = h->e_slots;
  }
  h->stW = dalloc(h, wsz); h->stWt = dalloc(h, mw); h->stX = dalloc(h, (size_t)mw * nc); h->stE = dalloc(h, (size_t)mw * 6);
  h->cum = dalloc(h, mw); h->xi_dev = dalloc(h, 4); h->est_dev = dalloc(h, 4); h->ovlp_tmp = dalloc(h, 2 * mw);
  h->pmap = (int*)dalloc(h, (mw + 1) / 2 + 1);
  h->qr_shifted = (int*)dalloc(h, 1);
  if (h->ws) {
    const int nsm = sm_count_current();
    h->sk.part_doubles = (size_t)nsm * 2 * 2 * ((2 * Nt + 7) / 8 + 1) * 2 * 256;
    h->sk.part = dalloc(h, h->sk.part_doubles);
    h->sk.flag = (int*)dalloc(h, (nsm + 1) / 2 + 1);
    h->sk.flags = nsm;
    h->sk.force = p->tuning_flags & 1;
    if (!h->sk.part || !h->sk.flag) return bail(AFQMC_ERR_ALLOC, "device allocation failed (stream-K scratch)");
    cudaMemsetAsync(h->sk.flag, 0, (size_t)nsm * sizeof(int), h->st);
  }
  if (h->qr_shifted) cudaMemsetAsync(h->qr_shifted, 0, 8, h->st);
  if (!h->cum || !h->xi_dev || !h->est_dev || !h->ovlp_tmp || !h->pmap || !h->qr_shifted)
    return bail(AFQMC_ERR_ALLOC, "device allocation failed (population control)");
  if (!h->det_old || !h->det_new || !h->ThT || !h->Xp || !h->X || !h->Cf || !h->cfb || !h->cmf || !h->A ||
      !h->T0 || !h->T1 || !h->Acc || !h->ovlp || !h->detR || !h->expart[0] || (h->nblk > 1 && !h->expart[1]) ||
      !h->Xe || !h->e1 || !h->stW || !h->stWt || !h->stX || !h->stE)
    return bail(AFQMC_ERR_ALLOC, "device allocation failed (workspaces)");

  h->ws_vhs = !cplx && h->ws && vhs_ws_usable(M, nc, h->L, h->Cf, h->A);   // Im K is antisymmetric: dense route
  if (cplx && h->ws && vhs_ws_usable(M, h->nf, h->L, h->Cf, h->A)) {
    // V_HS as two symmetric-half runs: Re planes (symmetric sum) and Im planes (antisymmetric sum, sign fixed below)
    std::vector<int> tl;
    h->vhs_ntile = vhs_ws_tile_list(M, &tl);
    h->vhs_tiles = (int*)dalloc(h, (tl.size() + 1) / 2 + 1);
    h->A2 = dalloc(h, (size_t)mw * 2 * MM);
    if (!h->vhs_tiles || !h->A2) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex V_HS)");
    if (cudaMemcpy(h->vhs_tiles, tl.data(), tl.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "tile list upload failed");
  }
  if (cplx) {
    h->e1i = dalloc(h, (size_t)mw * 2 * 2);
    h->Xe_s = dalloc(h, (size_t)h->nf * mwg * 2);
    bool ok = h->e1i && h->Xe_s;
    for (int b = 0; b < h->nblk; ++b) {
      const int G = h->ws ? exchange_ws_group_size(h->ns[b], M, true) : exchange_group_size(h->ns[b]);
      h->exgroups_c[b] = (h->nf + G - 1) / G;
      for (int k = 0; k < 2; ++k) {
        h->expart_c[k][b] = dalloc(h, (size_t)h->exgroups_c[b] * mwg * 2);
        ok = ok && h->expart_c[k][b];
      }
    }
    if (!ok) return bail(AFQMC_ERR_ALLOC, "device allocation failed (complex energy buffers)");
  }
  if (h->ws_vhs) {
    std::vector<int> tl;
    h->vhs_ntile = vhs_ws_tile_list(M, &tl);
    h->vhs_tiles = (int*)dalloc(h, (tl.size() + 1) / 2 + 1);
    if (!h->vhs_tiles) return bail(AFQMC_ERR_ALLOC, "device allocation failed (tile list)");
    if (cudaMemcpy(h->vhs_tiles, tl.data(), tl.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "tile list upload failed");
  }

  if (p->pack_chol) {
    if (!h->ws_vhs) return bail(AFQMC_ERR_UNSUPPORTED, "pack_chol needs even M and n_chol (TMA strides)");
    h->Lpk = dalloc(h, vhs_ws_packed_doubles(h->vhs_ntile, nc));
    if (!h->Lpk) return bail(AFQMC_ERR_ALLOC, "device allocation failed (packed Cholesky tensor)");
    h->launches += run_pack_tiles(h->L, h->Lpk, h->vhs_tiles, h->vhs_ntile, M, nc, h->st);
  }

  if (p->mixed_precision) {
    if (!h->ws_vhs) return bail(AFQMC_ERR_UNSUPPORTED, "mixed_precision needs even M and n_chol");
    if (p->pack_chol) return bail(AFQMC_ERR_INVALID, "mixed_precision keeps its own split tiles: pack_chol must be 0");
    {
      std::vector<int> tl;
      h->tc_ntile = vhs_tc_tile_list(M, &tl);
      h->tc_tiles = (int*)dalloc(h, (tl.size() + 1) / 2 + 1);
      if (!h->tc_tiles) return bail(AFQMC_ERR_ALLOC, "device allocation failed (tile list)");
      if (cudaMemcpy(h->tc_tiles, tl.data(), tl.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
        return bail(AFQMC_ERR_CUDA, "tile list upload failed");
    }
    h->Lb = dalloc(h, (vhs_tc_L_elems(h->tc_ntile, nc) * 2 + 7) / 8);
    h->Ab = dalloc(h, (vhs_tc_cf_elems(2 * mwg, nc) * 2 + 7) / 8);
    if (!h->Lb || !h->Ab) return bail(AFQMC_ERR_ALLOC, "device allocation failed (split Cholesky tensor)");
    h->launches += run_vhs_tc_split_L(h->L, h->Lb, h->tc_tiles, h->tc_ntile, M, nc, h->st);
    {   // force bias: split Lrot once; Theta^T is split per step
      h->fb_tc_nsplit = fb_tc_split(2 * mwg, nc, Nt * M, 16);
      if (h->fb_tc_nsplit > h->fb_split) {
        dfree_one(h, h->Xp);
        h->Xp = dalloc(h, (size_t)h->fb_tc_nsplit * 2 * mwg * nc);
        if (!h->Xp) return bail(AFQMC_ERR_ALLOC, "device allocation failed (force-bias partials)");
      }
      h->Lrb = dalloc(h, (fb_tc_L_elems(nc, Nt * M) * 2 + 7) / 8);
      h->Tfb = dalloc(h, (fb_tc_T_elems(2 * mwg, Nt * M) * 2 + 7) / 8);
      if (!h->Lrb || !h->Tfb) return bail(AFQMC_ERR_ALLOC, "device allocation failed (split half-rotated tensor)");
      h->launches += run_fb_tc_split_L(h->Lrot, h->Lrb, nc, Nt * M, h->st);
    }
    if (taylor_tc_usable(2 * Nt)) {
      const size_t ta = (taylor_tc_A_elems(mw, M) * 2 + 7) / 8, tt = (taylor_tc_T_elems(mw, M, 2 * Nt) * 2 + 7) / 8;
      h->Abf = dalloc(h, ta); h->Tb0 = dalloc(h, tt); h->Tb1 = dalloc(h, tt);
      h->E1b = dalloc(h, (taylor_tc_A_elems(1, M) * 2 + 7) / 8);
      if (!h->Abf || !h->Tb0 || !h->Tb1 || !h->E1b) return bail(AFQMC_ERR_ALLOC, "device allocation failed (split Taylor operands)");
      cudaMemsetAsync(h->Tb0, 0, tt * 8, h->st);      // the zero padding of k and n is never written again
      cudaMemsetAsync(h->Tb1, 0, tt * 8, h->st);
    }
  }

  // ---- E_shift = trial energy ---------------------------------------------------------------
  {
    std::vector<double> wt((size_t)M * Nt * 2, 0.0);
    for (size_t i = 0; i < th.size(); ++i) { wt[2 * i] = th[i]; if (ctrial) wt[2 * i + 1] = ti[i]; }
    cudaMemcpyAsync(h->stW, wt.data(), wt.size() * 8, cudaMemcpyHostToDevice, h->st);
    if (local_energy_device(h, h->stW, h->stE, 1) != AFQMC_OK) return bail(AFQMC_ERR_CUDA, h->err);
    double e[6];
    cudaMemcpyAsync(e, h->stE, 48, cudaMemcpyDeviceToHost, h->st);
    if (cudaStreamSynchronize(h->st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, std::string("trial energy failed: ") + cudaGetErrorString(cudaPeekAtLastError()));
    h->e_trial = e[0];
    h->e1b_trial = e[2];
    h->e2trial_part = e[4];
  }
  if (G > 1 && !h->ws_vhs) return bail(AFQMC_ERR_UNSUPPORTED, "a distributed Hamiltonian needs the TMA V_HS kernel (16-byte aligned L)");
  h->e_shift = p->e_shift_auto ? h->e_trial : p->e_shift;
  if (h->Lpk || h->Lb || h->cplx) {  // the caller's tensor is not touched after this point
    if (cudaStreamSynchronize(h->st) != cudaSuccess || cudaGetLastError() != cudaSuccess)
      return bail(AFQMC_ERR_CUDA, "packing / splitting the Cholesky tensor failed");
    h->L = h->cplx ? h->Ks : nullptr;
  }
  *out = h;
  return AFQMC_OK;
}

int32_t afqmc_exchange_plan(int32_t ns, int32_t M, int32_t pair, char* out, int32_t n) {
  if (ns < 1 || ns > afq::kMaxOcc || M < ns || !out || n < 1) return AFQMC_ERR_INVALID;
  afq::exchange_ws_describe(ns, M, pair != 0, out, n);
  return (int32_t)(afq::exchange_ws_efficiency(ns, M, pair != 0) * 1e6);
}

int32_t afqmc_exchange_plan_pin(int32_t ns, int32_t M, int32_t pair, int32_t warps, int32_t mi, int32_t ni, int32_t wm,
                                int32_t G, int32_t Wn, int32_t epi_warps) {
  if (ns < 1 || ns > afq::kMaxOcc || M < ns) return AFQMC_ERR_INVALID;
  return afq::exchange_ws_pin(ns, M, pair != 0, warps, mi, ni, wm, G, Wn, epi_warps) ? AFQMC_OK : AFQMC_ERR_UNSUPPORTED;
}

int32_t afqmc_exchange_plan_unpin(int32_t ns, int32_t M, int32_t pair) {
  if (ns > afq::kMaxOcc || (ns > 0 && M < ns)) return AFQMC_ERR_INVALID;
  afq::exchange_ws_unpin(ns, M, pair != 0);
  return AFQMC_OK;
}

int32_t afqmc_step(afqmc_handle* h, void* walkers, double* weights, const double* aux_fields, double dt, int32_t nw) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (h->G > 1) return fail(h, AFQMC_ERR_UNSUPPORTED, "distributed-Hamiltonian handle: use the afqmc_shard_* phases");
  if (!walkers || !weights || !aux_fields) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, AFQMC_ERR_INVALID, "dt must be positive");
  const size_t wlen = (size_t)nw * h->M * 2 * h->Nt;
  const bool hostW = !is_device_ptr(walkers), hostWt = !is_device_ptr(weights), hostX = !is_device_ptr(aux_fields);
  double* W = (double*)walkers;
  double* wt = weights;
  const double* x = aux_fields;
  if (hostW) { to_device(h, h->stW, walkers, wlen); W = h->stW; }
  if (hostWt) { to_device(h, h->stWt, weights, nw); wt = h->stWt; }
  if (hostX) { to_device(h, h->stX, aux_fields, (size_t)nw * h->nf); x = h->stX; }
  {
    const int rc = step_device(h, W, wt, x, dt, nw);
    if (rc != AFQMC_OK) return rc;
  }
  if (hostW) cudaMemcpyAsync(walkers, W, wlen * 8, cudaMemcpyDeviceToHost, h->st);
  if (hostWt) cudaMemcpyAsync(weights, wt, (size_t)nw * 8, cudaMemcpyDeviceToHost, h->st);
  if (hostW || hostWt) {
    if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_step");
  }
  return check_cuda(h, "afqmc_step");
}

int32_t afqmc_local_energy(afqmc_handle* h, const void* walkers, void* E_out, int32_t nw) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (h->G > 1) return fail(h, AFQMC_ERR_UNSUPPORTED, "distributed-Hamiltonian handle: use the afqmc_shard_* phases");
  if (!walkers || !E_out) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  const size_t wlen = (size_t)nw * h->M * 2 * h->Nt;
  const bool hostW = !is_device_ptr(walkers), hostE = !is_device_ptr(E_out);
  const double* W = (const double*)walkers;
  double* E = (double*)E_out;
  if (hostW) { to_device(h, h->stW, walkers, wlen); W = h->stW; }
  if (hostE) E = h->stE;
  {
    const int rc = local_energy_device(h, W, E, nw);
    if (rc != AFQMC_OK) return rc;
  }
  if (hostE) {
    cudaMemcpyAsync(E_out, E, (size_t)nw * 48, cudaMemcpyDeviceToHost, h->st);
    if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_local_energy");
  }
  return check_cuda(h, "afqmc_local_energy");
}

int32_t afqmc_population_control(afqmc_handle* h, void* walkers, double* weights, const double* xi, int32_t nw,
                                 int32_t* map_out) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (h->G > 1) return fail(h, AFQMC_ERR_UNSUPPORTED, "distributed-Hamiltonian handle: use the afqmc_shard_* phases");
  if (!walkers || !weights || !xi) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  const size_t wlen = (size_t)nw * h->M * 2 * h->Nt;
  const bool hostW = !is_device_ptr(walkers), hostWt = !is_device_ptr(weights), hostXi = !is_device_ptr(xi);
  if (hostXi && !(xi[0] >= 0.0 && xi[0] < 1.0)) return fail(h, AFQMC_ERR_INVALID, "xi must be in [0, 1)");
  double* W = (double*)walkers;
  double* wt = weights;
  const double* xd = xi;
  if (hostW) { to_device(h, h->stW, walkers, wlen); W = h->stW; }
  if (hostWt) { to_device(h, h->stWt, weights, nw); wt = h->stWt; }
  if (hostXi) { to_device(h, h->xi_dev, xi, 1); xd = h->xi_dev; }
  population_control_device(h, W, wt, xd, nw);
  bool sync = false;
  if (hostW) { cudaMemcpyAsync(walkers, W, wlen * 8, cudaMemcpyDeviceToHost, h->st); sync = true; }
  if (hostWt) { cudaMemcpyAsync(weights, wt, (size_t)nw * 8, cudaMemcpyDeviceToHost, h->st); sync = true; }
  if (map_out) {
    cudaMemcpyAsync(map_out, h->pmap, (size_t)nw * 4, cudaMemcpyDefault, h->st);
    if (!is_device_ptr(map_out)) sync = true;
  }
  if (sync && cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_population_control");
  return check_cuda(h, "afqmc_population_control");
}

int32_t afqmc_estimators(afqmc_handle* h, const double* weights, const void* E, double* est_out, int32_t nw) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (!weights || !E || !est_out) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  const bool hostWt = !is_device_ptr(weights), hostE = !is_device_ptr(E), hostO = !is_device_ptr(est_out);
  const double* wt = weights;
  const double* Ed = (const double*)E;
  if (hostWt) { to_device(h, h->stWt, weights, nw); wt = h->stWt; }
  if (hostE) { to_device(h, h->stE, E, (size_t)nw * 6); Ed = h->stE; }
  double* out = hostO ? h->est_dev : est_out;
  estimators_device(h, wt, Ed, out, nw);
  if (hostO) {
    cudaMemcpyAsync(est_out, out, 32, cudaMemcpyDeviceToHost, h->st);
    if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_estimators");
  }
  return check_cuda(h, "afqmc_estimators");
}

int32_t afqmc_run_block(afqmc_handle* h, void* walkers, double* weights, const double* aux_fields, const double* xi,
                        double dt, int32_t nw, int32_t n_steps, int32_t pop_every, void* E_out, double* est_out) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (h->G > 1) return fail(h, AFQMC_ERR_UNSUPPORTED, "distributed-Hamiltonian handle: use the afqmc_shard_* phases");
  if (!walkers || !weights || !aux_fields) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  if (n_steps <= 0 || pop_every < 0) return fail(h, AFQMC_ERR_INVALID, "bad n_steps / pop_every");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, AFQMC_ERR_INVALID, "dt must be positive");
  const int n_pop = pop_every > 0 ? n_steps / pop_every : 0;
  if (n_pop > 0 && !xi) return fail(h, AFQMC_ERR_INVALID, "xi is needed when pop_every > 0");
  const int nc = h->nf;
  const size_t wlen = (size_t)nw * h->M * 2 * h->Nt;
  const bool hostW = !is_device_ptr(walkers), hostWt = !is_device_ptr(weights), hostX = !is_device_ptr(aux_fields);
  const bool hostXi = n_pop > 0 && !is_device_ptr(xi);
  const bool hostE = E_out && !is_device_ptr(E_out), hostO = est_out && !is_device_ptr(est_out);
  if (hostXi)
    for (int j = 0; j < n_pop; ++j)
      if (!(xi[j] >= 0.0 && xi[j] < 1.0)) return fail(h, AFQMC_ERR_INVALID, "xi must be in [0, 1)");
  double* W = (double*)walkers;
  double* wt = weights;
  if (!hostW && !hostWt && !hostX && !hostXi && !hostE && !hostO) {
    double* E = E_out ? (double*)E_out : (est_out ? h->stE : nullptr);
    const int rc = block_graphed(h, W, wt, aux_fields, xi, dt, nw, n_steps, pop_every, E, est_out);
    return rc != AFQMC_OK ? rc : check_cuda(h, "afqmc_run_block");
  }
  if (hostW) { to_device(h, h->stW, walkers, wlen); W = h->stW; }
  if (hostWt) { to_device(h, h->stWt, weights, nw); wt = h->stWt; }
  int j = 0;
  for (int s = 0; s < n_steps; ++s) {
    const double* x = aux_fields + (size_t)s * nw * nc;
    if (hostX) { to_device(h, h->stX, x, (size_t)nw * nc); x = h->stX; }
    const int rc = step_device(h, W, wt, x, dt, nw);
    if (rc != AFQMC_OK) return rc;
    if (pop_every > 0 && (s + 1) % pop_every == 0) {
      const double* xd = xi + j;
      // a host xi is staged one value at a time: the copy is stream ordered before its comb
      if (hostXi) { to_device(h, h->xi_dev + (j & 3), xi + j, 1); xd = h->xi_dev + (j & 3); }
      population_control_device(h, W, wt, xd, nw);
      ++j;
    }
  }
  if (E_out || est_out) {
    double* E = (hostE || !E_out) ? h->stE : (double*)E_out;
    const int rc = local_energy_device(h, W, E, nw);
    if (rc != AFQMC_OK) return rc;
    if (est_out) estimators_device(h, wt, E, hostO ? h->est_dev : est_out, nw);
    if (hostE) cudaMemcpyAsync(E_out, E, (size_t)nw * 48, cudaMemcpyDeviceToHost, h->st);
    if (hostO) cudaMemcpyAsync(est_out, h->est_dev, 32, cudaMemcpyDeviceToHost, h->st);
  }
  if (hostW) cudaMemcpyAsync(walkers, W, wlen * 8, cudaMemcpyDeviceToHost, h->st);
  if (hostWt) cudaMemcpyAsync(weights, wt, (size_t)nw * 8, cudaMemcpyDeviceToHost, h->st);
  if (hostW || hostWt || hostE || hostO) {
    if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_run_block");
  }
  return check_cuda(h, "afqmc_run_block");
}

int32_t afqmc_get_overlaps(afqmc_handle* h, void* ovlp_out) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (!ovlp_out) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (h->last_nw <= 0) return fail(h, AFQMC_ERR_INVALID, "no step has been taken");
  const bool host = !is_device_ptr(ovlp_out);
  cudaMemcpyAsync(ovlp_out, h->ovlp, (size_t)h->last_nw * 16, cudaMemcpyDefault, h->st);
  if (host && cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_get_overlaps");
  return check_cuda(h, "afqmc_get_overlaps");
}

int32_t afqmc_reorthonormalise(afqmc_handle* h, void* walkers, double* detR_out, int32_t nw) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (!walkers) return fail(h, AFQMC_ERR_INVALID, "null argument");
  if (nw <= 0 || nw > h->maxw) return fail(h, AFQMC_ERR_DIMS, "nw out of range");
  const size_t wlen = (size_t)nw * h->M * 2 * h->Nt;
  const bool hostW = !is_device_ptr(walkers);
  double* W = (double*)walkers;
  if (hostW) { to_device(h, h->stW, walkers, wlen); W = h->stW; }
  reortho_device(h, W, nw, h->last_nw == nw);
  bool sync = false;
  if (hostW) { cudaMemcpyAsync(walkers, W, wlen * 8, cudaMemcpyDeviceToHost, h->st); sync = true; }
  if (detR_out) {
    cudaMemcpyAsync(detR_out, h->detR, (size_t)nw * h->nblk * 8, cudaMemcpyDefault, h->st);
    sync = sync || !is_device_ptr(detR_out);
  }
  if (sync && cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_reorthonormalise");
  return check_cuda(h, "afqmc_reorthonormalise");
}

int64_t afqmc_qr_shifted_passes(afqmc_handle* h) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  int v = 0;
  cudaMemcpyAsync(&v, h->qr_shifted, sizeof(int), cudaMemcpyDeviceToHost, h->st);
  if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_qr_shifted_passes");
  return v;
}

int32_t afqmc_get_constants(afqmc_handle* h, double* out3) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (!out3) return fail(h, AFQMC_ERR_INVALID, "null argument");
  out3[0] = h->E_const; out3[1] = h->e_shift; out3[2] = h->e_trial;
  return AFQMC_OK;
}

int64_t afqmc_debug_read(afqmc_handle* h, int32_t which, double* out) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  const double* src = nullptr;
  int64_t n = 0;
  const long MM = (long)h->M * h->M;
  const int nw = h->last_nw;
  switch (which) {
    case 0: src = h->X; n = (int64_t)2 * nw * h->nf; break;
    case 1: src = h->A; n = (int64_t)2 * nw * MM; break;
    case 2: src = h->E1; n = MM; break;
    case 3: src = h->hmod; n = MM; break;
    case 4: src = h->m; n = h->n_chol; break;
    case 5: src = h->Lrot; n = (int64_t)h->n_chol * h->Nt * h->M; break;
    default: return fail(h, AFQMC_ERR_INVALID, "unknown debug array");
  }
  if (!out) return n;
  cudaMemcpyAsync(out, src, (size_t)n * 8, cudaMemcpyDefault, h->st);
  if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_debug_read");
  int rc = check_cuda(h, "afqmc_debug_read");
  return rc == AFQMC_OK ? n : rc;
}

int64_t afqmc_set_block_graph(afqmc_handle* h, int32_t on) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (on >= 0) h->graph_on = on != 0;
  return h->graph_replays;
}

int32_t afqmc_set_profiling(afqmc_handle* h, int32_t on) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  h->prof = on != 0;
  return AFQMC_OK;
}

int32_t afqmc_get_stage_times(afqmc_handle* h, double* ms_out, int64_t* count_out, int32_t reset) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  if (!ms_out) return fail(h, AFQMC_ERR_INVALID, "null argument");
  cudaError_t e = cudaStreamSynchronize(h->st);
  if (e != cudaSuccess) return fail(h, AFQMC_ERR_CUDA, std::string("get_stage_times: ") + cudaGetErrorString(e));
  for (auto& br : h->ev_pending) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, br.a, br.b) == cudaSuccess) {
      h->stage_ms[br.stage] += ms;
      h->stage_n[br.stage] += 1;
    } else {
      cudaGetLastError();
    }
    h->ev_free.push_back(br.a);
    h->ev_free.push_back(br.b);
  }
  h->ev_pending.clear();
  for (int i = 0; i < AFQMC_STAGE_COUNT; ++i) {
    ms_out[i] = h->stage_ms[i];
    if (count_out) count_out[i] = h->stage_n[i];
    if (reset) { h->stage_ms[i] = 0.0; h->stage_n[i] = 0; }
  }
  return AFQMC_OK;
}

int64_t afqmc_launch_count(const afqmc_handle* h) { return h ? h->launches : -1; }

// ------------------------------------------------------------------ distributed Hamiltonian
#define SHARD_CHECK(h, need_ready)                                                                     \
  if (!h) return AFQMC_ERR_INVALID;                                                                    \
  DevGuard dg_(h->dev);                                                                                \
  if (h->G <= 1) return fail(h, AFQMC_ERR_INVALID, "not a distributed-Hamiltonian handle (group_size <= 1)"); \
  if (need_ready && !h->shard_ready) return fail(h, AFQMC_ERR_INVALID, "afqmc_shard_setup_finish has not been called"); \
  if (need_ready && !h->peers_set) return fail(h, AFQMC_ERR_INVALID, "afqmc_shard_set_peers has not been called");

int32_t afqmc_shard_setup_partial(afqmc_handle* h, double* out) {
  SHARD_CHECK(h, false);
  if (!out) return fail(h, AFQMC_ERR_INVALID, "null argument");
  const long MM = (long)h->M * h->M;
  const double sc[2] = {h->Ec_part, h->e2trial_part};
  cudaMemcpyAsync(h->setup_buf, h->hmod_part, MM * 8, cudaMemcpyDeviceToDevice, h->st);
  cudaMemcpyAsync(h->setup_buf + MM, sc, 16, cudaMemcpyHostToDevice, h->st);
  cudaMemcpyAsync(out, h->setup_buf, (MM + 2) * 8, cudaMemcpyDefault, h->st);
  if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_shard_setup_partial");
  return check_cuda(h, "afqmc_shard_setup_partial");
}

int32_t afqmc_shard_setup_reduce(const double* parts, int32_t n_members, int64_t n, double* out) {
  if (!parts || !out || n_members < 1 || n_members > kMaxGroup || n < 1) return AFQMC_ERR_INVALID;
  for (int64_t i = 0; i < n; ++i) {
    double s = parts[i];
    for (int r = 1; r < n_members; ++r) s += parts[(size_t)r * n + i];     // member order 0 .. G-1
    out[i] = s;
  }
  return AFQMC_OK;
}

int32_t afqmc_shard_setup_finish(afqmc_handle* h, const double* sum) {
  SHARD_CHECK(h, false);
  if (!sum) return fail(h, AFQMC_ERR_INVALID, "null argument");
  const int M = h->M;
  const long MM = (long)M * M;
  std::vector<double> s((size_t)MM + 2), hh((size_t)MM);
  if (cudaMemcpyAsync(s.data(), sum, (MM + 2) * 8, cudaMemcpyDefault, h->st) != cudaSuccess ||
      cudaMemcpyAsync(hh.data(), h->h1, MM * 8, cudaMemcpyDeviceToHost, h->st) != cudaSuccess ||
      cudaStreamSynchronize(h->st) != cudaSuccess)
    return check_cuda(h, "afqmc_shard_setup_finish");
  double n1 = 0.0;
  for (long i = 0; i < MM; ++i) hh[i] += s[i];
  for (int c = 0; c < M; ++c) {
    double cs = 0.0;
    for (int r = 0; r < M; ++r) cs += fabs(hh[(size_t)r * M + c]);
    if (cs > n1) n1 = cs;
  }
  cudaMemcpyAsync(h->hmod, hh.data(), MM * 8, cudaMemcpyHostToDevice, h->st);
  if (cudaStreamSynchronize(h->st) != cudaSuccess) return check_cuda(h, "afqmc_shard_setup_finish");
  h->hmod_norm1 = n1;
  h->E_const = s[MM];
  h->e_trial = h->e1b_trial + s[MM + 1];
  h->e_shift = h->p.e_shift_auto ? h->e_trial : h->p.e_shift;
  h->dt_cached = NAN;
  h->shard_ready = true;
  return check_cuda(h, "afqmc_shard_setup_finish");
}

int32_t afqmc_shard_get_buffers(afqmc_handle* h, uint64_t* out4) {
  SHARD_CHECK(h, false);
  if (!out4) return fail(h, AFQMC_ERR_INVALID, "null argument");
  for (int k = 0; k < 4; ++k) out4[k] = (uint64_t)(uintptr_t)h->peer[k][h->rank];
  return AFQMC_OK;
}

int32_t afqmc_shard_ipc_export(afqmc_handle* h, int32_t which, void* handle64) {
  SHARD_CHECK(h, false);
  if (!handle64 || which < 0 || which > 3) return fail(h, AFQMC_ERR_INVALID, "bad argument");
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
  cudaIpcMemHandle_t mh;
  if (cudaIpcGetMemHandle(&mh, h->peer[which][h->rank]) != cudaSuccess) return check_cuda(h, "cudaIpcGetMemHandle");
  memcpy(handle64, &mh, 64);
  return AFQMC_OK;
}

int32_t afqmc_shard_ipc_open(afqmc_handle* h, const void* handle64, uint64_t* addr_out) {
  if (!handle64 || !addr_out) return AFQMC_ERR_INVALID;
  int cur = 0;
  cudaGetDevice(&cur);
  DevGuard dg_(h ? h->dev : cur);          // the import is mapped on the importing member's device
  cudaIpcMemHandle_t mh;
  memcpy(&mh, handle64, 64);
  void* p = nullptr;
  const cudaError_t e = cudaIpcOpenMemHandle(&p, mh, cudaIpcMemLazyEnablePeerAccess);
  if (e != cudaSuccess) {
    g_create_err = std::string("cudaIpcOpenMemHandle: ") + cudaGetErrorString(e);
    cudaGetLastError();
    return AFQMC_ERR_CUDA;
  }
  *addr_out = (uint64_t)(uintptr_t)p;
  return AFQMC_OK;
}

int32_t afqmc_shard_ipc_close(uint64_t addr) {
  if (!addr) return AFQMC_ERR_INVALID;
  if (cudaIpcCloseMemHandle((void*)(uintptr_t)addr) != cudaSuccess) {
    cudaGetLastError();
    return AFQMC_ERR_CUDA;
  }
  return AFQMC_OK;
}

int32_t afqmc_shard_set_peers(afqmc_handle* h, const uint64_t* addrs) {
  SHARD_CHECK(h, false);
  if (!addrs) return fail(h, AFQMC_ERR_INVALID, "null argument");
  for (int k = 0; k < 4; ++k)
    if (addrs[(size_t)h->rank * 4 + k] != (uint64_t)(uintptr_t)h->peer[k][h->rank])
      return fail(h, AFQMC_ERR_INVALID, "row group_rank of addrs must hold this handle's own buffers");
  for (int r = 0; r < h->G; ++r)
    for (int k = 0; k < 4; ++k) {
      if (!addrs[(size_t)r * 4 + k] || (addrs[(size_t)r * 4 + k] & 15)) return fail(h, AFQMC_ERR_INVALID, "null or misaligned peer buffer");
      h->peer[k][r] = (double*)(uintptr_t)addrs[(size_t)r * 4 + k];
    }
  // members on other devices of this process: the kernels store into their buffers, so peer access must
  // be on (buffers imported through CUDA IPC were opened with cudaIpcMemLazyEnablePeerAccess already)
  for (int r = 0; r < h->G; ++r) {
    const int pd = device_of(h->peer[1][r]);
    if (pd >= 0 && pd != h->dev) {
      int can = 0;
      cudaDeviceCanAccessPeer(&can, h->dev, pd);
      if (!can) return fail(h, AFQMC_ERR_UNSUPPORTED, "no peer access between the devices of the group");
      const cudaError_t e = cudaDeviceEnablePeerAccess(pd, 0);
      if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled)
        return fail(h, AFQMC_ERR_CUDA, std::string("cudaDeviceEnablePeerAccess: ") + cudaGetErrorString(e));
      cudaGetLastError();
    }
  }
  h->peers_set = true;
  return AFQMC_OK;
}

int32_t afqmc_shard_theta(afqmc_handle* h, const void* walkers, int32_t nw, int32_t for_energy) {
  SHARD_CHECK(h, true);
  if (!walkers || !is_device_ptr(walkers)) return fail(h, AFQMC_ERR_INVALID, "walkers must be a device pointer");
  if (nw != h->maxw) return fail(h, AFQMC_ERR_DIMS, "a distributed Hamiltonian needs nw == max_walkers");
  const size_t wsz = (size_t)h->maxw * h->M * 2 * h->Nt;
  double* own = h->theta_buf + (size_t)h->rank * wsz;
  {
    StageTimer tm(h, for_energy ? AFQMC_STAGE_E_THETA : AFQMC_STAGE_OVERLAP_THETA);
    h->launches += run_overlap_theta(ot_args(h, (const double*)walkers, h->det_old, 1, for_energy ? 1 : 0, own), nw, h->st);
  }
  StageTimer tm(h, AFQMC_STAGE_SHARD_EXCHANGE);
  for (int r = 0; r < h->G; ++r)
    if (r != h->rank)
      cudaMemcpyAsync(h->peer[0][r] + (size_t)h->rank * wsz, own, wsz * 8, cudaMemcpyDefault, h->st);
  return check_cuda(h, "afqmc_shard_theta");
}

int32_t afqmc_shard_vhs(afqmc_handle* h, const double* aux_local, double dt, int32_t nw) {
  SHARD_CHECK(h, true);
  if (!aux_local || !is_device_ptr(aux_local)) return fail(h, AFQMC_ERR_INVALID, "aux_local must be a device pointer");
  if (nw != h->maxw) return fail(h, AFQMC_ERR_DIMS, "a distributed Hamiltonian needs nw == max_walkers");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, AFQMC_ERR_INVALID, "dt must be positive");
  const int G = h->G, mw = h->maxw, nwg = G * nw;
  const long MM = (long)h->M * h->M;
  {
    const int rc = force_bias_shift_device(h, aux_local, dt, nwg);
    if (rc != AFQMC_OK) return rc;
  }
  {
    StageTimer tm(h, AFQMC_STAGE_SHARD_EXCHANGE);
    for (int o = 0; o < G; ++o) {
      double* dst = h->peer[2][o] + (size_t)h->rank * mw * 4;
      cudaMemcpyAsync(dst, h->cfb + (size_t)o * nw * 2, (size_t)nw * 16, cudaMemcpyDefault, h->st);
      cudaMemcpyAsync(dst + (size_t)mw * 2, h->cmf + (size_t)o * nw * 2, (size_t)nw * 16, cudaMemcpyDefault, h->st);
    }
  }
  StageTimer tm(h, AFQMC_STAGE_VHS);
  double* Cb[kMaxGroup];
  for (int o = 0; o < G; ++o) Cb[o] = h->peer[1][o] + (size_t)h->rank * mw * 2 * MM;
  const int r = h->Lb ? run_vhs_tc(h->Cf, h->Ab, h->Lb, Cb, G, 2 * nw, h->tc_tiles, h->tc_ntile, h->M, h->n_chol, h->st)
                      : run_vhs_ws_scatter(h->Cf, h->Lpk ? h->Lpk : h->L, Cb, G, 2 * nw, h->vhs_tiles, h->vhs_ntile,
                                           h->M, h->n_chol, h->Lpk != nullptr, h->st);
  if (r < 0) return fail(h, AFQMC_ERR_CUDA, "vhs: tensor map encode failed");
  h->launches += r;
  return check_cuda(h, "afqmc_shard_vhs");
}

int32_t afqmc_shard_propagate(afqmc_handle* h, void* walkers, double* weights, double dt, int32_t nw) {
  SHARD_CHECK(h, true);
  if (!walkers || !weights || !is_device_ptr(walkers) || !is_device_ptr(weights))
    return fail(h, AFQMC_ERR_INVALID, "walkers and weights must be device pointers");
  if (nw != h->maxw) return fail(h, AFQMC_ERR_DIMS, "a distributed Hamiltonian needs nw == max_walkers");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(h, AFQMC_ERR_INVALID, "dt must be positive");
  const int G = h->G, mw = h->maxw;
  const long MM = (long)h->M * h->M;
  {
    StageTimer tm(h, AFQMC_STAGE_SHARD_REDUCE);
    const double *sa[kMaxGroup], *ss[kMaxGroup];
    for (int r = 0; r < G; ++r) {
      sa[r] = h->a_slots + (size_t)r * mw * 2 * MM;
      ss[r] = h->scal_slots + (size_t)r * mw * 4;
    }
    h->launches += run_sum_slots(h->A, sa, G, (long)nw * 2 * MM, h->st);
    h->launches += run_sum_slots(h->scal_sum, ss, G, (long)mw * 4, h->st);
  }
  const int rc = propagate_device(h, (double*)walkers, weights, h->scal_sum, h->scal_sum + (size_t)mw * 2, dt, nw);
  return rc != AFQMC_OK ? rc : check_cuda(h, "afqmc_shard_propagate");
}

int32_t afqmc_shard_energy(afqmc_handle* h, int32_t nw) {
  SHARD_CHECK(h, true);
  if (nw != h->maxw) return fail(h, AFQMC_ERR_DIMS, "a distributed Hamiltonian needs nw == max_walkers");
  const int G = h->G, mw = h->maxw;
  const int rc = energy_from_theta(h, h->e1zero, h->Etmp, G * nw);
  if (rc != AFQMC_OK) return rc;
  StageTimer tm(h, AFQMC_STAGE_SHARD_EXCHANGE);
  for (int o = 0; o < G; ++o)
    h->launches += run_push_e2(h->peer[3][o] + (size_t)h->rank * mw * 2, h->Etmp + (size_t)o * nw * 6, nw, h->st);
  return check_cuda(h, "afqmc_shard_energy");
}

int32_t afqmc_shard_energy_finish(afqmc_handle* h, void* E_out, int32_t nw) {
  SHARD_CHECK(h, true);
  if (!E_out || !is_device_ptr(E_out)) return fail(h, AFQMC_ERR_INVALID, "E_out must be a device pointer");
  if (nw != h->maxw) return fail(h, AFQMC_ERR_DIMS, "a distributed Hamiltonian needs nw == max_walkers");
  StageTimer tm(h, AFQMC_STAGE_SHARD_REDUCE);
  const double* se[kMaxGroup];
  for (int r = 0; r < h->G; ++r) se[r] = h->e_slots + (size_t)r * h->maxw * 2;
  h->launches += run_energy_finish((double*)E_out, h->e1, se, h->G, h->nblk, h->sf, nw, h->st);
  return check_cuda(h, "afqmc_shard_energy_finish");
}

int32_t afqmc_sync(afqmc_handle* h) {
  if (!h) return AFQMC_ERR_INVALID;
  DevGuard dg_(h->dev);
  cudaError_t e = cudaStreamSynchronize(h->st);
  if (e != cudaSuccess) return fail(h, AFQMC_ERR_CUDA, std::string("sync: ") + cudaGetErrorString(e));
  return check_cuda(h, "afqmc_sync");
}

}  // extern "C"
