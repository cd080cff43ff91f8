/* afqmc.h - C ABI of libafqmc: one batched phaseless-AFQMC walker step and the local energy,
 * single-determinant RHF/UHF trial, Cholesky-factorised Hamiltonian, on one B200 (sm_100a).
 *
 * The operations are those of /root/reference/PAPER.md (arXiv 2406.16238) Sec. II,
 * Eqs. (2)-(18); the working formulas derived from them are listed in
 * DESIGN.md ("Readings") and follow SURVEY.md 8(c).
 *
 * Conventions
 *   - All matrices are row-major.  complex128 = two consecutive doubles (re, im).
 *   - H = sum_pq h1[p][q] a+_p a_q + 1/2 sum (ps|qr) a+_p a+_q a_r a_s with
 *     (ps|qr) = sum_g L[g][p][s] L[g][q][r]            (Eqs. 2-3)
 *   - v_g = i L_g (Eq. 6); B(x) = e^{-dt/2 v0} e^{-sqrt(dt) x.v} e^{-dt/2 v0} (Eq. 9),
 *     so the two-body propagator is exp(A), A = -i sqrt(dt) sum_g (x_g - xbar_g) L_g, applied
 *     by a Taylor series of order `taylor_order`.  The force bias is
 *     xbar_g = +i sqrt(dt) (X_g - m_g), X_g = <Psi_T|L_g|phi>/<Psi_T|phi>, m_g = <L_g>_T
 *     (Eq. 14 with the sign that is consistent with Eq. 9: DESIGN.md reading S1).
 *   - Trial columns are [alpha | beta], real, orthonormal per spin block.
 *   - walker_kind 0 (RHF): restricted walkers, ONE block [M][n_alpha] per walker used for
 *     both spins, Nt = n_alpha.  walker_kind 1 (UHF): Nt = n_alpha + n_beta, alpha first.
 *
 * Pointers: every pointer argument says HOST, DEVICE or EITHER.  EITHER pointers are
 * classified with cudaPointerGetAttributes; host buffers are staged through the handle's
 * stream inside the call (and, for outputs, the call returns after the copy back).
 * Calls on device buffers are asynchronous on the handle's stream.
 *
 * Errors: every int32_t entry point returns AFQMC_OK or a negative code; nothing throws or
 * aborts across the ABI.  afqmc_last_error() gives a message for the last failure on that
* handle (or for a failed afqmc_create when passed NULL).  A handle lives on the CUDA device that holds
 * L_chol; every entry point switches to that device for the duration of the call, so handles on
 * different devices can be driven from one host thread.  A walker whose overlap with the
 * trial is zero or non-finite is NOT an error: its weight becomes exactly 0 (Eq. 15,
 * reading S10).
 *
 * Threads: a handle may be driven by one host thread at a time; different handles may be driven from
 * different host threads concurrently.  Process-wide state: the per-device bookkeeping of one-off kernel
 * attributes (mutex protected); the message of a failed afqmc_create, kept per host thread
 * (afqmc_last_error(NULL) returns the calling thread's); the exchange kernel's plan table, which only the tuning
 * hooks afqmc_exchange_plan_pin / _unpin write (mutex protected, and it changes what handles created LATER launch:
 * see there); and the built-in scratch array of afqmc_comb_static (one per GPU, shared by all callers: see there).
 */
#ifndef AFQMC_H_
#define AFQMC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define AFQMC_OK 0
#define AFQMC_ERR_INVALID (-1)     /* null pointer / bad struct_size / bad value          */
#define AFQMC_ERR_DIMS (-2)        /* nw > max_walkers, RHF with n_alpha != n_beta, ...   */
#define AFQMC_ERR_ALLOC (-3)       /* device or host allocation failed                    */
#define AFQMC_ERR_CUDA (-4)        /* CUDA runtime error, see afqmc_last_error            */
#define AFQMC_ERR_TRIAL (-5)       /* trial columns not orthonormal to 1e-10              */
#define AFQMC_ERR_UNSUPPORTED (-6) /* taylor_order > 16, occupied block > 64 columns, ... */

typedef struct afqmc_handle afqmc_handle; /* opaque, library-owned */

typedef struct {
  int32_t struct_size;  /* = sizeof(afqmc_params) */
  int32_t M;            /* orbitals (the paper's N)                          */
  int32_t n_alpha;      /* occupied alpha                                                 */
  int32_t n_beta;       /* occupied beta                                                  */
  int32_t n_chol;       /* Cholesky vectors N_gamma                         */
  int32_t max_walkers;  /* workspaces are sized for this many walkers per call            */
  int32_t walker_kind;  /* 0 RHF restricted walkers, 1 UHF [alpha|beta]                   */
  int32_t taylor_order; /* 0 -> 6; at most 16                                             */
  int32_t ortho_every;  /* 0 never; n: QR after every n-th afqmc_step on this handle      */
  int32_t e_shift_auto; /* 1: E_shift = local energy of the trial; 0: use e_shift         */
  double e_shift;       /* energy shift in the weight, exp(-dt (E_const - E_shift))       */
  void* stream;         /* cudaStream_t to run on; NULL = the library creates its own     */
  int32_t pack_chol;    /* 1: keep a tile-packed copy of the upper triangle of every L_g    */
                        /* (the paper's pack_chol) and stop borrowing L_chol  */
                        /* when afqmc_create returns; needs even M and n_chol               */
  int32_t group_size;   /* distributed Hamiltonian: members G of the group that  */
                        /* shares one Cholesky tensor, 0 or 1 = none, at most 8; with G > 1 L_chol, */
                        /* n_chol describe THIS member's gamma slice and max_walkers its own walkers */
  int32_t group_rank;   /* this member's index in the group, 0 .. G-1                             */
  int32_t mixed_precision; /* 0: everything in double.  1: the propagation - force bias (a3), V_HS      */
                        /* build (a5), one-body half steps (a6, a8), Taylor terms (a7) - in         */
                        /* EMULATED single precision on the tcgen05 tensor                          */
                        /* cores - operands split into three bfloat16 numbers, six partial products, */
                        /* FP32 accumulation in tensor memory -, everything else incl. the local     */
                        /* energy in double ("mixed precision").  The handle keeps the */
                        /* split upper-triangle tiles (6 bytes per kept element) and, as with        */
                        /* pack_chol, stops borrowing L_chol when afqmc_create returns.  Needs even  */
                        /* M and n_chol.  Results agree with the double path to ~1e-6 relative.      */
  int32_t complex_chol; /* 1: complex Cholesky vectors.  L_chol is DEVICE complex128     */
                        /* [n_chol][M][M] with (ps|qr) = sum_g L^g_ps conj(L^g_rq) a (ps|qr) = (qr|ps)      */
                        /* symmetric tensor, h1 is EITHER complex128 [M][M] Hermitian; trial: see complex_trial. */
                        /* The handle works with the 2 n_chol Hermitian matrices A_g = (L_g + L_g^+)/2,      */
                        /* B_g = (L_g - L_g^+)/(2i): aux_fields is [nw][2 n_chol] (fields of the A_g first), */
                        /* L_chol is not referenced after afqmc_create; a set that does not factorise a      */
                        /* symmetric tensor is rejected (AFQMC_ERR_INVALID).  Not combinable with pack_chol, */
                        /* mixed_precision or group_size > 1.                                                */
  int32_t kernel_path;  /* 0: the TMA warp-specialised kernels wherever the shapes allow (even M), the cp.async    */
                        /* kernels otherwise.  1: force the cp.async kernels (what odd M runs; lets a test cover   */
                        /* them at even M on the same inputs).  2: the one-kernel overlap / Theta route instead of */
                        /* the batched DMMA GEMMs.  3: as 0 but without the one-kernel step / local energy that 0  */
                        /* picks for systems whose walker fits one CTA's shared memory (M <= 64, occupied blocks   */
                        /* <= 16, n_chol <= 2048; c1).  Results agree to rounding; ignored for group_size > 1.     */
  int32_t complex_trial; /* 1: `trial` is complex128 [M][Nt] (PAPER.md:219 gives the trial no dtype; PAPER.md:328:   */
                        /* magnetic fields, spin-orbit coupling, Bloch orbitals).  <Psi_T| carries conj(psi):       */
                        /* O = psi^+ phi, Lrot = psi^+ K, hrot = psi^+ h, P = psi psi^+, m_g = tr(K_g P) (real).    */
                        /* Needs complex_chol = 1 (a real tensor is passed as complex vectors with zero imaginary  */
                        /* part; half of the 2 n_chol fields then multiply zero matrices).                          */
  int32_t tuning_flags; /* 0 (default).  Bit 0: use stream-K in the batched Taylor / one-body GEMMs whenever the tile  */
                        /* count leaves a partial last wave, also where the library's cost rule would not (lets a     */
                        /* test reach that code at sizes where every walker is checked; results agree to rounding).   */
                        /* Other bits must be 0.  (The field also keeps the doubles below 8-byte aligned.)            */
  double xbar_bound;    /* > 0: every component of the force-bias shift is capped in modulus, xbar_g <- xbar_g      */
                        /* min(1, bound / |xbar_g|), BEFORE xs, c_fb and c_mf are formed (Eqs. 12, 16 hold for any  */
                        /* xbar, so the estimator stays exact).  0: no bound (default).  SURVEY 8f NEXT-1, S8.      */
  double ehyb_bound;    /* > 0: the modulus of the importance function is bounded, |I| <- exp(-dt clip(D, -b, b))   */
                        /* with D = -log|I| / dt (the real part of the hybrid energy relative to E_shift); the      */
                        /* phase factor max(0, cos theta) is untouched.  0: no bound (default).                     */
} afqmc_params;

/* Setup (Eqs. 4-6; mean-field shift PAPER.md:108;
 * "half rotation").  Computes m_g = tr(L_g P), h' = h1 - 1/2 sum_g L_g L_g,
 * h_mod = h' + sum_g m_g L_g, E_const = -1/2 sum_g m_g^2, Lrot^g = trial^T L_g,
 * hrot = trial^T h1 and (if e_shift_auto) the trial's local energy, all on the device.
 *   h1     EITHER [M][M] symmetric, COPIED.
 *   L_chol DEVICE [n_chol][M][M], each L_g symmetric; BORROWED read-only until afqmc_destroy
 *          (it is the dominant resident array, 55 GB in the largest configuration).  With
 *          pack_chol = 1 it is borrowed only for the duration of afqmc_create: the handle keeps
 *          Lrot and a tile-packed copy of the upper triangles ([tiles][n_chol][8][16] doubles,
 *          0.51x the dense size at M = 1200) and every later call gives the same bits as with
 *          the dense tensor, so the caller may free L_chol afterwards.
 *   trial  EITHER [M][Nt] real, COPIED.
 *   out    receives the handle; NULL on failure.
 * Ordering: the handle runs on its own non-blocking stream (or params.stream).  afqmc_create synchronises the
 * device once on entry, so h1, L_chol and trial may have been written on any stream before the call; for every
 * LATER call the caller orders its own streams against the handle's (afqmc_sync, or events on params.stream).
 * max_walkers is at most 65535. */
int32_t afqmc_create(const double* h1, const double* L_chol, const double* trial,
                     const afqmc_params* p, afqmc_handle** out);

/* One walker step for nw walkers (Eqs. 12-18):
 * overlap and Theta = phi O^-1, force bias, field shift, A = V_HS build, phi <- E1 e^A E1 phi
 * with E1 = expm(-dt/2 h_mod) (cached per dt), new overlap, w <- w |I| max(0, cos arg S),
 * and, every ortho_every-th call, thin QR with R_ii > 0 (weights unchanged).
 *   walkers    EITHER complex128 [nw][M][Nt], in/out.
 *   weights    EITHER double [nw], in/out.
 *   aux_fields EITHER double [nw][n_chol], standard normal draws x (Eq. 8), read-only.
 * The overlap of the walkers as returned is kept in the handle (afqmc_get_overlaps). */
int32_t afqmc_step(afqmc_handle* h, void* walkers, double* weights, const double* aux_fields,
                   double dt, int32_t nw);

/* Local energy E_loc = <Psi_T|H|phi>/<Psi_T|phi> (Eq. 11):
 * one-body, Coulomb 1/2 sum_g X_g^2 and exchange -1/2 sum_g sum_spin tr(T_g T_g),
 * T_g = Lrot^g Theta.
 *   walkers EITHER complex128 [nw][M][Nt], read-only.
 *   E_out   EITHER complex128 [nw][3] = (E, E_1body, E_2body) per walker, as
 *           energy[:, 0..2] of the paper's Code Snippet 9. */
int32_t afqmc_local_energy(afqmc_handle* h, const void* walkers, void* E_out, int32_t nw);

/* Population control by the comb ("population control"; done locally on one
 * GPU; the algorithm is DESIGN.md reading S21 - the paper names none).  With
 * c_i = w_0 + ... + w_i (sequential float64 sum), W = c_{nw-1}, s = W / nw and the teeth
 * t_k = (k + xi) s, the new walker k is a copy of the old walker i_k = min(#{j : c_j <= t_k},
 * first j with c_j == W), and every new weight is s.  The overlaps kept in the handle are
 * permuted with the walkers.  If W is not finite or not > 0 nothing changes (identity map).
 *   walkers EITHER complex128 [nw][M][Nt], in/out.   weights EITHER double [nw], in/out.
 *   xi      EITHER one double in [0, 1), drawn by the caller (the library draws no random numbers).  A host value
 *           outside [0, 1) is rejected (AFQMC_ERR_INVALID); a device value is clamped into [0, 1) (NaN -> 0).
 *   map_out EITHER int32 [nw] or NULL: receives i_k (non-decreasing). */
int32_t afqmc_population_control(afqmc_handle* h, void* walkers, double* weights, const double* xi,
                                 int32_t nw, int32_t* map_out);

/* The comb of afqmc_population_control WITHOUT a handle and without any allocation: weights in, resampling map and
 * equalised weights out - the same map and the same weights, bit for bit, that afqmc_population_control returns for
 * these weights and this xi (permuting walkers, overlaps or anything else by map_out is left to the caller).
 * For whom: every other entry point needs an afqmc_handle, and afqmc_create cudaMallocs the workspaces of the whole
 * step.  A driver that only resamples, or that runs when no device memory is left to hand out (the Cholesky tensor and
 * the application's own memory pool own the GPU, so cudaMalloc fails), or that must not take the device-wide stall a
 * cudaMalloc / cudaFree implies while its other streams are busy, calls this instead: the comb's only scratch, the
 * running sum of the weights, sits in a fixed array inside the library image (8 bytes x
 * AFQMC_COMB_STATIC_MAX_WALKERS = 512 KiB, held on every GPU that loads the library until the process exits).  The
 * call makes no cudaMalloc, cudaFree or other allocating call and creates no stream or event.
 *   weights DEVICE double [nw], in/out: on return every weight is W / nw (unchanged if W is not finite or not > 0).
 *   xi      DEVICE one double, the caller's uniform draw; clamped into [0, 1) on the device (NaN -> 0).
 *   map_out DEVICE int32 [nw]: new walker k is a copy of old walker map_out[k] (non-decreasing).
 *   nw      1 .. AFQMC_COMB_STATIC_MAX_WALKERS; anything larger is refused with AFQMC_ERR_DIMS and a message.
 *   stream  cudaStream_t of the device that holds the three arrays (they must be plain device memory of ONE GPU;
 *           host and managed pointers are refused); NULL = that device's default stream.  The call is asynchronous.
 *   err     HOST char [err_len] or NULL: receives a message when the return value is not AFQMC_OK.
 * First call on each device: the library looks up the array's address on that device (cudaGetSymbolAddress, which
 * may load the library's device code there).  Make that first call outside any stream capture.
 * Sharing: all calls on one device use the same array.  Calls queued on ONE stream are safe back to back (every
 * call rewrites the part it reads; nothing needs clearing).  Calls that can run at the same time on one GPU - two
 * streams, two host threads, two handles' drivers - overwrite each other's sums and return garbage maps: order
 * them yourself.  Different GPUs have different copies and do not interfere. */
#define AFQMC_COMB_STATIC_MAX_WALKERS 65536
int32_t afqmc_comb_static(double* weights, const double* xi, int32_t* map_out, int32_t nw, void* stream, char* err,
                          int32_t err_len);

/* Estimator sums of the paper's Code Snippet 9:
 * est_out[0..3] = (ENumer, EDenom, E1Body, E2Body) = sum_w weights[w] (Re E[w][0], 1, Re E[w][1],
 * Re E[w][2]); the mixed energy estimate of Eq. (11) with Eq. (10)'s weights is ENumer/EDenom.
 *   weights EITHER double [nw];  E EITHER complex128 [nw][3] (from afqmc_local_energy);
 *   est_out EITHER double [4]. */
int32_t afqmc_estimators(afqmc_handle* h, const double* weights, const void* E, double* est_out,
                         int32_t nw);

/* One block ("100 blocks, each containing 25 steps"): n_steps times
 * afqmc_step (re-orthonormalising on the handle's ortho_every schedule), the comb after every
 * pop_every-th step of the block (pop_every = 0: never) with xi[0], xi[1], ... in order, then
 * afqmc_local_energy of the final walkers and afqmc_estimators.  One stream, no host
 * synchronisation between the steps when every buffer is a device buffer.
 *   walkers, weights  EITHER, in/out as in afqmc_step.
 *   aux_fields EITHER double [n_steps][nw][n_chol].
 *   xi         EITHER double [n_steps / pop_every] (may be NULL when pop_every = 0).
 *   E_out      EITHER complex128 [nw][3] or NULL.    est_out EITHER double [4] or NULL. */
int32_t afqmc_run_block(afqmc_handle* h, void* walkers, double* weights, const double* aux_fields,
                        const double* xi, double dt, int32_t nw, int32_t n_steps, int32_t pop_every,
                        void* E_out, double* est_out);

/* afqmc_run_block on device buffers replays a CUDA graph of the whole block from the third call
 * with the same arguments on (first call: eager, second: stream capture); the graph is keyed by
 * every pointer, nw, n_steps, pop_every, dt and the phase of the ortho_every schedule, so a
 * caller that reuses its buffers block after block pays one cudaGraphLaunch per block.
 * on = 1/0 switches this on (default) / off, on < 0 leaves it unchanged.  Returns the number of
 * graph launches issued so far on this handle (or a negative code). */
int64_t afqmc_set_block_graph(afqmc_handle* h, int32_t on);

/* Overlaps <Psi_T|phi_w> of the walkers as left by the last afqmc_step (permuted by any
 * afqmc_population_control since).
 *   ovlp_out EITHER complex128 [nw of that step]. */
int32_t afqmc_get_overlaps(afqmc_handle* h, void* ovlp_out);

/* Row a10 on its own ("stabilization"; reading S9): every walker block phi_sigma = Q R with R_ii
 * real > 0 is replaced by Q, in place - what afqmc_step does on the ortho_every schedule.  Repeated Cholesky-QR
 * passes with a shifted pass when the Gram matrix is numerically singular (cond(phi) up to ~1e15).
 *   walkers  EITHER complex128 [nw][M][Nt], in/out.
 *   detR_out EITHER double [nw][n_blocks] = prod_i R_ii per block (n_blocks = 1 RHF, 2 UHF), or NULL.
 * SIDE EFFECT on the handle's stored overlaps (afqmc_get_overlaps): the library cannot tell whose walkers it is
 * given, so whenever nw equals the nw of the last afqmc_step it ASSUMES these are that step's walkers and divides the
 * stored overlaps by prod_sigma det R_sigma (squared for RHF), as on the schedule.  Passing unrelated walkers of the
 * same count therefore leaves afqmc_get_overlaps meaningless until the next afqmc_step (which recomputes them from
 * scratch; nothing else in the library reads them).  Use a second handle, or a different nw, to orthonormalise
 * walkers that are not the handle's current population. */
int32_t afqmc_reorthonormalise(afqmc_handle* h, void* walkers, double* detR_out, int32_t nw);
/* Number of shifted Cholesky-QR passes (numerically singular Gram matrices) since afqmc_create; synchronises. */
int64_t afqmc_qr_shifted_passes(afqmc_handle* h);

/* Scalars fixed at create: out[0] = E_const, out[1] = E_shift in use, out[2] = trial energy
 * (NaN if never computed).  HOST pointer. */
int32_t afqmc_get_constants(afqmc_handle* h, double* out3);

/* Diagnostics for stage-by-stage parity tests: copies an internal device array of the last
 * step / energy call to `out` (EITHER).  which: 0 = X [nw][2][n_chol] (re plane, im plane;
 * the force-bias expectation <L_g> of the last step, spin summed), 1 = A = V_HS
 * [nw][2][M][M] (re plane, im plane), 2 = E1 [M][M], 3 = h_mod [M][M], 4 = m [n_chol],
 * 5 = Lrot [n_chol][Nt][M].  Returns the number of doubles written, or a negative code;
 * with out == NULL only returns the count.  With complex_chol: 0 = X [nw][2][2 n_chol] (the Hermitian matrices'
 * expectation values), 4 and 5 refer to the 4 n_chol real planes (Re K_1..Re K_2n, Im K_1..Im K_2n), 3 = Re h_mod. */
int64_t afqmc_debug_read(afqmc_handle* h, int32_t which, double* out);

/* Number of kernel launches issued by this handle since create (for bench.py). */
int64_t afqmc_launch_count(const afqmc_handle* h);

/* Per-stage device timing (for bench.py's roofline figures; off by default).  With profiling on,
 * every stage of afqmc_step / afqmc_local_energy is bracketed by two CUDA events recorded on the
 * handle's stream (no synchronisation is added).  afqmc_get_stage_times synchronises the stream,
 * adds the elapsed time of every bracket recorded since the last call to running totals and
 * writes totals (milliseconds) and bracket counts; reset != 0 clears the totals afterwards.
 * Stage indices: */
#define AFQMC_STAGE_OVERLAP_THETA 0  /* a1/a2 overlap, inverse, Theta (step)                  */
#define AFQMC_STAGE_FORCE_BIAS 1     /* a3 GEMM                                               */
#define AFQMC_STAGE_FIELD_SHIFT 2    /* a4                                                    */
#define AFQMC_STAGE_VHS 3            /* a5 GEMM over the Cholesky index                       */
#define AFQMC_STAGE_ONE_BODY 4       /* a6 + a8                                               */
#define AFQMC_STAGE_TAYLOR 5         /* a7, all orders                                        */
#define AFQMC_STAGE_OVERLAP_NEW 6    /* a9 overlap of the propagated walkers                  */
#define AFQMC_STAGE_WEIGHT 7         /* a9 weight update                                      */
#define AFQMC_STAGE_REORTHO 8        /* a10                                                   */
#define AFQMC_STAGE_E_THETA 9        /* a11: overlap, Theta, one-body energy                  */
#define AFQMC_STAGE_EXCHANGE 10      /* a11: T = Lrot Theta, tr(TT), tr(T)                    */
#define AFQMC_STAGE_E_REDUCE 11      /* a11: Coulomb sum and final energies                   */
#define AFQMC_STAGE_E1_BUILD 12      /* expm(-dt/2 h_mod), only when dt changes               */
#define AFQMC_STAGE_POP_CONTROL 13   /* comb + walker permutation                            */
#define AFQMC_STAGE_ESTIMATORS 14    /* weighted sums of Code Snippet 9                       */
#define AFQMC_STAGE_SHARD_EXCHANGE 15 /* distributed Hamiltonian: pushes into peer slots (copies)  */
#define AFQMC_STAGE_SHARD_REDUCE 16   /* distributed Hamiltonian: fixed-order sums of the slots    */
#define AFQMC_STAGE_FUSED_STEP 17     /* small systems: rows a1-a9 in one kernel (fused_small.cu)   */
#define AFQMC_STAGE_FUSED_ENERGY 18   /* small systems: row a11 in one kernel                       */
#define AFQMC_STAGE_COUNT 19
int32_t afqmc_set_profiling(afqmc_handle* h, int32_t on);
/*   ms_out HOST double [AFQMC_STAGE_COUNT]; count_out HOST int64 [AFQMC_STAGE_COUNT] or NULL. */
int32_t afqmc_get_stage_times(afqmc_handle* h, double* ms_out, int64_t* count_out, int32_t reset);

/* Stream synchronise and surface any deferred CUDA error. */
int32_t afqmc_sync(afqmc_handle* h);

const char* afqmc_last_error(const afqmc_handle* h);

void afqmc_destroy(afqmc_handle* h);

/* ---- Distributed Hamiltonian ("Distributed Hamiltonian for limited memory", PAPER.md:308-318,
 * Fig. 6) -------------------------------------------------------------------
 * When the Cholesky tensor does not fit one GPU it is split over the gamma index among the G
 * members of a group; every member owns its own nw walkers.  Everything that is a sum over gamma
 *     h_mod - h1, E_const, A = V_HS (Eq. 9), c_fb, c_mf (Eqs. 12, 16), E_C + E_X (Eq. 11)
 * is computed slice by slice by the member holding the slice FOR ALL G * nw WALKERS OF THE GROUP
 * and added up by the walker's owner in fixed member order 0 .. G-1 (results do not depend on
 * timing).  The paper passes walkers cyclically over MPI; here the members' buffers
 * are mapped into each other's address space (NVLink peer memory, CUDA IPC between processes, or
 * simply the same device) and
 *   - Theta^T of a member's walkers is pushed into every member's gather buffer (slot = owner),
 *   - the V_HS kernel's epilogue stores each walker's partial A straight into its OWNER's receive
 *     slot [source member] (the scatter of the reduce-scatter is the GEMM epilogue itself),
 *   - the partial scalars and energies follow the same way.
 * The library never synchronises members: the caller puts a group barrier ORDERED ON EVERY
 * MEMBER'S STREAM (e.g. a one-element NCCL all-reduce on that stream, or a stream synchronise
 * plus a host barrier) where "== barrier ==" stands below.  One step of the whole group is
 *     afqmc_shard_theta(for_energy = 0)  == barrier ==  afqmc_shard_vhs  == barrier ==
 *     afqmc_shard_propagate
 * and one local-energy evaluation
 *     afqmc_shard_theta(for_energy = 1)  == barrier ==  afqmc_shard_energy  == barrier ==
 *     afqmc_shard_energy_finish.
 * Two more barriers are needed only where a phase overwrites what a peer may still read: none in
 * the sequences above as long as every member issues the same sequence.
 * Restrictions: even M and even local n_chol; nw == max_walkers on every member (the group batch
 * is contiguous); device pointers only.  afqmc_step / afqmc_local_energy / afqmc_run_block /
 * afqmc_population_control return AFQMC_ERR_UNSUPPORTED on such a handle.
 *
 * Setup.  afqmc_create on a member computes everything that is local to its slice (m_g, Lrot,
 * its share of h_mod - h1, of E_const and of the trial's two-body energy).
 * afqmc_shard_setup_partial writes these M*M + 2 doubles to `out` (EITHER); the caller adds them
 * over the group (all-reduce, or member order 0..G-1) and gives every member the same sums
 * through afqmc_shard_setup_finish (`sum` EITHER, [M*M + 2]).  Phases fail with AFQMC_ERR_INVALID
 * before that. */
int32_t afqmc_shard_setup_partial(afqmc_handle* h, double* out);
int32_t afqmc_shard_setup_finish(afqmc_handle* h, const double* sum);
/* The member-order sum for callers that hold all partials in one place (one process driving G members, or after
 * an all-gather): out[i] = parts[0][i] + parts[1][i] + ... + parts[n_members-1][i] in exactly that order.
 *   parts HOST [n_members][n], out HOST [n], n = M*M + 2. */
int32_t afqmc_shard_setup_reduce(const double* parts, int32_t n_members, int64_t n, double* out);

/* The four exchange buffers of this member, as device addresses: out[0] Theta^T gather buffer
 * [G][nw][2][Nt][M], out[1] V_HS receive slots [G][nw][2][M][M], out[2] scalar slots
 * [G][2][nw] complex (c_fb, c_mf), out[3] energy slots [G][nw] complex.  HOST pointer. */
int32_t afqmc_shard_get_buffers(afqmc_handle* h, uint64_t* out4);
/* CUDA IPC handle (64 bytes, HOST) of buffer `which` (0..3) for members in other processes, and
 * the matching open / close in the importing process (cudaIpcOpenMemHandle / Close). */
int32_t afqmc_shard_ipc_export(afqmc_handle* h, int32_t which, void* handle64);
/*   h: the importing member (the mapping is made on ITS device); NULL = the current device. */
int32_t afqmc_shard_ipc_open(afqmc_handle* h, const void* handle64, uint64_t* addr_out);
int32_t afqmc_shard_ipc_close(uint64_t addr);
/* addrs HOST [G][4]: the buffers of every member as seen from THIS process (row group_rank
 * must be this handle's own).  The pointers are borrowed until afqmc_destroy. */
int32_t afqmc_shard_set_peers(afqmc_handle* h, const uint64_t* addrs);

/* a1-a2 on this member's own walkers (DEVICE complex128 [nw][M][Nt]); Theta^T goes to slot
 * group_rank of every member's gather buffer.  for_energy != 0 also keeps the one-body energy. */
int32_t afqmc_shard_theta(afqmc_handle* h, const void* walkers, int32_t nw, int32_t for_energy);
/* a3-a5 with this member's Cholesky vectors for all G * nw walkers of the group.
 *   aux_local DEVICE double [G * nw][n_chol]: the fields x of every group walker (member-major
 *   order) restricted to this member's gamma slice.
 * Partial c_fb, c_mf and V_HS go to the owners' slots. */
int32_t afqmc_shard_vhs(afqmc_handle* h, const double* aux_local, double dt, int32_t nw);
/* Owner side: A, c_fb, c_mf = sums of the G slots, then a6-a10 on the own walkers (as afqmc_step).
 *   walkers DEVICE in/out, weights DEVICE in/out. */
int32_t afqmc_shard_propagate(afqmc_handle* h, void* walkers, double* weights, double dt, int32_t nw);
/* a11 with this member's Cholesky vectors for all group walkers (after afqmc_shard_theta with
 * for_energy = 1 on every member): partial E_C + E_X to the owners' slots. */
int32_t afqmc_shard_energy(afqmc_handle* h, int32_t nw);
/* Owner side: E_out DEVICE complex128 [nw][3] = (E, E_1body, E_2body). */
int32_t afqmc_shard_energy_finish(afqmc_handle* h, void* E_out, int32_t nw);

/* Measurement helper (not part of the method): register-only issue loops on all SMs for
 * `ms` milliseconds each.  out[0] = FP64 mma.sync m8n8k4 (DMMA) TFLOP/s, out[1] = FP64 FMA
 * (DFMA) TFLOP/s, out[2] = SM clock seen (MHz, from clock64/elapsed).  HOST pointer. */
int32_t afqmc_measure_fp64_peak(double ms, double* out3);

/* Measurement helper (host only, no GPU work): the tile plan of the exchange kernel (a11, Eq. 11) for an occupied
 * block of `ns` columns and `M` basis functions (the K loop), as text in `out` (HOST, at most `n` bytes incl. the terminator): consumer warps, vectors and
 * walkers per tile, useful fraction of the issued DMMA blocks, ring depth, epilogue passes.  `pair` = 1: the plan
 * of the complex (two-plane) half-rotated tensor.  Returns that useful fraction times 1e6, or AFQMC_ERR_INVALID. */
int32_t afqmc_exchange_plan(int32_t ns, int32_t M, int32_t pair, char* out, int32_t n);
/* Tuning hook (host only): replace the plan chosen for (ns, M, pair) in this process by the candidate with `warps`
 * consumer warps (8 or 12) arranged as wm x (warps / wm), warp rectangles of at most mi x ni DMMA blocks, G vectors x
 * Wn walkers per tile, epi_warps (3, or 7 with 8 consumer warps) epilogue warps.  Results do not depend on the plan beyond the order of the fixed-order sums.  Handles
 * created BEFORE the call keep buffers sized for the old plan: pin first, then create (afqmc_local_energy on an older
 * handle returns AFQMC_ERR_INVALID if the new plan groups the vectors differently).  AFQMC_ERR_UNSUPPORTED if
 * no such candidate exists (does not fit shared memory or registers). */
int32_t afqmc_exchange_plan_pin(int32_t ns, int32_t M, int32_t pair, int32_t warps, int32_t mi, int32_t ni, int32_t wm,
                                int32_t G, int32_t Wn, int32_t epi_warps);
/* Undo afqmc_exchange_plan_pin for (ns, M, pair): the next handle gets the library's own plan again.  ns <= 0 forgets
 * every pin of the process.  The same ordering rule applies as for pinning: handles that exist keep buffers sized for
 * the plan they were created under.  The plan table is process-wide and mutex protected; a launch works on its own
 * copy of the plan, so pinning from one host thread while another thread launches is safe (that launch uses the old
 * or the new plan, never a mixture). */
int32_t afqmc_exchange_plan_unpin(int32_t ns, int32_t M, int32_t pair);

#ifdef __cplusplus
}
#endif
#endif /* AFQMC_H_ */
