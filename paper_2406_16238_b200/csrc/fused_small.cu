// fused_small.cu - the whole walker step (rows a1-a9) and the whole local energy (a11) as ONE kernel each, one CTA
// per walker, for systems small enough that a walker's working set (phi, Theta, the Taylor terms, V_HS, E1) lives in
// shared memory (c1: M = 24, N_occ = 5, 96 Cholesky vectors).  SURVEY 8(d): "c1 is launch-latency-bound" - with one
// kernel per stage a c1 step was 18 launches for 1.2e7 flops, 81 us per step even inside a CUDA graph.  Plain FP64
// FMAs: at these sizes the tensor-core tiles would be mostly padding.  Same formulas, same order of stages as the
// general path (api.cu: step_device / local_energy_device); only the summation orders differ.
//   Eqs. (9), (12)-(18); Eq. (11).
#include "internal.h"
#include "tma.cuh"

namespace afq {

namespace {

__device__ __forceinline__ void bulk_load_1d(void* smem, const void* gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(smem_u32(smem)), "l"(gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ double2 cmul2(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cinv2(double2 a) {
  const double d = a.x * a.x + a.y * a.y;
  return make_double2(a.x / d, -a.y / d);
}

// sum of NV doubles per thread over the CTA (256 threads); result valid in every thread
template <int NV>
__device__ __forceinline__ void cta_sum(double (&v)[NV], double* red /* [8 * NV] */) {
#pragma unroll
  for (int k = 0; k < NV; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0)
    for (int k = 0; k < NV; ++k) red[warp * NV + k] = v[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NV; ++k) {
    double s = 0.0;
    for (int q = 0; q < 8; ++q) s += red[q * NV + k];
    v[k] = s;
  }
}

// O = psi_b^T phi_b into Aug = [O | 1] (ns x 2 ns), then Gauss-Jordan with row pivoting: Aug = [1 | O^-1].
// Returns det O (valid in every thread).  phi: [M][Nt] complex in shared memory, psi: [M][Nt] real.
__device__ double2 overlap_inverse(const double2* phi, const double* psi, double2* Aug, int M, int Nt, int off, int ns,
                                   int* /*s_piv*/, double2* s_det) {
  const int tid = threadIdx.x, ld = 2 * ns;
  for (int idx = tid; idx < ns * ns; idx += blockDim.x) {
    const int i = idx / ns, j = idx - i * ns;
    double2 s = make_double2(0.0, 0.0);
    for (int q = 0; q < M; ++q) {
      const double p = psi[q * Nt + off + i];
      const double2 z = phi[q * Nt + off + j];
      s.x = fma(p, z.x, s.x);
      s.y = fma(p, z.y, s.y);
    }
    Aug[i * ld + j] = s;
    Aug[i * ld + ns + j] = make_double2(i == j ? 1.0 : 0.0, 0.0);
  }
  __syncthreads();
  // the elimination itself is small (ns <= 16): warp 0 runs it with warp-level synchronisation only
  if (tid < 32) {
    double2 det = make_double2(1.0, 0.0);
    for (int c = 0; c < ns; ++c) {
      int bi = c;
      double best = -1.0;
      for (int r = c; r < ns; ++r) {                    // every lane scans the column: same result in every lane
        const double2 v = Aug[r * ld + c];
        const double m = v.x * v.x + v.y * v.y;
        if (!(m <= best)) { best = m; bi = r; }         // NaN counts as a candidate so it propagates
      }
      const double2 d = cmul2(det, Aug[bi * ld + c]);
      det = bi != c ? make_double2(-d.x, -d.y) : d;
      __syncwarp();
      if (bi != c)
        for (int j = tid; j < ld; j += 32) {
          const double2 u = Aug[c * ld + j];
          Aug[c * ld + j] = Aug[bi * ld + j];
          Aug[bi * ld + j] = u;
        }
      __syncwarp();
      const double2 ipv = cinv2(Aug[c * ld + c]);
      __syncwarp();
      for (int j = tid; j < ld; j += 32) Aug[c * ld + j] = cmul2(Aug[c * ld + j], ipv);
      __syncwarp();
      for (int idx = tid; idx < ns * ld; idx += 32) {
        const int r = idx / ld, j = idx - r * ld;
        if (r != c && j != c) {
          const double2 f = Aug[r * ld + c], t = Aug[c * ld + j];
          double2 v = Aug[r * ld + j];
          v.x -= f.x * t.x - f.y * t.y;
          v.y -= f.x * t.y + f.y * t.x;
          Aug[r * ld + j] = v;
        }
      }
      __syncwarp();
      for (int r = tid; r < ns; r += 32)
        if (r != c) Aug[r * ld + c] = make_double2(0.0, 0.0);
      __syncwarp();
    }
    if (tid == 0) *s_det = det;
  }
  __syncthreads();
  return *s_det;
}

// Theta_b = phi_b O^-1 for the block whose inverse sits in Aug[:, ns:2ns]
__device__ void theta_block(const double2* phi, const double2* Aug, double2* th, int M, int Nt, int off, int ns) {
  const int ld = 2 * ns;
  for (int idx = threadIdx.x; idx < M * ns; idx += blockDim.x) {
    const int q = idx / ns, i = idx - q * ns;
    double2 s = make_double2(0.0, 0.0);
    for (int k = 0; k < ns; ++k) {
      const double2 z = phi[q * Nt + off + k], o = Aug[k * ld + ns + i];
      s.x += z.x * o.x - z.y * o.y;
      s.y += z.x * o.y + z.y * o.x;
    }
    th[q * Nt + off + i] = s;
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------ step
__global__ void __launch_bounds__(256) small_step_kernel(SmallArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int w = blockIdx.x, tid = threadIdx.x;
  const int M = a.M, Nt = a.Nt, nc = a.n_chol, MN = M * Nt, MM = M * M;
  int nsmax = a.ns[0];
  if (a.nblk > 1 && a.ns[1] > nsmax) nsmax = a.ns[1];
  double2* phi = reinterpret_cast<double2*>(smraw);      // [M][Nt] walker, later E1 phi
  double2* th = phi + MN;                                // Theta, later Taylor term (ping)
  double2* t1 = th + MN;                                 // Taylor term (pong)
  double2* acc = t1 + MN;                                // running sum of the Taylor terms
  double2* A = acc + MN;                                 // [M][M] V_HS
  double2* Aug = A + MM;                                 // [nsmax][2 nsmax]
  double2* xs = Aug + nsmax * 2 * nsmax;                 // [nc] X, then xs
  double* E1s = reinterpret_cast<double*>(xs + nc);      // [M][M]
  double* psi = E1s + MM;                                // [M][Nt]
  double* red = psi + MN;                                // [64]
  double* Lbuf = red + 64;                               // [2][lchunk][M][M] staging of L (16-byte aligned: see step_smem)
  __shared__ int s_piv;
  __shared__ double2 s_det;
  __shared__ __align__(8) uint64_t lbar[2];

  double2* Wg = reinterpret_cast<double2*>(a.W) + (size_t)w * MN;
  if (tid == 0) { mbar_init(&lbar[0], 1); mbar_init(&lbar[1], 1); fence_barrier_init(); }
  for (int i = tid; i < MN; i += blockDim.x) { phi[i] = Wg[i]; psi[i] = a.trial[i]; }
  for (int i = tid; i < MM; i += blockDim.x) E1s[i] = a.E1[i];
  __syncthreads();

  // a1 / a2: overlap, inverse, Theta per stored block
  double2 ov_old = make_double2(1.0, 0.0);
  for (int b = 0; b < a.nblk; ++b) {
    const double2 d = overlap_inverse(phi, psi, Aug, M, Nt, a.off[b], a.ns[b], &s_piv, &s_det);
    ov_old = cmul2(ov_old, d);
    if (a.rhf) ov_old = cmul2(ov_old, d);
    theta_block(phi, Aug, th, M, Nt, a.off[b], a.ns[b]);
    __syncthreads();
  }

  // a3 / a4: X_g = sf sum_iq Lrot[g][i][q] Theta[q][i]; xbar = i sqrt(dt) (X - m); xs = x - xbar; scalars
  const double sq = a.sqrt_dt;
  double v[4] = {0.0, 0.0, 0.0, 0.0};      // c_fb (re, im), sum xs m (re, im)
  // a warp per vector, lanes over the Nt x M products (Lrot rows are contiguous: coalesced)
  const int lane = tid & 31, wp = tid >> 5;
  for (int g = wp; g < nc; g += 8) {
    const double* lr = a.Lrot + (size_t)g * MN;
    double xr = 0.0, xi = 0.0;
    for (int e = lane; e < MN; e += 32) {
      const int i = e / M, q = e - i * M;
      const double l = lr[e];
      const double2 t = th[q * Nt + i];
      xr = fma(l, t.x, xr);
      xi = fma(l, t.y, xi);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      xr += __shfl_xor_sync(0xffffffffu, xr, o);
      xi += __shfl_xor_sync(0xffffffffu, xi, o);
    }
    if (lane == 0) xs[g] = make_double2(a.sf * xr, a.sf * xi);
  }
  __syncthreads();
  for (int g = tid; g < nc; g += blockDim.x) {
    const double xr = xs[g].x, xi = xs[g].y;
    if (a.Xdbg) {
      a.Xdbg[(size_t)(2 * w) * nc + g] = xr;
      a.Xdbg[(size_t)(2 * w + 1) * nc + g] = xi;
    }
    const double mg = a.m[g], x = a.x[(size_t)w * nc + g];
    double br = -sq * xi, bi = sq * (xr - mg);
    if (a.xbar_bound > 0.0) {
      const double mag = hypot(br, bi);
      if (mag > a.xbar_bound) { const double sc = a.xbar_bound / mag; br *= sc; bi *= sc; }
    }
    const double sr = x - br, si = -bi;
    v[0] += x * br - 0.5 * (br * br - bi * bi);
    v[1] += x * bi - br * bi;
    v[2] += sr * mg;
    v[3] += si * mg;
    xs[g] = make_double2(sr, si);
  }
  cta_sum<4>(v, red);
  const double cfb_r = v[0], cfb_i = v[1], cmf_r = -sq * v[3], cmf_i = sq * v[2];

  // a5: A = -i sqrt(dt) sum_g xs_g L_g  (Re A = sqrt(dt) sum Im xs L, Im A = -sqrt(dt) sum Re xs L)
  // L is streamed through shared memory by the bulk-copy engine (cp.async.bulk, two buffers of `lchunk` vectors, one
  // mbarrier each): a thread's own loads would come out of L2 a few at a time with ~1000 clocks of latency each,
  // which made this loop half of the kernel.  Needs 16-byte slices (even M * M); otherwise direct loads.
  if (a.lchunk > 0) {
    const int nchunks = (nc + a.lchunk - 1) / a.lchunk;
    const uint32_t slice = (uint32_t)MM * 8u;
    if (tid == 0) {
      for (int c = 0; c < 2 && c < nchunks; ++c) {
        const int gn = min(a.lchunk, nc - c * a.lchunk);
        mbar_expect_tx(&lbar[c], slice * gn);
        bulk_load_1d(Lbuf + (size_t)c * a.lchunk * MM, a.L + (size_t)c * a.lchunk * MM, slice * gn, &lbar[c]);
      }
    }
    double sr[4] = {0.0, 0.0, 0.0, 0.0}, si[4] = {0.0, 0.0, 0.0, 0.0};      // MM <= 4 * 1024: up to 16 elements / thread
    double sr2[12], si2[12];
#pragma unroll
    for (int u = 0; u < 12; ++u) sr2[u] = si2[u] = 0.0;
    for (int c = 0; c < nchunks; ++c) {
      const int b = c & 1, gn = min(a.lchunk, nc - c * a.lchunk);
      mbar_wait(&lbar[b], (c >> 1) & 1);
      const double* Lb = Lbuf + (size_t)b * a.lchunk * MM;
      for (int g = 0; g < gn; ++g) {
        const double2 cx = xs[c * a.lchunk + g];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int pq = tid + u * 256;
          if (pq < MM) { const double l = Lb[g * MM + pq]; sr[u] = fma(cx.x, l, sr[u]); si[u] = fma(cx.y, l, si[u]); }
        }
        if (MM > 1024) {
#pragma unroll
          for (int u = 0; u < 12; ++u) {
            const int pq = tid + (u + 4) * 256;
            if (pq < MM) { const double l = Lb[g * MM + pq]; sr2[u] = fma(cx.x, l, sr2[u]); si2[u] = fma(cx.y, l, si2[u]); }
          }
        }
      }
      __syncthreads();                                   // everyone is done with buffer b
      if (tid == 0 && c + 2 < nchunks) {
        const int gn2 = min(a.lchunk, nc - (c + 2) * a.lchunk);
        mbar_expect_tx(&lbar[b], slice * gn2);
        bulk_load_1d(Lbuf + (size_t)b * a.lchunk * MM, a.L + (size_t)(c + 2) * a.lchunk * MM, slice * gn2, &lbar[b]);
      }
    }
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const int pq = tid + u * 256;
      if (pq < MM) {
        const double vr = u < 4 ? sr[u & 3] : sr2[(u - 4) % 12], vi = u < 4 ? si[u & 3] : si2[(u - 4) % 12];
        const double2 z = make_double2(sq * vi, -sq * vr);
        A[pq] = z;
        if (a.Adbg) {
          a.Adbg[(size_t)(2 * w) * MM + pq] = z.x;
          a.Adbg[(size_t)(2 * w + 1) * MM + pq] = z.y;
        }
      }
    }
  } else {
    for (int pq = tid; pq < MM; pq += blockDim.x) {
      double sr = 0.0, si = 0.0;
      const double* Lp = a.L + pq;
#pragma unroll 8
      for (int g = 0; g < nc; ++g) {
        const double l = Lp[(size_t)g * MM];
        sr = fma(xs[g].x, l, sr);
        si = fma(xs[g].y, l, si);
      }
      const double2 z = make_double2(sq * si, -sq * sr);
      A[pq] = z;
      if (a.Adbg) {
        a.Adbg[(size_t)(2 * w) * MM + pq] = z.x;
        a.Adbg[(size_t)(2 * w + 1) * MM + pq] = z.y;
      }
    }
  }
  // a6: T0 = acc = E1 phi   (phi is read, th / acc written)
  for (int idx = tid; idx < MN; idx += blockDim.x) {
    const int p = idx / Nt, j = idx - p * Nt;
    double sr = 0.0, si = 0.0;
    for (int q = 0; q < M; ++q) {
      const double e = E1s[p * M + q];
      const double2 z = phi[q * Nt + j];
      sr = fma(e, z.x, sr);
      si = fma(e, z.y, si);
    }
    th[idx] = make_double2(sr, si);
    acc[idx] = make_double2(sr, si);
  }
  __syncthreads();
  // a7: T_n = A T_{n-1} / n, acc += T_n
  double2 *Tp = th, *Tn = t1;
  for (int n = 1; n <= a.K; ++n) {
    const double inv = 1.0 / n;
    for (int idx = tid; idx < MN; idx += blockDim.x) {
      const int p = idx / Nt, j = idx - p * Nt;
      double sr = 0.0, si = 0.0;
      for (int q = 0; q < M; ++q) {
        const double2 c = A[p * M + q], z = Tp[q * Nt + j];
        sr += c.x * z.x - c.y * z.y;
        si += c.x * z.y + c.y * z.x;
      }
      sr *= inv; si *= inv;
      Tn[idx] = make_double2(sr, si);
      acc[idx].x += sr; acc[idx].y += si;
    }
    __syncthreads();
    double2* tmp = Tp; Tp = Tn; Tn = tmp;
  }
  // a8: phi = E1 acc, to shared memory and to the caller's walker
  for (int idx = tid; idx < MN; idx += blockDim.x) {
    const int p = idx / Nt, j = idx - p * Nt;
    double sr = 0.0, si = 0.0;
    for (int q = 0; q < M; ++q) {
      const double e = E1s[p * M + q];
      const double2 z = acc[q * Nt + j];
      sr = fma(e, z.x, sr);
      si = fma(e, z.y, si);
    }
    phi[idx] = make_double2(sr, si);
    Wg[idx] = make_double2(sr, si);
  }
  __syncthreads();
  // a9: new overlap and the phaseless weight (as weight_update_kernel, small.cu)
  double2 ov_new = make_double2(1.0, 0.0);
  for (int b = 0; b < a.nblk; ++b) {
    const double2 d = overlap_inverse(phi, psi, Aug, M, Nt, a.off[b], a.ns[b], &s_piv, &s_det);
    ov_new = cmul2(ov_new, d);
    if (a.rhf) ov_new = cmul2(ov_new, d);
    __syncthreads();
  }
  if (tid == 0) {
    reinterpret_cast<double2*>(a.ovlp)[w] = ov_new;
    const double d = ov_old.x * ov_old.x + ov_old.y * ov_old.y;
    const double2 r = make_double2((ov_new.x * ov_old.x + ov_new.y * ov_old.y) / d,
                                   (ov_new.y * ov_old.x - ov_new.x * ov_old.y) / d);
    const double em = exp(cmf_r);
    double sn, cs;
    sincos(cmf_i, &sn, &cs);
    const double2 S = cmul2(r, make_double2(em * cs, em * sn));
    const double absS = hypot(S.x, S.y);
    double absI = absS * exp(cfb_r) * exp(a.expo);
    const bool finI = isfinite(absI);          // before the bound, as in weight_update_kernel (small.cu)
    if (a.ehyb_bound > 0.0 && absI > 0.0) {
      const double D = -log(absI) / a.dt;
      if (fabs(D) > a.ehyb_bound) absI = exp(-a.dt * copysign(a.ehyb_bound, D));
    }
    const bool ok = isfinite(S.x) && isfinite(S.y) && finI && absS > 0.0 &&
                    (ov_old.x != 0.0 || ov_old.y != 0.0) && isfinite(ov_new.x) && isfinite(ov_new.y) && isfinite(cfb_i);
    double wt = a.weights[w];
    if (!ok) {
      wt = 0.0;
    } else {
      const double c = S.x / absS;
      wt = wt * absI * (c > 0.0 ? c : 0.0);
    }
    a.weights[w] = wt;
  }
}

// ------------------------------------------------------------------------------------------ local energy
// E1b = sf sum_b sum_iq hrot[i][q] Theta[q][i];  X_g = sum_b tr(T^g_b);  E_C = 1/2 sum_g (sf X_g)^2;
// E_X = -1/2 sf sum_g sum_b tr(T^g_b T^g_b),  T^g_b = Lrot^g_b Theta_b   (Eq. 11)
__global__ void __launch_bounds__(256) small_energy_kernel(SmallArgs a) {
  extern __shared__ __align__(16) unsigned char smraw[];
  const int w = blockIdx.x, tid = threadIdx.x;
  const int M = a.M, Nt = a.Nt, nc = a.n_chol, MN = M * Nt;
  int nsmax = a.ns[0];
  if (a.nblk > 1 && a.ns[1] > nsmax) nsmax = a.ns[1];
  double2* phi = reinterpret_cast<double2*>(smraw);
  double2* th = phi + MN;
  double2* Aug = th + MN;                                // [nsmax][2 nsmax]
  double2* Xs = Aug + nsmax * 2 * nsmax;                 // [nc] sum over blocks of tr(T)
  double2* Tb = Xs + nc;                                 // [gchunk][ns][ns]
  double* psi = reinterpret_cast<double*>(Tb + (size_t)a.gchunk * nsmax * nsmax);
  double* red = psi + MN;
  __shared__ int s_piv;
  __shared__ double2 s_det;

  const double2* Wg = reinterpret_cast<const double2*>(a.W) + (size_t)w * MN;
  for (int i = tid; i < MN; i += blockDim.x) { phi[i] = Wg[i]; psi[i] = a.trial[i]; }
  for (int g = tid; g < nc; g += blockDim.x) Xs[g] = make_double2(0.0, 0.0);
  __syncthreads();
  for (int b = 0; b < a.nblk; ++b) {
    overlap_inverse(phi, psi, Aug, M, Nt, a.off[b], a.ns[b], &s_piv, &s_det);
    theta_block(phi, Aug, th, M, Nt, a.off[b], a.ns[b]);
    __syncthreads();
  }
  double v[4] = {0.0, 0.0, 0.0, 0.0};      // e1 (re, im), sum tr(TT) (re, im)
  for (int idx = tid; idx < MN; idx += blockDim.x) {
    const int q = idx / Nt, i = idx - q * Nt;
    const double hr = a.hrot[i * M + q];
    v[0] = fma(hr, th[idx].x, v[0]);
    v[1] = fma(hr, th[idx].y, v[1]);
  }
  for (int b = 0; b < a.nblk; ++b) {
    const int ns = a.ns[b], off = a.off[b], nn = ns * ns;
    for (int g0 = 0; g0 < nc; g0 += a.gchunk) {
      const int gc = min(a.gchunk, nc - g0);
      for (int idx = tid; idx < gc * nn; idx += blockDim.x) {
        const int gl = idx / nn, ij = idx - gl * nn, i = ij / ns, j = ij - i * ns;
        const double* lr = a.Lrot + ((size_t)(g0 + gl) * Nt + off + i) * M;
        double sr = 0.0, si = 0.0;
        for (int q = 0; q < M; ++q) {
          const double l = lr[q];
          const double2 t = th[q * Nt + off + j];
          sr = fma(l, t.x, sr);
          si = fma(l, t.y, si);
        }
        Tb[idx] = make_double2(sr, si);
      }
      __syncthreads();
      for (int gl = tid; gl < gc; gl += blockDim.x) {
        const double2* T = Tb + (size_t)gl * nn;
        double tr_r = 0.0, tr_i = 0.0, xr = 0.0, xi = 0.0;
        for (int i = 0; i < ns; ++i) {
          xr += T[i * ns + i].x; xi += T[i * ns + i].y;
          for (int j = 0; j < ns; ++j) {
            const double2 p = T[i * ns + j], q = T[j * ns + i];
            tr_r += p.x * q.x - p.y * q.y;
            tr_i += p.x * q.y + p.y * q.x;
          }
        }
        v[2] += tr_r; v[3] += tr_i;
        Xs[g0 + gl].x += xr; Xs[g0 + gl].y += xi;
      }
      __syncthreads();
    }
  }
  double c[2] = {0.0, 0.0};                // sum (sf X)^2
  for (int g = tid; g < nc; g += blockDim.x) {
    const double xr = a.sf * Xs[g].x, xi = a.sf * Xs[g].y;
    c[0] += xr * xr - xi * xi;
    c[1] += 2.0 * xr * xi;
  }
  double s[6] = {v[0], v[1], v[2], v[3], c[0], c[1]};
  cta_sum<6>(s, red);
  if (tid == 0) {
    const double e1r = a.sf * s[0], e1i = a.sf * s[1];
    const double e2r = 0.5 * s[4] - 0.5 * a.sf * s[2], e2i = 0.5 * s[5] - 0.5 * a.sf * s[3];
    double* o = a.E_out + (size_t)w * 6;
    o[0] = e1r + e2r; o[1] = e1i + e2i;
    o[2] = e1r;       o[3] = e1i;
    o[4] = e2r;       o[5] = e2i;
  }
}

namespace {
size_t step_smem(const SmallArgs& a, int nsmax) {
  const size_t MN = (size_t)a.M * a.Nt, MM = (size_t)a.M * a.M;
  // the 16-byte parts first; E1 (MM doubles) + psi (MN doubles) + red (64): round their sum to an even count so
  // that the bulk-copy buffers behind them stay 16-byte aligned
  const size_t dbl = ((MM + MN + 64 + 1) & ~(size_t)1) + (size_t)2 * a.lchunk * MM;
  return (4 * MN + MM + (size_t)nsmax * 2 * nsmax + a.n_chol) * 16 + dbl * 8;
}
// vectors per bulk copy: two buffers of about 32 KB each; 0 (direct loads) when a slice is not a multiple of 16 bytes
int pick_lchunk(int M, int n_chol, const void* L) {
  const size_t MM = (size_t)M * M;
  if ((MM & 1) || ((uintptr_t)L & 15)) return 0;
  int c = (int)(32768 / (MM * 8));
  if (c < 1) c = 1;
  if (c > n_chol) c = n_chol;
  return c;
}
size_t energy_smem(const SmallArgs& a, int nsmax, int gchunk) {
  const size_t MN = (size_t)a.M * a.Nt;
  return (2 * MN + (size_t)nsmax * 2 * nsmax + a.n_chol + (size_t)gchunk * nsmax * nsmax) * 16 + (MN + 64) * 8;
}
int ns_max(const SmallArgs& a) { return (a.nblk > 1 && a.ns[1] > a.ns[0]) ? a.ns[1] : a.ns[0]; }
}  // namespace

// a walker's working set fits one CTA's shared memory and the per-thread loops stay short
bool small_path_fits(int M, int Nt, int nsmax, int n_chol) {
  if (M > 64 || Nt > 32 || nsmax > 16 || n_chol > 2048) return false;
  SmallArgs a{};
  a.M = M; a.Nt = Nt; a.n_chol = n_chol; a.lchunk = pick_lchunk(M, n_chol, nullptr);
  return step_smem(a, nsmax) <= 200 * 1024 && energy_smem(a, nsmax, 1) <= 200 * 1024;
}

int run_small_step(SmallArgs a, int nw, cudaStream_t st) {
  a.lchunk = pick_lchunk(a.M, a.n_chol, a.L);
  const size_t sm = step_smem(a, ns_max(a));
  static size_t cur[64] = {0};
  if (auto grow_ = grow_on_device(cur, sm)) {
    cudaFuncSetAttribute(small_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  }
  small_step_kernel<<<nw, 256, sm, st>>>(a);
  return 1;
}

int run_small_energy(SmallArgs a, int nw, cudaStream_t st) {
  const int nsmax = ns_max(a);
  int gc = 4096 / (nsmax * nsmax);
  if (gc > a.n_chol) gc = a.n_chol;
  if (gc < 1) gc = 1;
  a.gchunk = gc;
  const size_t sm = energy_smem(a, nsmax, gc);
  static size_t cur[64] = {0};
  if (auto grow_ = grow_on_device(cur, sm)) {
    cudaFuncSetAttribute(small_energy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  }
  small_energy_kernel<<<nw, 256, sm, st>>>(a);
  return 1;
}

}  // namespace afq
